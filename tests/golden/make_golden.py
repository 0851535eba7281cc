"""Writes tests/golden/long_runs.txt: end states of full-length runs of BASELINE.json's configs computed by the CPU oracle
ONLY (this script imports nothing from the CUDA path; the seeded input generators are the shared, arithmetic-free module).

  python tests/golden/make_golden.py [config3] [config4]

config3: 128^3 decaying turbulence, all 500 steps.
config4: 256^3 ABC dynamo, all 100 steps (config 4).
Stored per run: diagnostics at the end, the L2 norm of each conservative field, and each field at 48 seeded sample points.
The GPU parity test tests/test_gpu_parity.py::test_full_length_runs_against_stored_oracle_states compares with these;
tests/test_oracle_pins.py::test_golden_file_is_the_oracles re-derives a cheap prefix so the file cannot drift from the oracle.
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle                                            # noqa: E402
from paper_1810_12707_b200 import inputs                 # noqa: E402  (seeded generators only)

RUNS = {"config3": ("3", 128, 500), "config4": ("4", 256, 100)}
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "long_runs.txt")


def sample_points(N, n=48, seed=20181012):
    rng = np.random.default_rng(seed + N)
    return rng.integers(0, N, size=(n, 3))


def record(name):
    cfgname, N, nsteps = RUNS[name]
    cfg = inputs.by_name(cfgname, N)
    o = oracle.Oracle(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt)
    o.set_fields(cfg.prim, "primitive")
    t0 = time.time()
    prefix = None
    done = 0
    while done < nsteps:
        n = min(10, nsteps - done)
        o.step(n)
        done += n
        if done == 10:
            prefix = o.diagnostics()
        print(name, done, "steps", round(time.time() - t0), "s", flush=True)
    U = o.get_fields("conservative")
    pts = sample_points(N)
    d = o.diagnostics()
    return {"name": name, "config": cfgname, "N": N, "steps": nsteps, "dt": cfg.dt,
            "diag": {k: d[k] for k in ("ke", "me", "ie", "mass", "etot", "rho_min", "p_min")},
            "diag_after_10": {k: prefix[k] for k in ("ke", "me", "ie")},
            "norms": [float(np.linalg.norm(u)) for u in U],
            "points": pts.tolist(),
            "samples": [[float(u[z, y, x]) for (z, y, x) in pts] for u in U]}


def augment(rec):
    """Adds a cheap prefix to an existing record, for the CPU drift test (tests/test_oracle_pins.py):
    config3 (128^3): diagnostics and the first 8 sample points of every field after the first 2 steps;
    config4 (256^3): the same after the first step, at 8 seeded points whose indices are multiples of 4 — the drift test
    re-derives them on a 64^3 grid (after one Euler step every mode of config 4 is <= 12 <= k_c(64), so the two
    resolutions agree at the shared grid points to roundoff)."""
    cfg = inputs.by_name(rec["config"], rec["N"])
    o = oracle.Oracle(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt)
    o.set_fields(cfg.prim, "primitive")
    if rec["name"] == "config4":
        nst, key = 1, "after_1"
        pts = (np.random.default_rng(4).integers(0, rec["N"] // 4, size=(8, 3)) * 4).tolist()
    else:
        nst, key = 2, "after_2"
        pts = rec["points"][:8]
    o.step(nst)
    d = o.diagnostics()
    U = o.get_fields("conservative")
    rec["diag_" + key] = {k: d[k] for k in ("ke", "me", "ie", "max_divb")}
    rec["points_" + key] = pts
    rec["samples_" + key] = [[float(u[z, y, x]) for (z, y, x) in pts] for u in U]
    return rec


def main():
    if sys.argv[1:2] == ["--augment"]:          # python tests/golden/make_golden.py --augment config3
        recs = {}
        for line in open(OUT):
            if line.startswith("{"):
                r = json.loads(line)
                recs[r["name"]] = r
        for n in sys.argv[2:]:
            recs[n] = augment(recs[n])
        write(recs)
        return
    names = sys.argv[1:] or list(RUNS)
    have = {}
    if os.path.exists(OUT):
        for line in open(OUT):
            if line.startswith("{"):
                r = json.loads(line)
                have[r["name"]] = r
    for n in names:
        have[n] = record(n)
        write(have)


def write(have):
    with open(OUT, "w") as f:
        f.write("# Oracle end states of full-length runs (tests/golden/make_golden.py; oracle/ only). Cite: BASELINE.json configs 3, 4;\n")
        f.write("# SURVEY.md 8(d). One JSON record per line; floats are repr-exact.\n")
        for k in sorted(have):
            f.write(json.dumps(have[k]) + "\n")


if __name__ == "__main__":
    main()
