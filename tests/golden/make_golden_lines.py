"""Writes tests/golden/rhs_lines.txt: the CPU oracle's right-hand side (Eq. 17-19; Eq. 12) of seeded
states on full grid LINES along x, along y and along z — dense along every transformed axis, so a defect of one butterfly
stage, twiddle or pruning decision of the 3-D transforms shows up, which scattered sample points would miss.
The oracle ONLY: this script imports nothing from the CUDA path (the seeded input generators are the shared,
arithmetic-free module).

  python tests/golden/make_golden_lines.py [64] [512]        (default: both; 512^3 needs ~46 GB of RAM and ~15 min per state)

Per record: the state's recipe, rhs_scales' per-field flux norm phi and diffusion scale dsc (for the backward-error bar
beta of tests/test_gpu_parity.py), the line anchors, and R_f on every line.  The 64^3 records are re-derived by
tests/test_oracle_pins.py::test_golden_lines_are_the_oracles so that the file cannot drift from the oracle; the GPU test
tests/test_gpu_parity.py::test_rhs_on_dense_lines_against_stored_oracle compares libmhd with every record.
"""
import json
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle                                            # noqa: E402
from paper_1810_12707_b200 import inputs                 # noqa: E402  (seeded generators only)

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "rhs_lines.txt")
NLINES = 3          # lines per axis and field


def state(kind, N):
    """(prim, L, gamma, mu, eta): 'abc' = BASELINE config 4/5 (ABC dynamo) at N^3; 'random' = a smooth random state that
    fills every mode up to |n| = 6 in all eight fields (non-uniform density, compressive velocity, solenoidal B)."""
    if kind == "abc":
        cfg = inputs.config45(N)
        return cfg.prim, cfg.L, cfg.gamma, cfg.mu, cfg.eta
    return inputs.random_smooth_state(N, 512, kmax=6), 2 * math.pi, 5.0 / 3.0, 0.01, 0.02


def anchors(N, kind):
    """NLINES seeded (z, y, x) anchors; the line along axis a through anchor p keeps p's other two coordinates."""
    rng = np.random.default_rng(20181012 + N + (0 if kind == "abc" else 1))
    return rng.integers(0, N, size=(NLINES, 3)).tolist()


def lines_of(field, pts):
    """[axis][line] -> N values: axis 0 = along x, 1 = along y, 2 = along z."""
    return [[field[z, y, :].tolist() for (z, y, x) in pts],
            [field[z, :, x].tolist() for (z, y, x) in pts],
            [field[:, y, x].tolist() for (z, y, x) in pts]]


def record(kind, N):
    prim, L, gamma, mu, eta = state(kind, N)
    o = oracle.Oracle(N, L, gamma, mu, eta, 1e-3)
    o.set_fields(prim, "primitive")
    R, phi, dsc = o.rhs_scales()
    pts = anchors(N, kind)
    return {"kind": kind, "N": N, "L": L, "gamma": gamma, "mu": mu, "eta": eta, "anchors": pts,
            "phi": phi.tolist(), "dsc": dsc.tolist(), "norms": [float(np.linalg.norm(r)) for r in R],
            "lines": [lines_of(r, pts) for r in R]}


def read():
    if not os.path.exists(OUT):
        return []
    return [json.loads(l) for l in open(OUT) if l.strip() and not l.startswith("#")]


def main():
    sizes = [int(a) for a in sys.argv[1:]] or [64, 512]
    have = {(r["kind"], r["N"]): r for r in read()}
    for N in sizes:
        for kind in ("abc", "random"):
            have[(kind, N)] = record(kind, N)
            print("done", kind, N, flush=True)
            with open(OUT + ".tmp", "w") as f:
                f.write("# oracle right-hand sides on dense grid lines; written by tests/golden/make_golden_lines.py (oracle/ only)\n")
                for key in sorted(have):
                    f.write(json.dumps(have[key]) + "\n")
            os.replace(OUT + ".tmp", OUT)


if __name__ == "__main__":
    main()
