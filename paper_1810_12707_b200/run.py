"""Run one of BASELINE.json's configurations through the C ABI and print the diagnostics series (thin driver: argument
marshalling and printing only; every step of the path runs in libmhd's kernels).

  python -m paper_1810_12707_b200.run --config 4 [--N 256] [--steps 100] [--diag-every 10] [--integrator ab2|rk4|pc]

Config 4 / 5 of BASELINE.json: ABC-flow dynamo at 256^3 / 512^3, 100 steps, energy and div B diagnostics every 10 steps.
"""
from __future__ import annotations

import argparse
import json
import sys


def run(config="4", N=None, steps=None, diag_every=10, integrator="ab2", device="cuda:0", out=sys.stdout):
    from . import MHD, inputs
    from . import binding as B
    cfg = inputs.by_name(config, N)
    steps = cfg.nsteps if steps is None else steps
    g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, device=device)
    g.set_option(B.MHD_OPT_INTEGRATOR, {"ab2": 0, "rk4": 1, "pc": 2}[integrator])
    g.set_fields(cfg.prim, "primitive")
    series = [g.diagnostics()]
    done = 0
    while done < steps:
        n = min(diag_every, steps - done)
        g.step(n)
        done += n
        series.append(g.diagnostics())
    for d in series:
        out.write(json.dumps({k: d[k] for k in ("step", "t", "ke", "me", "ie", "etot", "mass", "mom", "max_divb", "rho_min",
                                                 "p_min")}) + "\n")
    return series


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="4", choices=["1", "2", "3", "4", "5"])
    ap.add_argument("--N", type=int, default=None)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--diag-every", type=int, default=10)
    ap.add_argument("--integrator", default="ab2", choices=["ab2", "rk4", "pc"])
    a = ap.parse_args()
    run(a.config, a.N, a.steps, a.diag_every, a.integrator)


if __name__ == "__main__":
    main()
