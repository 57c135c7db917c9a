#!/usr/bin/env python
"""Run one of the Rayleigh-Taylor configurations on the GPU and log the mixing-layer widths.

    python -m paper_1405_1253_b200.run_rt --config 2 [--steps N] [--every 100] [--out widths.csv]

Every `--every` steps it calls lbm_mixing_widths (eq. 12) and lbm_totals and writes
step, t/tau_RT, L_u, L_d, L_tot, mass, alpha_tot (eq. 14 via lbm_growth_rate), with tau_RT = sqrt(Lx / (g At)) and
At = (T_d - T_u)/(T_d + T_u) (Table II).  All arithmetic runs in the CUDA library.
"""
from __future__ import annotations

import argparse
import math
import os
import sys
import time

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import synthetic_inputs as si  # noqa: E402


def run(cfg, steps: int, every: int, seed: int = si.DEFAULT_SEED, out=None, variant: int | None = None):
    import torch

    import paper_1405_1253_b200 as pkg
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    if variant is not None:
        lat.set_variant(variant)
    lat.init_rt(seed, **cfg.rt_args())
    At = (cfg.T_d - cfg.T_u) / (cfg.T_d + cfg.T_u)
    tau_rt = math.sqrt(cfg.Lx / (cfg.g * At))
    rows = []

    def log():
        lu, ld, _ = lat.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u, want_tbar=False)
        mass = lat.totals()[0]
        rows.append((lat.steps_done, lat.steps_done / tau_rt, lu, ld, lu + ld, mass))

    log()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    done = 0
    while done < steps:
        n = min(every, steps - done)
        lat.step(n)
        done += n
        log()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    lat.close()
    # alpha_tot(t) of eq. 14 from the logged L_tot; appended as a 7th column
    alpha = pkg.growth_rate([r[0] for r in rows], [r[4] for r in rows], cfg.g, At) if len(rows) > 1 and cfg.g > 0 else [0.0] * len(rows)
    rows = [r + (float(a),) for r, a in zip(rows, alpha)]
    return rows, wall


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--steps", type=int, default=0, help="default: the config's own step count")
    ap.add_argument("--every", type=int, default=100)
    ap.add_argument("--seed", type=int, default=si.DEFAULT_SEED)
    ap.add_argument("--out", default="")
    args = ap.parse_args()
    cfg = si.rt_config(args.config)
    steps = args.steps or cfg.steps
    fh = open(args.out, "w") if args.out else None
    rows, wall = run(cfg, steps, args.every, args.seed)
    if fh:
        fh.write("step,t_over_tau,L_u,L_d,L_tot,mass,alpha_tot\n")
        for r in rows:
            fh.write("%d,%.6f,%.9f,%.9f,%.9f,%.15e,%.6e\n" % r)
        fh.close()
    sites = cfg.Lx * cfg.Lz
    print(f"{cfg.name}: {steps} steps in {wall:.2f} s incl. {len(rows)} diagnostics = "
          f"{sites * steps / wall / 1e6:.0f} MLUPS; L_tot {rows[0][4]:.3f} -> {rows[-1][4]:.3f}; "
          f"mass drift {abs(rows[-1][5] / rows[0][5] - 1):.2e}")


if __name__ == "__main__":
    main()
