#!/usr/bin/env python
"""Run one of the Rayleigh-Taylor configurations on the GPU and log the mixing-layer widths.

    python -m paper_1405_1253_b200.run_rt --config 2 [--steps N] [--every 100] [--out widths.csv]

Every `--every` steps it calls lbm_diagnostics (mixing widths of eq. 12, and the lattice totals in
one pass over the lattice) and writes step, t/tau_RT, L_u, L_d, L_tot, mass, alpha_tot (eq. 14 via lbm_growth_rate),
with tau_RT = sqrt(Lx / (g At)) and At = (T_d - T_u)/(T_d + T_u) (Table II) from
lbm_rt_scales.  All arithmetic runs in the library.  --wall-kind 1: isothermal walls at T_d / T_u (reading 19).
"""
from __future__ import annotations

import argparse
import os
import sys
import time

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import synthetic_inputs as si  # noqa: E402


def run(cfg, steps: int, every: int, seed: int = si.DEFAULT_SEED, out=None, variant: int | None = None,
        wall_kind: int = 0, inplace: bool = False):
    import torch

    import paper_1405_1253_b200 as pkg
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g, wall_kind=wall_kind, T_wall=(cfg.T_d, cfg.T_u), inplace=inplace)
    if variant is not None:
        lat.set_variant(variant)
    lat.init_rt(seed, **cfg.rt_args())
    At, tau_rt = pkg.rt_scales(cfg.Lx, cfg.g, cfg.T_d, cfg.T_u)
    rows = []

    def log():
        d = lat.diagnostics(cfg.T_d, cfg.T_m, cfg.T_u, profiles=False)
        rows.append((lat.steps_done, lat.steps_done / tau_rt, d["L_u"], d["L_d"], d["L_u"] + d["L_d"], d["totals"][0]))

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
    ap.add_argument("--wall-kind", type=int, default=0)
    ap.add_argument("--inplace", action="store_true")
    args = ap.parse_args()
    cfg = si.rt_config(args.config)
    steps = args.steps or cfg.steps
    fh = open(args.out, "w") if args.out else None
    rows, wall = run(cfg, steps, args.every, args.seed, wall_kind=args.wall_kind, inplace=args.inplace)
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
