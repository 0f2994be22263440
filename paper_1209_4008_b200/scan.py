"""Parameter scan: sweeps needed to reach theta < tol as a function of the overrelaxation / stochastic-relaxation
parameter (the shape of Fig. 2 left of the paper, on a seeded synthetic field -- the paper's
Monte-Carlo configuration is not available).

    python -m paper_1209_4008_b200.scan [--dims 32 32 32 32] [--eps 0.4] [--seed 3] [--precision fp64]
        [--tol 1e-12] [--check-every 100] [--max-sweeps 20000]
        [--or2 1.5,1.6,1.7,1.8,1.9] [--or1 1.5,1.6,1.7] [--sr 0.5,0.7,0.9]

Every run starts from the same field and goes through gf_fix (Alg. 1 with its stop rule).  Prints one line per
parameter: update, parameter, sweeps, theta, F, seconds on the device.
"""
from __future__ import annotations

import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--dims", type=int, nargs=4, default=[32, 32, 32, 32])
    ap.add_argument("--eps", type=float, default=0.4)
    ap.add_argument("--seed", type=int, default=3)
    ap.add_argument("--precision", default="fp64", choices=["fp32", "fp64"])
    ap.add_argument("--reals-per-link", type=int, default=18)
    ap.add_argument("--gauge", default="landau", choices=["landau", "coulomb"])
    ap.add_argument("--tol", type=float, default=1e-12)
    ap.add_argument("--check-every", type=int, default=100)
    ap.add_argument("--max-sweeps", type=int, default=20000)
    ap.add_argument("--or2", default="1.5,1.6,1.7,1.8,1.9")
    ap.add_argument("--or1", default="1.5,1.7")
    ap.add_argument("--sr", default="0.5,0.7,0.9")
    args = ap.parse_args()

    import torch

    import gf_inputs
    import paper_1209_4008_b200 as gfm

    dims = tuple(args.dims)
    U = gf_inputs.smooth_random(dims, args.eps, args.seed)
    canon = torch.from_numpy(U.view("float64").reshape(-1)).to("cuda")
    fx = gfm.GaugeFixer(dims, precision=args.precision, gauge=args.gauge, reals_per_link=args.reals_per_link)
    runs = [("OR2", gfm.GF_UPDATE_OVERRELAX2, float(x)) for x in args.or2.split(",") if x]
    runs += [("OR1", gfm.GF_UPDATE_OVERRELAX1, float(x)) for x in args.or1.split(",") if x]
    runs += [("SR", gfm.GF_UPDATE_STOCHASTIC, float(x)) for x in args.sr.split(",") if x]
    print(f"# dims {dims} eps {args.eps} seed {args.seed} {args.precision} R{args.reals_per_link} {args.gauge} "
          f"tol {args.tol} check every {args.check_every}")
    print("# update param sweeps theta F seconds")
    for name, update, param in runs:
        gfm.gf_pack(fx.ctx, canon, fx.U)
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        n, th, F = fx.fix(args.tol, update, param, args.check_every, args.max_sweeps, seed=1)
        t1.record()
        torch.cuda.synchronize()
        print(f"{name} {param:g} {n} {th:.3e} {F:.12f} {t0.elapsed_time(t1) * 1e-3:.3f}", flush=True)
    fx.close()


if __name__ == "__main__":
    main()
