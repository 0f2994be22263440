"""Fix one configuration: optional simulated-annealing preconditioner, then Alg. 1 until theta < tol.

    python -m paper_1209_4008_b200.fix --dims 48 48 48 64 --gauge coulomb --precision fp32 --eps 0.5 --seed 5 \\
        --anneal 1000 --T 1.4 0.01 --anneal-seed 7 --omega 1.7 --tol 1e-10 --tile          # BASELINE.json configs[4]
    python -m paper_1209_4008_b200.fix --in conf.npy --dims 24 24 24 48 --out fixed.npy    # a configuration on disk

Input: a numpy file holding complex128 (V, 4, 3, 3) in the canonical layout (include/gf.h), or a seeded synthetic
field (gf_inputs; --tile generates half the extents and repeats the field twice per direction, as bench.py does).
Prints F and theta after every stage, sweeps, device seconds and site-updates/s.
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
    ap.add_argument("--dims", type=int, nargs=4, required=True)
    ap.add_argument("--in", dest="infile")
    ap.add_argument("--out")
    ap.add_argument("--eps", type=float, default=0.4)
    ap.add_argument("--seed", type=int, default=3)
    ap.add_argument("--tile", action="store_true")
    ap.add_argument("--precision", default="fp64", choices=["fp32", "fp64"])
    ap.add_argument("--reals-per-link", type=int, default=18)
    ap.add_argument("--gauge", default="landau", choices=["landau", "coulomb"])
    ap.add_argument("--anneal", type=int, default=0, help="annealing sweeps before the relaxation (0 = none)")
    ap.add_argument("--T", type=float, nargs=2, default=[1.4, 0.01])
    ap.add_argument("--micro", type=int, default=0, help="microcanonical sweeps after every heatbath sweep")
    ap.add_argument("--anneal-seed", type=int, default=7)
    ap.add_argument("--update", default="or2", choices=["or2", "or1", "sr"])
    ap.add_argument("--omega", type=float, default=1.7, help="omega (or2, or1) or probability p (sr)")
    ap.add_argument("--tol", type=float, default=1e-10)
    ap.add_argument("--check-every", type=int, default=100)
    ap.add_argument("--max-sweeps", type=int, default=100000)
    ap.add_argument("--polish", type=float, default=0.0, help="mixed precision: after the fp32 run, convert to fp64 "
                    "(gf_convert) and continue to this tolerance")
    ap.add_argument("--all-slices", action="store_true", help="Coulomb: sweep every timeslice until the slowest is fixed")
    args = ap.parse_args()

    import numpy as np
    import torch

    import paper_1209_4008_b200 as gfm

    dims = tuple(args.dims)
    V = dims[0] * dims[1] * dims[2] * dims[3]
    if args.infile:
        U = np.load(args.infile)
        canon = torch.from_numpy(np.ascontiguousarray(U, dtype=np.complex128).view("float64").reshape(-1)).to("cuda")
    else:
        import gf_inputs

        gdims = tuple(d // 2 for d in dims) if args.tile else dims
        U = gf_inputs.smooth_random(gdims, args.eps, args.seed)
        canon = torch.from_numpy(U.view("float64").reshape(-1)).to("cuda")
        if args.tile:
            Nx, Ny, Nz, Nt = gdims
            canon = canon.view(Nt, Nz, Ny, Nx, 72).repeat(2, 2, 2, 2, 1).contiguous().view(-1)
    assert canon.numel() == V * 72, "field does not match --dims"
    fx = gfm.GaugeFixer(dims, precision=args.precision, gauge=args.gauge, reals_per_link=args.reals_per_link)
    gfm.gf_pack(fx.ctx, canon, fx.U)

    def timed(fn):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        out = fn()
        b.record()
        torch.cuda.synchronize()
        return out, a.elapsed_time(b) * 1e-3

    print(f"start: F = {fx.functional():.12f} theta = {fx.theta():.6e}")
    if args.anneal > 0:
        _, sec = timed(lambda: fx.anneal(args.T[0], args.T[1], args.anneal, args.anneal_seed, n_micro=args.micro))
        print(f"annealing: {args.anneal} steps T {args.T[0]} -> {args.T[1]} (+{args.micro} microcanonical each) in {sec:.3f} s "
              f"({V * args.anneal * (1 + args.micro) / sec:.3e} site-updates/s): F = {fx.functional():.12f} "
              f"theta = {fx.theta():.6e}")
    update = {"or2": gfm.GF_UPDATE_OVERRELAX2, "or1": gfm.GF_UPDATE_OVERRELAX1, "sr": gfm.GF_UPDATE_STOCHASTIC}[args.update]
    if args.gauge == "coulomb" and not args.all_slices:
        (n, th, F, per), sec = timed(lambda: fx.fix_slices(args.tol, update, args.omega, args.check_every, args.max_sweeps, 1))
        work = sum(per) * (V // dims[3])
        print(f"relaxation ({args.update} {args.omega}, stop rule per timeslice): slowest slice {n} sweeps, fastest {min(per)}, "
              f"mean {sum(per) / len(per):.1f} in {sec:.3f} s ({work / sec:.3e} site-updates/s): F = {F:.12f} max_t theta_t = {th:.6e}")
    else:
        (n, th, F), sec = timed(lambda: fx.fix(args.tol, update, args.omega, args.check_every, args.max_sweeps, 1))
        print(f"relaxation ({args.update} {args.omega}): {n} sweeps in {sec:.3f} s ({V * max(n, 1) / sec:.3e} site-updates/s): "
              f"F = {F:.12f} theta = {th:.6e}")
    if args.polish > 0.0 and args.precision == "fp32":
        wide = fx.convert_to(precision="fp64")
        fx.close()
        fx = wide
        (n, th, F), sec = timed(lambda: fx.fix(args.polish, update, args.omega, args.check_every, args.max_sweeps, 1))
        print(f"fp64 polish ({args.update} {args.omega}): {n} sweeps in {sec:.3f} s: F = {F:.12f} theta = {th:.6e}")
    if args.out:
        gfm.gf_unpack(fx.ctx, fx.U, canon)
        np.save(args.out, canon.cpu().numpy().view("complex128").reshape(V, 4, 3, 3))
    fx.close()


if __name__ == "__main__":
    main()
