"""Host logic of the t-slab path (paper_1209_4008_b200.slab) on the CPU: the schedule of a half-sweep
(which face, which parity block, which direction, interior first) and the two transports, driven with an engine built
on the oracle.  The sharded run must reproduce the unsharded oracle bit for bit: a wrong face, parity block or order
reads a stale or undefined (NaN) ghost.  World size 2 over gloo covers the N > 1 transport."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)

import gf_inputs
import oracle
from paper_1209_4008_b200 import slab
from slab_oracle_engine import OracleSlab

DIMS = (4, 4, 2, 8)


def test_slab_bounds():
    assert slab.slab_bounds(32, 4) == [(0, 8), (8, 16), (16, 24), (24, 32)]
    assert slab.slab_bounds(12, 4) == [(0, 2), (2, 6), (6, 8), (8, 12)]  # even sizes, as equal as evenness allows
    assert slab.slab_bounds(8, 1) == [(0, 8)]
    for Nt, n in ((8, 5), (7, 2), (4, 0)):
        with pytest.raises(ValueError):
            slab.slab_bounds(Nt, n)


@pytest.mark.parametrize("nslabs", [1, 2, 4])
@pytest.mark.parametrize("overlap", [False, True])
@pytest.mark.parametrize("gauge", [oracle.LANDAU, oracle.COULOMB])
def test_local_ring_reproduces_the_unsharded_oracle(nslabs, overlap, gauge):
    U = gf_inputs.smooth_random(DIMS, 0.4, 71)
    ref = U.copy()
    bounds = slab.slab_bounds(DIMS[3], nslabs)
    engines = {r: OracleSlab(DIMS, b[0], b[1], U, gauge) for r, b in enumerate(bounds)}
    run = slab.SlabRunner(engines, slab.LocalRing(nslabs), DIMS, "coulomb" if gauge == oracle.COULOMB else "landau", overlap)
    run.overrelax(1.7, 2)
    oracle.overrelax(ref, DIMS, 1.7, 2, gauge)
    Vs = DIMS[0] * DIMS[1] * DIMS[2]
    for r, b in enumerate(bounds):
        assert np.array_equal(engines[r].owned(), ref[b[0] * Vs: b[1] * Vs]), (r, b)
    F, th = run.functional_theta()
    assert F == pytest.approx(oracle.functional(ref, DIMS, gauge), rel=1e-13)
    assert th == pytest.approx(oracle.theta(ref, DIMS, gauge), rel=1e-12)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, out):
    import torch.distributed as dist

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    U = gf_inputs.smooth_random(DIMS, 0.4, 72)
    ref = U.copy()
    ring = slab.DistRing()
    b = slab.slab_bounds(DIMS[3], world)[rank]
    eng = OracleSlab(DIMS, b[0], b[1], U)
    run = slab.SlabRunner({rank: eng}, ring, DIMS, "landau", overlap=True)
    n, th, F = run.fix(1.7, 0.0, check_every=2, max_sweeps=3)  # 2 + 1 sweeps, a check (all-reduce) in between
    oracle.overrelax(ref, DIMS, 1.7, 3)
    Vs = DIMS[0] * DIMS[1] * DIMS[2]
    same = bool(np.array_equal(eng.owned(), ref[b[0] * Vs: b[1] * Vs]))
    out.put((rank, n, same, F, th, oracle.functional(ref, DIMS), oracle.theta(ref, DIMS)))
    dist.barrier()
    dist.destroy_process_group()


def test_dist_ring_world2_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=300) for _ in range(2))
    for p in procs:
        p.join(timeout=300)
        assert p.exitcode == 0
    for rank, n, same, F, th, F_ref, th_ref in got:
        assert n == 3 and same, rank
        assert F == pytest.approx(F_ref, rel=1e-13) and th == pytest.approx(th_ref, rel=1e-12)
    assert got[0][3] == got[1][3] and got[0][4] == got[1][4]  # the all-reduced values agree on both ranks
