"""t-slab sharding of one configuration on ONE GPU: 2 and 4 slab contexts in one process,
plain device-to-device copies standing in for the NVLink messages.  The sharded run must give the unsharded result bit
for bit (same kernels, same per-site arithmetic; the Philox counters carry the site of the whole lattice), and both
must match the oracle within the stated tolerances.  Unmeasured on multi-GPU hardware (no such node in this run)."""
import numpy as np
import pytest

import gf_inputs
import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gfm():
    import torch

    assert torch.cuda.is_available()
    import paper_1209_4008_b200 as m

    m.load_library()
    return m


def _load(run, bounds, U, dims):
    Vs = dims[0] * dims[1] * dims[2]
    for r, b in enumerate(bounds):
        run.eng[r].load(np.ascontiguousarray(U[b[0] * Vs: b[1] * Vs]))


def _gather(run, bounds):
    return np.concatenate([run.eng[r].download() for r in range(len(bounds))])


@pytest.mark.parametrize("nslabs", [2, 4])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_config2_16x3x32_slabs_bit_identical_fp64(gfm, nslabs, gauge):
    """BASELINE.json configs[1] shape, fp64: 5 overrelaxation sweeps sharded = unsharded, bit for bit; F and theta from the
    raw sums of the slabs; the oracle within 1e-12 per link after one sweep"""
    from paper_1209_4008_b200 import slab

    dims = (16, 16, 16, 32)
    og = oracle.COULOMB if gauge == "coulomb" else oracle.LANDAU
    U = gf_inputs.smooth_random(dims, 0.3, 2)
    fx = gfm.GaugeFixer(dims, precision="fp64", gauge=gauge)
    if gauge == "coulomb":
        gfm.gf_set_coulomb_reading(fx.ctx, False)  # the slabs run reading A
    fx.load(U)
    fx.overrelax(1.7, 1)
    one = fx.download()
    fx.overrelax(1.7, 4)
    whole = fx.download()
    for overlap in (False, True):
        run, bounds = slab.local_slabs(dims, nslabs, "fp64", gauge, overlap=overlap)
        _load(run, bounds, U, dims)
        run.overrelax(1.7, 1)
        assert np.array_equal(_gather(run, bounds), one)
        for s in range(1, 5):
            run.sweep(("relax", 0, 1.7, 0), s)
        assert np.array_equal(_gather(run, bounds), whole), (nslabs, overlap)
        F, th = run.functional_theta()
        assert F == pytest.approx(fx.functional(), rel=1e-13) and th == pytest.approx(fx.theta(), rel=1e-11)
        for e in run.eng.values():
            e.close()
    ref = U.copy()
    oracle.overrelax(ref, dims, 1.7, 1, og)
    assert np.abs(one - ref).max() <= 1e-12
    oracle.overrelax(ref, dims, 1.7, 4, og)
    assert fx.functional() == pytest.approx(oracle.functional(ref, dims, og), rel=1e-10)
    fx.close()


@pytest.mark.parametrize("precision,R", [("fp64", 12), ("fp32", 18), ("fp32", 12)])
def test_slabs_other_formats_and_random_updates(gfm, precision, R):
    """12-real storage and fp32 (plain fp32 chain on both sides: the hybrid chain keeps its roughness flags per context,
    so a sharded fp32 run may pick the double chain at other half-sweeps than the unsharded one -- within tolerance, not
    bit-identical); stochastic relaxation and annealing draw the numbers of the whole-lattice site: bit-identical"""
    from paper_1209_4008_b200 import slab

    dims = (8, 8, 8, 12)
    U = gf_inputs.smooth_random(dims, 0.4, 73)
    fx = gfm.GaugeFixer(dims, precision=precision, reals_per_link=R)
    gfm.gf_set_chain(fx.ctx, 0)
    run, bounds = slab.local_slabs(dims, 3, precision, "landau", R)  # slabs of 4 slices
    for e in run.eng.values():
        gfm.gf_set_chain(e.ctx, 0)
    fx.load(U)
    _load(run, bounds, U, dims)
    fx.relax(gfm.GF_UPDATE_STOCHASTIC, 0.5, 3, seed=2**33 + 9)
    run.overrelax(0.5, 3, update=gfm.GF_UPDATE_STOCHASTIC, seed=2**33 + 9)
    assert np.array_equal(_gather(run, bounds), fx.download())
    fx.anneal(1.2, 0.4, 3, 7)
    run.anneal(1.2, 0.4, 3, 7)
    assert np.array_equal(_gather(run, bounds), fx.download())
    fx.overrelax(1.7, 20)  # crosses the re-orthonormalisation cadence (sweep 16)
    run.overrelax(1.7, 20)
    assert np.array_equal(_gather(run, bounds), fx.download())
    fx.close()
    # default (hybrid) chain in fp32: within the fp32 tolerance of the oracle after one sweep
    if precision == "fp32":
        run2, b2 = slab.local_slabs(dims, 2, precision, "landau", R)
        _load(run2, b2, U, dims)
        run2.overrelax(1.8, 1)
        ref = U.copy()
        oracle.overrelax(ref, dims, 1.8, 1)
        assert np.abs(_gather(run2, b2) - ref).max() <= 5e-5
        for e in run2.eng.values():
            e.close()
    for e in run.eng.values():
        e.close()


@pytest.mark.parametrize("nslabs", [2, 4])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_slabs_on_their_own_streams_bit_identical(gfm, nslabs, gauge):
    """every slab on its own CUDA stream, the face copies ordered by events alone (StreamRing): interior launches,
    face traffic and the other slabs' launches may now run in any order the events allow, so a missing dependency in
    the schedule would show as a wrong link.  Relaxation, annealing and stochastic sweeps sharded = unsharded bit for
    bit, repeated so that an ordering that only sometimes fails has several chances; F and theta from the raw sums."""
    from paper_1209_4008_b200 import slab

    dims = (16, 16, 16, 16)
    U = gf_inputs.smooth_random(dims, 0.4, 75)
    fx = gfm.GaugeFixer(dims, precision="fp64", gauge=gauge)
    if gauge == "coulomb":
        gfm.gf_set_coulomb_reading(fx.ctx, False)  # the slabs run reading A
    fx.load(U)
    fx.overrelax(1.7, 6)
    fx.anneal(1.0, 0.2, 3, 11)
    fx.relax(gfm.GF_UPDATE_STOCHASTIC, 0.6, 4, seed=5)
    whole = fx.download()
    for rep in range(3):
        run, bounds = slab.local_slabs(dims, nslabs, "fp64", gauge, overlap=True, streams=True)
        assert len({e.stream.cuda_stream for e in run.eng.values()}) == nslabs
        _load(run, bounds, U, dims)
        run.overrelax(1.7, 6)
        run.anneal(1.0, 0.2, 3, 11)
        run.overrelax(0.6, 4, update=gfm.GF_UPDATE_STOCHASTIC, seed=5)
        assert np.array_equal(_gather(run, bounds), whole), (nslabs, rep)
        F, th = run.functional_theta()
        assert F == pytest.approx(fx.functional(), rel=1e-13) and th == pytest.approx(fx.theta(), rel=1e-11)
        for e in run.eng.values():
            e.close()
    fx.close()


def test_slab_fix_loop_and_errors(gfm):
    """the driver's Alg. 1 loop on slabs stops where gf_fix with the separate check stops (same theta to rounding);
    argument checks of the slab calls"""
    from paper_1209_4008_b200 import slab

    dims = (8, 8, 8, 8)
    U = gf_inputs.smooth_random(dims, 0.3, 74)
    fx = gfm.GaugeFixer(dims, precision="fp64")
    gfm.gf_set_monitor(fx.ctx, 0)
    fx.load(U)
    n, th, F = fx.fix(1e-9, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=5, max_sweeps=2000)
    run, bounds = slab.local_slabs(dims, 4, "fp64")
    _load(run, bounds, U, dims)
    n2, th2, F2 = run.fix(1.6, 1e-9, check_every=5, max_sweeps=2000)
    assert n2 == n and th2 == pytest.approx(th, rel=1e-9) and F2 == pytest.approx(F, rel=1e-13)
    assert np.array_equal(_gather(run, bounds), fx.download())
    e0 = run.eng[0]
    with pytest.raises(gfm.GFError):
        gfm.gf_relax_half(e0.ctx, e0.U, 0, 1.7, 2, 0, 0, 0, 2)      # parity
    with pytest.raises(gfm.GFError):
        gfm.gf_relax_half(e0.ctx, e0.U, 0, 1.7, 0, 0, 0, 1, 2)      # slices outside the slab
    with pytest.raises(gfm.GFError):
        gfm.gf_slab_pack_face(fx.ctx, fx.U, 0, 0, e0.new_face())    # not a slab context
    for bad in ((8, 8, 8, 8, 1, 5), (8, 8, 8, 8, 0, 1), (8, 8, 8, 8, 4, 10)):
        with pytest.raises(gfm.GFError):
            gfm.gf_create_slab(*bad)
    assert gfm.gf_slab_face_bytes(e0.ctx) == 8 * 8 * 8 // 2 * 18 * 8
    fx.close()
    for e in run.eng.values():
        e.close()
