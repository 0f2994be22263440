"""GPU-vs-oracle parity of the CUDA path, through the C ABI (include/gf.h), on the same seeded inputs.

Tolerances are BASELINE.json north_star's: per-link max|dU| after one sweep <= 1e-12 (fp64), <= 5e-5 (fp32);
after N sweeps F relative <= 1e-10 (fp64) / 1e-5 (fp32), theta relative <= 1e-6 (fp64); annealing: identical
Kennedy-Pendleton trial counts (accept decisions) given the shared Philox stream (fp64).
"""
import numpy as np
import pytest

import gf_inputs
import oracle

pytestmark = pytest.mark.gpu

TOL_LINK = {"fp64": 1e-12, "fp32": 5e-5}
TOL_F = {"fp64": 1e-10, "fp32": 1e-5}


@pytest.fixture(scope="module")
def gfm():
    import torch

    assert torch.cuda.is_available()
    import paper_1209_4008_b200 as m

    m.load_library()  # fails loudly if the CUDA library is missing
    return m


def _fixer(gfm, dims, precision, gauge="landau", R=18, tps=0, block=0):
    fx = gfm.GaugeFixer(dims, precision=precision, gauge=gauge, reals_per_link=R)
    gfm.gf_set_tuning(fx.ctx, tps, block)
    return fx


def _orc_gauge(gauge):
    return oracle.COULOMB if gauge == "coulomb" else oracle.LANDAU


# ---------------------------------------------------------------------------------------------------------
# layout round trip
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("R", [18, 12])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 8), (16, 8, 4, 6)])
def test_pack_unpack_roundtrip(gfm, precision, R, dims):
    U = gf_inputs.smooth_random(dims, 0.4, 21)
    fx = _fixer(gfm, dims, precision, R=R)
    fx.load(U)
    back = fx.download()
    if precision == "fp64" and R == 18:
        assert np.array_equal(back, U)  # bit exact
    elif precision == "fp64":
        assert np.array_equal(back[:, :, :2], U[:, :, :2])  # stored rows bit exact
        assert np.abs(back - U).max() < 4e-15  # row 2 rebuilt (C16)
    else:
        ref = U.astype(np.complex64).astype(np.complex128)
        if R == 18:
            assert np.array_equal(back, ref)  # each real rounded to nearest fp32
        else:
            assert np.array_equal(back[:, :, :2], ref[:, :, :2])
            assert np.abs(back - U).max() < 4e-7
    fx.close()


# ---------------------------------------------------------------------------------------------------------
# reductions
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("R", [18, 12])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (10, 6, 4, 8)])
def test_functional_and_theta(gfm, precision, R, gauge, dims):
    U = gf_inputs.smooth_random(dims, 0.4, 22)
    oracle.overrelax(U, dims, 1.7, 3, _orc_gauge(gauge))  # partly fixed: theta no longer O(1)
    fx = _fixer(gfm, dims, precision, gauge, R)
    fx.load(U)
    # the reductions run in fp64 on the STORED links: compare with the oracle on exactly those, formed on the host
    # (rounded to fp32 where the storage is; R = 12: row 2 = conj(row0 x row1) of the stored rows)
    stored = U.astype(np.complex64).astype(np.complex128) if precision == "fp32" else U.copy()
    if R == 12:
        r0, r1 = stored[:, :, 0, :], stored[:, :, 1, :]
        stored[:, :, 2, :] = np.conj(np.cross(r0, r1))
    og = _orc_gauge(gauge)
    tight = 1e-12 if not (precision == "fp32" and R == 12) else 1e-6  # fp32 R12 rebuilds row 2 in fp32
    assert fx.functional() == pytest.approx(oracle.functional(stored, dims, og), rel=tight)
    assert fx.theta() == pytest.approx(oracle.theta(stored, dims, og), rel=max(100 * tight, 1e-10))
    np.testing.assert_allclose(fx.theta_slices(), oracle.theta_slices(stored, dims, og), rtol=max(100 * tight, 1e-10))
    # and with the oracle on the original fp64 field, within the storage rounding
    rel = 1e-12 if precision == "fp64" else 2e-6
    assert fx.functional() == pytest.approx(oracle.functional(U, dims, og), rel=rel)
    assert fx.theta() == pytest.approx(oracle.theta(U, dims, og), rel=max(rel * 50, 1e-10))
    fx.close()


# ---------------------------------------------------------------------------------------------------------
# one sweep, link by link; every kernel variant
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("R", [18, 12])
@pytest.mark.parametrize("tps", [1, 2, 4])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_one_sweep_links(gfm, precision, R, tps, gauge):
    dims = (8, 6, 4, 10)  # V/2 = 960: several blocks, ragged last warp for every tps
    U = gf_inputs.smooth_random(dims, 0.4, 23)
    fx = _fixer(gfm, dims, precision, gauge, R, tps=tps, block=64)
    fx.load(U)
    fx.overrelax(1.7, 1)
    got = fx.download()
    oracle.overrelax(U, dims, 1.7, 1, _orc_gauge(gauge))
    assert np.abs(got - U).max() <= TOL_LINK[precision]
    fx.close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (2, 4, 2, 6), (4, 4, 4, 4), (34, 2, 2, 2)])
def test_one_sweep_small_and_extent_two(gfm, precision, dims):
    """degenerate sizes: extent 2 (x - mu and x + mu are the same site, the two links still distinct, C5)"""
    U = gf_inputs.hot(dims, 24)
    for tps in (1, 2, 4):
        for block in (32, 256):
            fx = _fixer(gfm, dims, precision, tps=tps, block=block)
            fx.load(U)
            fx.overrelax(1.5, 1)
            got = fx.download()
            fx.close()
            ref = U.copy()
            oracle.overrelax(ref, dims, 1.5, 1)
            assert np.abs(got - ref).max() <= TOL_LINK[precision], (dims, tps, block)


def test_half_sweep_order_and_reversal(gfm):
    """RED first then BLACK (C5); the traversal direction of the blocks must not matter (C6)."""
    dims = (8, 8, 4, 4)
    U = gf_inputs.smooth_random(dims, 0.4, 25)
    outs = []
    for rev in (0, 1):
        fx = _fixer(gfm, dims, "fp64")
        gfm.gf_set_l2_reversal(fx.ctx, rev)
        fx.load(U)
        fx.overrelax(1.7, 3)
        outs.append(fx.download())
        fx.close()
    assert np.array_equal(outs[0], outs[1])
    ref = U.copy()
    oracle.overrelax(ref, dims, 1.7, 3)
    assert np.abs(outs[0] - ref).max() <= 5e-12


# ---------------------------------------------------------------------------------------------------------
# N sweeps: F and theta
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision,R", [("fp64", 18), ("fp64", 12), ("fp32", 18), ("fp32", 12)])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_n_sweeps_F_theta(gfm, precision, R, gauge):
    dims = (8, 8, 8, 8)
    nsweeps = 60
    U = gf_inputs.smooth_random(dims, 0.4, 26)
    fx = _fixer(gfm, dims, precision, gauge, R)
    fx.load(U)
    fx.overrelax(1.7, nsweeps)
    og = _orc_gauge(gauge)
    oracle.overrelax(U, dims, 1.7, nsweeps, og)
    F_ref, th_ref = oracle.functional(U, dims, og), oracle.theta(U, dims, og)
    assert fx.functional() == pytest.approx(F_ref, rel=TOL_F[precision])
    if precision == "fp64":
        assert fx.theta() == pytest.approx(th_ref, rel=1e-6)
    else:
        assert fx.theta() == pytest.approx(th_ref, rel=5e-2, abs=1e-12)  # no tolerance stated for fp32 theta
    fx.close()


def test_config1_trivial_orbit(gfm):
    """BASELINE.json configs[0]: 4^4, trivial orbit seed 1, omega 1.7, until theta < 1e-14: F -> 1; links and
    theta checked against the oracle every sweep."""
    dims = (4, 4, 4, 4)
    U = gf_inputs.trivial_orbit(dims, 1)
    fx = _fixer(gfm, dims, "fp64")
    fx.load(U)
    sweeps = 0
    while fx.theta() >= 1e-14 and sweeps < 500:
        fx.overrelax(1.7, 1)
        oracle.overrelax(U, dims, 1.7, 1)
        sweeps += 1
        assert np.abs(fx.download() - U).max() <= 1e-12
        th_ref = oracle.theta(U, dims)
        assert fx.theta() == pytest.approx(th_ref, rel=1e-6, abs=1e-24)
    assert fx.theta() < 1e-14 and sweeps < 200
    assert abs(fx.functional() - 1.0) < 1e-12
    fx.close()


def test_fp32_long_run_unitarity(gfm):
    """C15: with the periodic re-orthonormalisation fp32 links stay unitary and F tracks the fp64 oracle"""
    dims = (8, 8, 8, 8)
    U = gf_inputs.smooth_random(dims, 0.4, 27)
    fx = _fixer(gfm, dims, "fp32")
    fx.load(U)
    fx.overrelax(1.7, 300)
    got = fx.download()
    uu, det = oracle.unitarity_defect(got, dims)
    assert uu < 5e-6 and det < 5e-6
    oracle.overrelax(U, dims, 1.7, 300)
    assert fx.functional() == pytest.approx(oracle.functional(U, dims), rel=1e-5)
    fx.close()


# ---------------------------------------------------------------------------------------------------------
# simulated annealing: decision parity
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("R", [18, 12])
@pytest.mark.parametrize("tps", [1, 2, 4])
def test_anneal_decisions_fp64(gfm, gauge, R, tps):
    import torch

    dims = (6, 4, 4, 8)
    V = int(np.prod(dims))
    U = gf_inputs.smooth_random(dims, 0.5, 28)
    fx = _fixer(gfm, dims, "fp64", gauge, R, tps=tps, block=64)
    trials = torch.zeros(V * 3, dtype=torch.int32, device="cuda")
    gfm.gf_set_trial_buffer(fx.ctx, trials)
    fx.load(U)
    fx.anneal(1.4, 0.2, 5, 7)
    got = fx.download()
    got_trials = trials.cpu().numpy().reshape(V, 3)
    ref_trials = oracle.anneal(U, dims, 1.4, 0.2, 5, 7, _orc_gauge(gauge), trials=True)
    assert np.array_equal(got_trials, ref_trials)  # identical accept decisions for every (site, subgroup)
    assert got_trials.max() > 1  # the test saw rejections
    assert np.abs(got - U).max() <= 1e-11
    fx.close()


@pytest.mark.parametrize("gauge,R,T,chain", [("coulomb", 18, 0.7, 2), ("landau", 18, 1.4, 2), ("landau", 12, 0.2, 2),
                                             ("landau", 18, 1.4, 1), ("coulomb", 12, 1.0, 1), ("landau", 18, 0.7, 0)])
def test_anneal_fp32_one_step(gfm, gauge, R, T, chain):
    """C14 in fp32: one step from identical input.  The fp32 kernel draws on the SFU and decides a trial again in
    double where u4^2 falls inside the error band of the threshold, so what can still flip an accept decision is the
    fp32 rounding of K (alpha differs from the oracle's at 1e-7): at most 1e-5 of the trial counts may differ (here:
    none of 12 288), and every link of every site without a flipped neighbour is within 5e-5."""
    import torch

    dims = (8, 8, 8, 8)
    V = int(np.prod(dims))
    U = gf_inputs.smooth_random(dims, 0.5, 29)
    fx = _fixer(gfm, dims, "fp32", gauge, R)
    gfm.gf_set_chain(fx.ctx, chain)  # 2: fp32 chain with the per-site repair (default), 1: double chain, 0: plain fp32
    trials = torch.zeros(V * 3, dtype=torch.int32, device="cuda")
    gfm.gf_set_trial_buffer(fx.ctx, trials)
    fx.load(U)
    # the input the kernel sees is the fp32-rounded field: give the oracle the same numbers, rounded on the host
    # (no oracle input comes from the CUDA path; gf_pack rounds to nearest like numpy, test_pack_unpack_roundtrip)
    U32 = U.astype(np.complex64).astype(np.complex128)
    if R == 12:
        U32[:, :, 2, :] = np.conj(np.cross(U32[:, :, 0, :], U32[:, :, 1, :]))
    fx.anneal(T, T, 1, 7)
    got = fx.download()
    got_trials = trials.cpu().numpy().reshape(V, 3)
    ref_trials = oracle.anneal(U32, dims, T, T, 1, 7, _orc_gauge(gauge), trials=True)
    assert (got_trials != ref_trials).mean() <= 1e-5
    assert np.abs(got - U32).max() <= TOL_LINK["fp32"]
    fx.close()


def test_anneal_then_overrelax_config5_shape(gfm):
    """BASELINE.json configs[4] in miniature: Coulomb gauge, anneal 1.4 -> 0.01 then overrelax until every
    timeslice has theta_t < 1e-10; plaquette invariant (P5), F rises."""
    dims = (8, 8, 8, 4)
    U = gf_inputs.smooth_random(dims, 0.5, 5)
    plaq0 = oracle.plaquette(U, dims)
    fx = _fixer(gfm, dims, "fp64", "coulomb")
    fx.load(U)
    F0 = fx.functional()
    fx.anneal(1.4, 0.01, 60, 7)
    F1 = fx.functional()
    sweeps = 0
    while fx.theta() >= 1e-10 and sweeps < 3000:
        fx.overrelax(1.7, 100)
        sweeps += 100
    assert max(fx.theta_slices()) < 1e-10
    F2 = fx.functional()
    assert F0 < F1 < F2
    got = fx.download()
    assert abs(oracle.plaquette(got, dims) - plaq0) < 1e-12
    uu, det = oracle.unitarity_defect(got, dims)
    assert uu < 1e-12 and det < 1e-12
    fx.close()


# ---------------------------------------------------------------------------------------------------------
# argument checking and the host-buffer path
# ---------------------------------------------------------------------------------------------------------
def test_argument_errors(gfm):
    with pytest.raises(gfm.GFError):
        gfm.gf_create(3, 4, 4, 4)
    with pytest.raises(gfm.GFError):
        gfm.gf_create(4, 4, 4, 0)
    ctx = gfm.gf_create(4, 4, 4, 4, gfm.GF_FP64, gfm.GF_LANDAU)
    with pytest.raises(gfm.GFError):
        gfm.gf_set_storage(ctx, 8)
    with pytest.raises(gfm.GFError):
        gfm.gf_overrelax(ctx, 1234, 2.0, 1)
    with pytest.raises(gfm.GFError):
        gfm.gf_overrelax(ctx, 1234, 0.9, 1)
    with pytest.raises(gfm.GFError):
        gfm.gf_overrelax(ctx, 0, 1.5, 1)
    with pytest.raises(gfm.GFError):
        gfm.gf_anneal(ctx, 1234, 0.0, 1.0, 1, 1)
    with pytest.raises(gfm.GFError):
        gfm.gf_set_tuning(ctx, 3, 64)
    gfm.gf_destroy(ctx)


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_host_buffer_path(gfm, precision):
    dims = (8, 4, 4, 6)
    U = gf_inputs.smooth_random(dims, 0.4, 30)
    ref = U.copy()
    ctx = gfm.gf_create(*dims, gfm.GF_FP64 if precision == "fp64" else gfm.GF_FP32, gfm.GF_LANDAU)
    F, th = gfm.gf_overrelax_host(ctx, U, 1.7, 2)
    gfm.gf_destroy(ctx)
    oracle.overrelax(ref, dims, 1.7, 2)
    assert np.abs(U - ref).max() <= TOL_LINK[precision] * 2
    assert F == pytest.approx(oracle.functional(ref, dims), rel=TOL_F[precision])
    assert th == pytest.approx(oracle.theta(ref, dims), rel=1e-6 if precision == "fp64" else 1e-3)


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_host_buffer_path_f32(gfm, precision):
    """canonical field held as float: fp32 contexts give the same links as the double-buffer call bit for bit
    (the pack rounds to the same fp32 numbers); fp64 contexts start from the widened floats"""
    dims = (8, 4, 4, 6)
    U = gf_inputs.smooth_random(dims, 0.4, 30)
    U32 = U.astype(np.complex64)
    prec = gfm.GF_FP64 if precision == "fp64" else gfm.GF_FP32
    ref = U32.astype(np.complex128)  # the input as the library sees it
    ctx = gfm.gf_create(*dims, prec, gfm.GF_LANDAU)
    F, th = gfm.gf_overrelax_host_f32(ctx, U32, 1.7, 2)
    gfm.gf_destroy(ctx)
    if precision == "fp32":
        ctx = gfm.gf_create(*dims, prec, gfm.GF_LANDAU)
        Ud = U.copy()
        F2, th2 = gfm.gf_overrelax_host(ctx, Ud, 1.7, 2)
        gfm.gf_destroy(ctx)
        assert np.array_equal(Ud.astype(np.complex64), U32) and F == F2 and th == th2
    oracle.overrelax(ref, dims, 1.7, 2)
    assert np.abs(U32.astype(np.complex128) - ref).max() <= 2 * TOL_LINK["fp32"]  # output is float either way
    assert F == pytest.approx(oracle.functional(ref, dims), rel=TOL_F[precision])


# ---------------------------------------------------------------------------------------------------------
# launch-time options change scheduling and caching, never a bit of the result
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("precision,R", [("fp64", 18), ("fp32", 12)])
def test_pdl_l2_policy_and_reversal_are_bit_neutral(gfm, precision, R):
    dims = (8, 6, 4, 10)
    U = gf_inputs.smooth_random(dims, 0.4, 31)
    results = []
    for pdl, ld, st, rev, pf in ((0, 0, 0, 0, 0), (1, 0, 2, 1, -1), (1, 1, 2, 0, 100), (0, 2, 1, 1, 7)):
        fx = _fixer(gfm, dims, precision, R=R)
        gfm.gf_set_pdl(fx.ctx, pdl)
        gfm.gf_set_l2_policy(fx.ctx, ld, st)
        gfm.gf_set_l2_reversal(fx.ctx, rev)
        gfm.gf_set_prefetch(fx.ctx, pf)
        fx.load(U)
        fx.overrelax(1.7, 3)
        fx.anneal(0.5, 0.3, 2, 9)
        results.append(fx.download())
        fx.close()
    for r in results[1:]:
        assert np.array_equal(r, results[0])
    ctx = gfm.gf_create(4, 4, 4, 4)
    with pytest.raises(gfm.GFError):
        gfm.gf_set_l2_policy(ctx, 3, 0)
    gfm.gf_destroy(ctx)


def test_fp32_chain_modes(gfm):
    """gf_set_chain: the hybrid chain runs the first sweep of a call in double (bit-identical to chain = 1), and on a
    nearly fixed field only that forced sweep; chain = 0 is the plain fp32 chain; all three within the fp32 bound on
    this small lattice; fp64 contexts ignore the setting"""
    dims = (8, 8, 8, 8)
    U = gf_inputs.smooth_random(dims, 0.4, 33)
    ref = U.copy()
    oracle.overrelax(ref, dims, 1.8, 1)
    outs = {}
    for chain in (0, 1, 2):
        fx = _fixer(gfm, dims, "fp32")
        gfm.gf_set_chain(fx.ctx, chain)
        fx.load(U)
        fx.overrelax(1.8, 1)
        outs[chain] = fx.download()
        assert np.abs(outs[chain] - ref).max() <= TOL_LINK["fp32"]
        launches, _ = gfm.gf_chain_count(fx.ctx)
        assert launches == (2 if chain == 2 else 0)  # the counter counts hybrid launches that went double
        if chain == 2:
            fx.overrelax(1.8, 80)           # rough at first, smooth later
            mid, _ = gfm.gf_chain_count(fx.ctx)
            fx.overrelax(1.8, 10)           # nearly fixed: only the forced first sweep
            end, _ = gfm.gf_chain_count(fx.ctx)
            assert 4 <= mid < 2 + 160 and end - mid == 2
        fx.close()
    assert np.array_equal(outs[1], outs[2])
    assert not np.array_equal(outs[0], outs[1])
    assert np.abs(outs[0] - outs[1]).max() < 2e-5
    fx = _fixer(gfm, dims, "fp64")
    gfm.gf_set_chain(fx.ctx, 0)
    fx.load(U)
    fx.overrelax(1.8, 1)
    assert np.abs(fx.download() - ref).max() <= TOL_LINK["fp64"]
    fx.close()
    ctx = gfm.gf_create(4, 4, 4, 4, gfm.GF_FP32)
    with pytest.raises(gfm.GFError):
        gfm.gf_set_chain(ctx, 3)
    gfm.gf_destroy(ctx)


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_host_batch_pipeline_matches_single_calls(gfm, precision):
    """gf_overrelax_host_batch (upload / sweep / download of consecutive configurations overlapped on three streams and
    three staging slots) gives every configuration exactly what the serial single-configuration call gives: links bit
    for bit, F and theta equal; more configurations than slots, pinned and pageable host memory"""
    import torch

    dims = (8, 4, 4, 6)
    n = 5
    dt = np.complex128 if precision == "fp64" else np.complex64
    fields = [gf_inputs.smooth_random(dims, 0.4, 80 + i).astype(dt) for i in range(n)]
    prec = gfm.GF_FP64 if precision == "fp64" else gfm.GF_FP32
    ctx = gfm.gf_create(*dims, prec, gfm.GF_LANDAU)
    single = gfm.gf_overrelax_host if precision == "fp64" else gfm.gf_overrelax_host_f32
    ref, vals = [], []
    for f in fields:
        g = f.copy()
        vals.append(single(ctx, g, 1.7, 3))
        ref.append(g)
    rdt = torch.float64 if precision == "fp64" else torch.float32
    pinned = [torch.from_numpy(f.copy().view(rdt.__str__().replace("torch.", "")).reshape(-1)).pin_memory() for f in fields]
    F, th = gfm.gf_overrelax_host_batch(ctx, pinned, 1.7, 3)
    for i in range(n):
        assert np.array_equal(pinned[i].numpy().view(dt).reshape(ref[i].shape), ref[i]), i
        assert F[i] == vals[i][0] and th[i] == vals[i][1]
    pageable = [f.copy() for f in fields[:2]]
    F2, th2 = gfm.gf_overrelax_host_batch(ctx, pageable, 1.7, 3)
    assert np.array_equal(pageable[1], ref[1]) and F2[0] == vals[0][0]
    assert gfm.gf_overrelax_host_batch(ctx, [], 1.7, 3) == ([], [])
    with pytest.raises(gfm.GFError):
        gfm.gf_overrelax_host_batch(ctx, pageable, 2.5, 1)
    gfm.gf_destroy(ctx)
    orc = fields[0].astype(np.complex128)
    oracle.overrelax(orc, dims, 1.7, 3)
    assert np.abs(ref[0].astype(np.complex128) - orc).max() <= 3 * TOL_LINK[precision]
