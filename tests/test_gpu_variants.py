"""CUDA path vs oracle for the update variants (gf_relax: first-order overrelaxation, stochastic relaxation;
gf_anneal_micro: microcanonical sweeps inside the annealing).  Tolerances as for the second-order sweep
(north_star): per link 1e-12 (fp64) / 5e-5 (fp32) after one sweep; decisions (g^2 taken or not) are taken in
double on both sides from the same Philox word, so they must be identical in fp32 too."""
import numpy as np
import pytest

import gf_inputs
import oracle

pytestmark = pytest.mark.gpu

TOL_LINK = {"fp64": 1e-12, "fp32": 5e-5}
ORC_GAUGE = {"landau": oracle.LANDAU, "coulomb": oracle.COULOMB}


@pytest.fixture(scope="module")
def gfm():
    import torch

    assert torch.cuda.is_available()
    import paper_1209_4008_b200 as m

    m.load_library()
    return m


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("R", [18, 12])
@pytest.mark.parametrize("tps", [0, 1, 2, 4])
@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("update,param", [(1, 1.6), (2, 0.35)])
def test_one_sweep_links(gfm, precision, R, tps, gauge, update, param):
    dims = (8, 6, 4, 10)
    U = gf_inputs.smooth_random(dims, 0.4, 51)
    fx = gfm.GaugeFixer(dims, precision=precision, gauge=gauge, reals_per_link=R)
    gfm.gf_set_tuning(fx.ctx, tps, 0 if tps == 0 else 64)
    fx.load(U)
    ref = U.copy()
    fx.relax(update, param, 1, seed=13)
    got = fx.download()
    oracle.relax(ref, dims, update, param, 1, 13, ORC_GAUGE[gauge])
    assert np.abs(got - ref).max() <= TOL_LINK[precision]
    fx.close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_stochastic_sweep_counter_and_limits(gfm, precision):
    """three sweeps in one call use sweep counters 0,1,2 (as the oracle); p = 1 conserves F (C19); p = 0 is
    relaxation; the update 0 of gf_relax is gf_overrelax"""
    dims = (6, 4, 4, 8)
    U = gf_inputs.smooth_random(dims, 0.4, 52)
    fx = gfm.GaugeFixer(dims, precision=precision)
    fx.load(U)
    ref = U.copy()
    fx.relax(gfm.GF_UPDATE_STOCHASTIC, 0.5, 3, seed=2**40 + 5)
    oracle.relax(ref, dims, oracle.UPDATE_STOCHASTIC, 0.5, 3, 2**40 + 5)
    assert np.abs(fx.download() - ref).max() <= 3 * TOL_LINK[precision]
    F0 = fx.functional()
    fx.relax(gfm.GF_UPDATE_STOCHASTIC, 1.0, 2, seed=1)
    assert abs(fx.functional() - F0) < (1e-13 if precision == "fp64" else 2e-6)
    fx.load(U)
    fx.relax(gfm.GF_UPDATE_STOCHASTIC, 0.0, 1, seed=1)
    b = U.copy()
    oracle.overrelax(b, dims, 1.0, 1)
    assert np.abs(fx.download() - b).max() <= TOL_LINK[precision]
    fx.load(U)
    fx.relax(gfm.GF_UPDATE_OVERRELAX2, 1.7, 2)
    c = fx.download()
    fx.load(U)
    fx.overrelax(1.7, 2)
    assert np.array_equal(c, fx.download())
    fx.close()


def test_first_order_fixes_the_gauge(gfm):
    """config 1 with the first-order update: theta < 1e-14 and F -> 1 (P1), per-sweep parity with the oracle"""
    dims = (4, 4, 4, 4)
    U = gf_inputs.trivial_orbit(dims, 1)
    fx = gfm.GaugeFixer(dims, precision="fp64")
    fx.load(U)
    for sweep in range(300):
        fx.relax(gfm.GF_UPDATE_OVERRELAX1, 1.3, 1)
        oracle.relax(U, dims, oracle.UPDATE_OVERRELAX1, 1.3, 1)
        if sweep < 20:
            assert np.abs(fx.download() - U).max() <= 1e-12
        if fx.theta() < 1e-14:
            break
    assert fx.theta() < 1e-14 and abs(fx.functional() - 1.0) < 1e-12
    assert fx.theta() == pytest.approx(oracle.theta(U, dims), rel=1e-6, abs=1e-24)
    fx.close()


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_anneal_micro_decisions_fp64(gfm, gauge):
    import torch

    dims = (6, 4, 4, 8)
    V = int(np.prod(dims))
    U = gf_inputs.smooth_random(dims, 0.5, 53)
    fx = gfm.GaugeFixer(dims, precision="fp64", gauge=gauge)
    trials = torch.zeros(V * 3, dtype=torch.int32, device="cuda")
    gfm.gf_set_trial_buffer(fx.ctx, trials)
    fx.load(U)
    fx.anneal(1.2, 0.3, 2, 7, n_micro=2)
    ref_trials = oracle.anneal_micro(U, dims, 1.2, 0.3, 2, 2, 7, ORC_GAUGE[gauge], trials=True)
    assert np.array_equal(trials.cpu().numpy().reshape(V, 3), ref_trials)
    # 2 heatbath + 4 microcanonical sweeps; the g^2 sweeps do not damp rounding differences (they grow by
    # roughly 5x per sweep from 1e-14), so the bar after 6 sweeps is 1e-10
    assert np.abs(fx.download() - U).max() <= 1e-10
    fx.close()


def test_argument_errors(gfm):
    ctx = gfm.gf_create(4, 4, 4, 4)
    for args in ((1234, 1, 2.0, 1), (1234, 1, 0.5, 1), (1234, 2, 1.5, 1), (1234, 2, -0.1, 1), (1234, 3, 1.5, 1),
                 (1234, 1, 1.5, -1), (0, 1, 1.5, 1)):
        with pytest.raises(gfm.GFError):
            gfm.gf_relax(ctx, *args)
    with pytest.raises(gfm.GFError):
        gfm.gf_anneal_micro(ctx, 1234, 1.0, 1.0, 1, -1, 1)
    gfm.gf_destroy(ctx)


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
def test_fix_loop_matches_oracle(gfm, gauge):
    """Alg. 1 with its stop rule (gf_fix vs orc_fix): same number of sweeps, theta within 1e-6 relative"""
    dims = (6, 6, 6, 4)
    U = gf_inputs.smooth_random(dims, 0.3, 54)
    fx = gfm.GaugeFixer(dims, precision="fp64", gauge=gauge)
    # the stop rule is the context's setting alone: 0 = the paper's loop (lag 0); the default = C21's (lag 1), run here
    # with the separate check because this lattice's blocks straddle timeslices (the fused kernels do not apply)
    for monitor, lag in ((0, 0), (1, 1)):
        gfm.gf_set_monitor(fx.ctx, monitor)
        fx.load(U)
        n, th, F = fx.fix(1e-10, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=10, max_sweeps=2000)
        ref = U.copy()
        n_ref, th_ref, F_ref = oracle.fix(ref, dims, oracle.UPDATE_OVERRELAX2, 1.6, 1e-10, 10, 2000, 0, ORC_GAUGE[gauge], lag=lag)
        assert n == n_ref and 0 < n < 2000 and th < 1e-10
        assert th == pytest.approx(th_ref, rel=1e-6) and F == pytest.approx(F_ref, rel=1e-10)
        assert gfm.gf_fix_last_form(fx.ctx) == (lag, 0)
        assert np.abs(fx.download() - ref).max() < 1e-9
    if gauge == "coulomb":
        assert max(fx.theta_slices()) == th
    # cut by max_sweeps; zero sweeps when already fixed
    assert fx.fix(1e-10, max_sweeps=50)[0] == 0
    assert fx.fix(0.0, check_every=7, max_sweeps=10)[0] == 10
    with pytest.raises(gfm.GFError):
        fx.fix(1e-10, check_every=0)
    fx.close()


def test_fix_config1_fp32_and_stochastic(gfm):
    dims = (4, 4, 4, 4)
    U = gf_inputs.trivial_orbit(dims, 1)
    fx = gfm.GaugeFixer(dims, precision="fp32")
    fx.load(U)
    n, th, F = fx.fix(1e-11, gfm.GF_UPDATE_STOCHASTIC, 0.6, check_every=5, max_sweeps=1000, seed=3)
    assert n < 1000 and th < 1e-11 and abs(F - 1) < 1e-5
    fx.close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_fix_slices_matches_oracle(gfm, precision):
    """Coulomb gauge, stop rule per timeslice (C20): gf_fix_slices vs orc_fix_slices -- the same sweeps for every
    slice (fp64), every slice below the tolerance, links of the fp64 run within the N-sweep growth of 1e-12"""
    dims = (6, 6, 6, 8)
    U = gf_inputs.smooth_random(dims, 0.5, 45)
    fx = gfm.GaugeFixer(dims, precision=precision, gauge="coulomb")
    tol = 1e-9 if precision == "fp64" else 1e-8
    if precision == "fp64":  # the default rule (lag 1, C21) with the separate check: blocks straddle timeslices here
        fx.load(U)
        n, th, F, per = fx.fix_slices(tol, gfm.GF_UPDATE_OVERRELAX2, 1.5, check_every=5, max_sweeps=3000)
        ref = U.copy()
        n_ref, th_ref, F_ref, per_ref = oracle.fix_slices(ref, dims, oracle.UPDATE_OVERRELAX2, 1.5, tol, 5, 3000, lag=1)
        assert gfm.gf_fix_last_form(fx.ctx) == (1, 0)
        assert per == per_ref.tolist() and n == n_ref and len(set(per)) > 1
        assert th == pytest.approx(th_ref, rel=1e-5) and F == pytest.approx(F_ref, rel=1e-10)
        assert np.abs(fx.download() - ref).max() < 1e-9
    gfm.gf_set_monitor(fx.ctx, 0)  # the paper's rule
    fx.load(U)
    n, th, F, per = fx.fix_slices(tol, gfm.GF_UPDATE_OVERRELAX2, 1.5, check_every=5, max_sweeps=3000)
    n_ref, th_ref, F_ref, per_ref = oracle.fix_slices(U, dims, oracle.UPDATE_OVERRELAX2, 1.5, tol, 5, 3000)
    sl = fx.theta_slices()
    assert max(sl) < tol and th == max(sl) and n == max(per) and len(set(per)) > 1
    if precision == "fp64":
        assert per == per_ref.tolist() and n == n_ref
        assert th == pytest.approx(th_ref, rel=1e-5) and F == pytest.approx(F_ref, rel=1e-10)
        assert np.abs(fx.download() - U).max() < 1e-9
    else:
        assert abs(n - n_ref) <= 10 and F == pytest.approx(F_ref, rel=1e-5)
    assert fx.fix_slices(tol, check_every=5)[0] == 0  # already fixed
    fx.close()
    lx = gfm.GaugeFixer(dims, precision=precision, gauge="landau")
    with pytest.raises(gfm.GFError):
        lx.fix_slices(1e-9)
    lx.close()


def test_convert_and_mixed_precision_fixing(gfm):
    """gf_convert: fp64 -> fp32 rounds like gf_pack, fp32 -> fp64 re-orthonormalises in fp64, R18 <-> R12 rebuilds row 2; fp32 sweeps
    followed by an fp64 polish reach theta < 1e-13 in few fp64 sweeps and the same maximum as the pure fp64 run"""
    dims = (8, 8, 8, 8)
    U = gf_inputs.smooth_random(dims, 0.3, 55)
    a = gfm.GaugeFixer(dims, precision="fp64")
    a.load(U)
    b = a.convert_to(precision="fp32", reals_per_link=12)
    c = gfm.GaugeFixer(dims, precision="fp32", reals_per_link=12)
    c.load(U)
    assert np.array_equal(b.download(), c.download())
    d = b.convert_to(precision="fp64", reals_per_link=18)
    wide = d.download()
    assert np.abs(wide - b.download()).max() < 1e-6
    uu, det = oracle.unitarity_defect(wide, dims)
    assert uu < 1e-14 and det < 1e-14
    c.close(); d.close()
    # mixed precision
    n32, th32, _ = b.fix(1e-9, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=10, max_sweeps=5000)
    e = b.convert_to(precision="fp64", reals_per_link=18)
    n64, th64, F_mixed = e.fix(1e-13, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=10, max_sweeps=5000)
    n_pure, th_pure, F_pure = a.fix(1e-13, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=10, max_sweeps=5000)
    assert th32 < 1e-9 and th64 < 1e-13 and th_pure < 1e-13
    assert n64 < n_pure / 2 and n32 + n64 <= n_pure + 40
    assert F_mixed == pytest.approx(F_pure, rel=1e-6)
    got = e.download()
    uu, det = oracle.unitarity_defect(got, dims)
    assert uu < 1e-12 and det < 1e-12  # widening re-orthonormalised the links
    assert abs(oracle.plaquette(got, dims) - oracle.plaquette(U, dims)) < 1e-5
    with pytest.raises(gfm.GFError):
        other = gfm.gf_create(4, 4, 4, 4)
        try:
            gfm.gf_convert(a.ctx, a.U, other, a.U)
        finally:
            gfm.gf_destroy(other)
    a.close(); b.close(); e.close()


@pytest.mark.parametrize("precision,tol", [("fp32", 2e-5), ("fp64", 1e-12)])
def test_r12_stays_unitary_under_hot_updates(gfm, precision, tol):
    """12-real storage feeds norm errors of rows 0,1 back through the rebuilt row: without re-orthonormalisation
    they grow exponentially under large rotations (measured: fp32 heatbath at T = 1 reaches O(1) after 60 sweeps,
    fp64 diverges within a 200-step annealing).  With the automatic policy the links stay unitary and the plaquette
    invariant; switching the policy off shows the growth."""
    dims = (8, 8, 8, 8)
    U = gf_inputs.smooth_random(dims, 0.4, 56)
    P0 = oracle.plaquette(U, dims)
    fx = gfm.GaugeFixer(dims, precision=precision, reals_per_link=12)
    fx.load(U)
    fx.anneal(1.0, 1.0, 60, 7)
    fx.relax(gfm.GF_UPDATE_STOCHASTIC, 1.0, 40, 3)
    fx.anneal(1.4, 0.01, 100, 8, n_micro=1)
    got = fx.download()
    uu, det = oracle.unitarity_defect(got, dims)
    assert uu < tol and det < tol
    assert abs(oracle.plaquette(got, dims) - P0) < 20 * tol
    gfm.gf_set_reunit(fx.ctx, 0)  # never: the instability shows
    fx.load(U)
    fx.anneal(1.0, 1.0, 60, 7)
    uu_off, _ = oracle.unitarity_defect(fx.download(), dims)
    assert uu_off > 1e3 * tol
    fx.close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("R", [18, 12])
@pytest.mark.parametrize("tps", [0, 1, 2, 4])
def test_coulomb_reading_b_matches_reading_a_and_oracle(gfm, precision, R, tps):
    """C12 reading B (temporal links transformed once per call from the accumulated g(x)) against the oracle
    (reading A): one sweep within the per-link tolerance, several sweeps and the other update kinds within its
    growth; spatial links bit-identical to reading A of the CUDA path (same arithmetic, they never see G)"""
    dims = (8, 6, 4, 10)
    U = gf_inputs.smooth_random(dims, 0.4, 57)
    tol = TOL_LINK[precision]
    a = gfm.GaugeFixer(dims, precision=precision, gauge="coulomb", reals_per_link=R)
    b = gfm.GaugeFixer(dims, precision=precision, gauge="coulomb", reals_per_link=R)
    for fx in (a, b):
        gfm.gf_set_tuning(fx.ctx, tps, 0 if tps == 0 else 64)
        fx.load(U)
    gfm.gf_set_coulomb_reading(a.ctx, False)
    gfm.gf_set_coulomb_reading(b.ctx, True)
    ref = U.copy()
    a.overrelax(1.7, 1); b.overrelax(1.7, 1)
    oracle.overrelax(ref, dims, 1.7, 1, oracle.COULOMB)
    ga, gb = a.download(), b.download()
    # same launch shape: same arithmetic on the spatial links (automatic shape differs between the readings in fp32)
    same_shape = tps != 0
    assert np.array_equal(ga[:, :3], gb[:, :3]) if same_shape else np.abs(ga - gb).max() <= 2 * tol
    assert np.abs(gb - ref).max() <= tol
    a.overrelax(1.7, 4); b.overrelax(1.7, 4)
    a.relax(gfm.GF_UPDATE_STOCHASTIC, 0.4, 2, seed=5); b.relax(gfm.GF_UPDATE_STOCHASTIC, 0.4, 2, seed=5)
    a.relax(gfm.GF_UPDATE_OVERRELAX1, 1.5, 2); b.relax(gfm.GF_UPDATE_OVERRELAX1, 1.5, 2)
    ga, gb = a.download(), b.download()
    assert np.abs(ga - gb).max() <= 20 * tol
    if same_shape:
        assert np.array_equal(ga[:, :3], gb[:, :3])
        assert b.functional() == a.functional() and b.theta() == a.theta()  # F, theta do not see the temporal links
    assert abs(oracle.plaquette(gb, dims) - oracle.plaquette(U, dims)) < (1e-12 if precision == "fp64" else 2e-5)
    a.close(); b.close()


def test_coulomb_reading_b_with_fix_slices_and_errors(gfm):
    dims = (6, 6, 6, 8)
    U = gf_inputs.smooth_random(dims, 0.5, 45)
    fx = gfm.GaugeFixer(dims, precision="fp64", gauge="coulomb")
    gfm.gf_set_coulomb_reading(fx.ctx, True)
    gfm.gf_set_monitor(fx.ctx, 0)  # the paper's stop rule
    fx.load(U)
    n, th, F, per = fx.fix_slices(1e-9, gfm.GF_UPDATE_OVERRELAX2, 1.5, check_every=5, max_sweeps=3000)
    n_ref, th_ref, F_ref, per_ref = oracle.fix_slices(U, dims, oracle.UPDATE_OVERRELAX2, 1.5, 1e-9, 5, 3000)
    assert per == per_ref.tolist() and F == pytest.approx(F_ref, rel=1e-10)
    assert np.abs(fx.download() - U).max() < 1e-9
    fx.close()
    lx = gfm.GaugeFixer(dims, precision="fp64", gauge="landau")
    with pytest.raises(gfm.GFError):
        gfm.gf_set_coulomb_reading(lx.ctx, True)
    lx.close()


@pytest.mark.parametrize("R,tps", [(18, 0), (18, 1), (12, 2), (18, 4)])
def test_coulomb_reading_b_annealing_decisions_fp64(gfm, R, tps):
    """annealing (heatbath + microcanonical sweeps) under reading B: the draw never sees the temporal links, so the
    accept decisions are those of the oracle (reading A) and the links agree to rounding"""
    import torch

    dims = (6, 4, 4, 8)
    V = int(np.prod(dims))
    U = gf_inputs.smooth_random(dims, 0.5, 58)
    fx = gfm.GaugeFixer(dims, precision="fp64", gauge="coulomb", reals_per_link=R)
    gfm.gf_set_tuning(fx.ctx, tps, 0 if tps == 0 else 64)
    gfm.gf_set_coulomb_reading(fx.ctx, True)
    trials = torch.zeros(V * 3, dtype=torch.int32, device="cuda")
    gfm.gf_set_trial_buffer(fx.ctx, trials)
    fx.load(U)
    fx.anneal(1.2, 0.3, 3, 7, n_micro=1)
    ref_trials = oracle.anneal_micro(U, dims, 1.2, 0.3, 3, 1, 7, oracle.COULOMB, trials=True)
    assert np.array_equal(trials.cpu().numpy().reshape(V, 3), ref_trials)
    assert np.abs(fx.download() - U).max() <= 1e-10
    fx.close()


def _degenerate_field(dims):
    """U_mu(y) = 1 on even sites, diag(-1,-1,1) on odd sites: K(x) = 4 (1 + D) = diag(0,0,8) at every site, so the
    (0,1) block of K vanishes identically (the |k| = 0 guard of C9) while (0,2) and (1,2) give g = 1"""
    V = int(np.prod(dims))
    s = np.arange(V)
    x = s % dims[0] + (s // dims[0]) % dims[1] + (s // (dims[0] * dims[1])) % dims[2] + s // (dims[0] * dims[1] * dims[2])
    U = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    U[:, :, 0, 0] = U[:, :, 1, 1] = np.where(x % 2 == 0, 1.0, -1.0)[:, None]
    U[:, :, 2, 2] = 1.0
    return U


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_degenerate_block_and_empty_calls(gfm, precision):
    import torch

    dims = (4, 4, 2, 6)
    V = int(np.prod(dims))
    U = _degenerate_field(dims)
    ref = U.copy()
    oracle.overrelax(ref, dims, 1.7, 2)
    assert np.array_equal(ref, U)  # the oracle takes G = 1 in the vanishing block and g = 1 in the others
    fx = gfm.GaugeFixer(dims, precision=precision)
    gfm.gf_set_reunit(fx.ctx, 0)
    fx.load(U)
    fx.overrelax(1.7, 2)
    fx.relax(gfm.GF_UPDATE_OVERRELAX1, 1.5, 1)
    fx.relax(gfm.GF_UPDATE_STOCHASTIC, 0.5, 1, seed=3)
    assert np.array_equal(fx.download(), U)
    assert fx.theta() == 0.0 and fx.functional() == pytest.approx(1.0 / 3.0, abs=1e-15)
    # heatbath: the vanishing block takes no trial (count 0) on both sides
    trials = torch.zeros(V * 3, dtype=torch.int32, device="cuda")
    gfm.gf_set_trial_buffer(fx.ctx, trials)
    fx.anneal(0.7, 0.7, 1, 7)
    got = trials.cpu().numpy().reshape(V, 3)
    work = U.copy()
    ref_tr = oracle.anneal(work, dims, 0.7, 0.7, 1, 7, trials=True)
    red = np.array([(s % 4 + (s // 4) % 4 + (s // 16) % 2 + s // 32) % 2 == 0 for s in range(V)])
    assert (got[red, 0] == 0).all() and (ref_tr[red, 0] == 0).all()  # RED sites see the untouched degenerate K
    # empty calls leave every bit alone
    fx.load(U)
    fx.overrelax(1.7, 0)
    fx.relax(gfm.GF_UPDATE_STOCHASTIC, 0.5, 0)
    fx.anneal(1.0, 0.5, 0, 1)
    assert fx.fix(1e-30, max_sweeps=0)[0] == 0
    assert np.array_equal(fx.download(), U)
    fx.close()


@pytest.mark.parametrize("precision,R,gauge", [("fp32", 18, "landau"), ("fp32", 12, "coulomb"), ("fp64", 18, "coulomb"),
                                               ("fp64", 12, "landau")])
def test_no_write_outside_the_field(gfm, precision, R, gauge):
    """compute-sanitizer is closed on this pool: guard bands of a sentinel pattern before and after the native field
    (and around the canonical buffer) must survive every kernel -- pack, all sweep kinds with every launch shape on a
    lattice with a ragged last warp, reductions, convert, unpack"""
    import torch

    dims = (6, 2, 6, 10)  # V/2 = 360: ragged for 32-thread blocks at 1, 2 and 4 threads per site
    V = int(np.prod(dims))
    U = gf_inputs.smooth_random(dims, 0.4, 59)
    prec = gfm.GF_FP64 if precision == "fp64" else gfm.GF_FP32
    ctx = gfm.gf_create(*dims, prec, gfm.GF_COULOMB if gauge == "coulomb" else gfm.GF_LANDAU)
    gfm.gf_set_storage(ctx, R)
    nbytes = gfm.gf_field_bytes(ctx)
    band = 1 << 16
    buf = torch.full((nbytes + 2 * band,), 0xA5, dtype=torch.uint8, device="cuda")
    field = buf[band:band + nbytes]
    assert field.data_ptr() % 256 == 0
    cbuf = torch.full((V * 72 + 2 * 8192,), float("nan"), dtype=torch.float64, device="cuda")
    canon = cbuf[8192:8192 + V * 72]
    canon.copy_(torch.from_numpy(U.view("float64").reshape(-1)))
    gfm.gf_pack(ctx, canon, field)
    for tps in (0, 1, 2, 4):
        for block in ((0,) if tps == 0 else (32, 96)):
            gfm.gf_set_tuning(ctx, tps, block)
            gfm.gf_set_prefetch(ctx, 100)
            gfm.gf_overrelax(ctx, field, 1.7, 2)
            gfm.gf_relax(ctx, field, gfm.GF_UPDATE_STOCHASTIC, 0.5, 1, 3)
            gfm.gf_relax(ctx, field, gfm.GF_UPDATE_OVERRELAX1, 1.4, 1, 0)
            gfm.gf_anneal_micro(ctx, field, 1.0, 0.5, 2, 1, 7)
            for chain in (0, 1, 2):  # fp32: every precision of the site chain
                gfm.gf_set_chain(ctx, chain)
                gfm.gf_overrelax(ctx, field, 1.7, 3)
                gfm.gf_anneal(ctx, field, 0.7, 0.7, 1, 9)
    gfm.gf_functional(ctx, field)
    gfm.gf_theta(ctx, field)
    if gauge == "coulomb":
        gfm.gf_fix_slices(ctx, field, dims[3], gfm.GF_UPDATE_OVERRELAX2, 1.5, 1e-3, 2, 6)
    gfm.gf_unpack(ctx, field, canon)
    torch.cuda.synchronize()
    assert bool((buf[:band] == 0xA5).all()) and bool((buf[band + nbytes:] == 0xA5).all())
    assert bool(torch.isnan(cbuf[:8192]).all()) and bool(torch.isnan(cbuf[8192 + V * 72:]).all())
    assert not bool(torch.isnan(canon).any())
    gfm.gf_destroy(ctx)


# ---------------------------------------------------------------------------------------------------------
# fused F / theta monitor of the fixing loops (C21)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision,gauge,R", [("fp64", "landau", 18), ("fp64", "coulomb", 18), ("fp64", "landau", 12),
                                               ("fp32", "landau", 18), ("fp32", "coulomb", 18)])
def test_fused_monitor_values_match_the_oracle(gfm, precision, gauge, R):
    """theta, theta_t and F that the sweep kernels accumulate for the state after sweep n are those of orc_theta /
    orc_functional on that state: fp64 theta 1e-6 (measured 1e-12), F 1e-10; fp32 within its storage rounding"""
    dims = (8, 8, 8, 8)  # (V_s / 2) * threads per site divisible by the 32-thread block: the fused form applies
    U = gf_inputs.smooth_random(dims, 0.4, 61)
    og = ORC_GAUGE[gauge]
    fx = gfm.GaugeFixer(dims, precision=precision, gauge=gauge, reals_per_link=R)
    fx.load(U)
    # a tolerance out of reach in 9 sweeps (fp32: the smallest the fused form takes); checks after sweeps 3 and 6 (none
    # at the last allowed sweep 9: it needs sweep 10)
    n, th_end, F_end = fx.fix(0.0 if precision == "fp64" else 1e-10, gfm.GF_UPDATE_OVERRELAX2, 1.7, check_every=3, max_sweeps=9)
    assert n == 9
    k, th, F, th_t = gfm.gf_monitor_last(fx.ctx, dims[3])
    assert k == 6
    ref = U.copy()
    oracle.overrelax(ref, dims, 1.7, 6, og)
    tol_th, tol_F = (1e-6, 1e-10) if precision == "fp64" else (2e-3, 1e-5)
    assert th == pytest.approx(oracle.theta(ref, dims, og), rel=tol_th)
    assert F == pytest.approx(oracle.functional(ref, dims, og), rel=tol_F)
    if gauge == "coulomb":
        np.testing.assert_allclose(th_t, oracle.theta_slices(ref, dims, og), rtol=tol_th)
    oracle.overrelax(ref, dims, 1.7, 3, og)
    assert th_end == pytest.approx(oracle.theta(ref, dims, og), rel=1e-6 if precision == "fp64" else 2e-2)
    assert F_end == pytest.approx(oracle.functional(ref, dims, og), rel=tol_F)
    assert np.abs(fx.download() - ref).max() <= (1e-11 if precision == "fp64" else 3e-4)
    fx.close()


@pytest.mark.parametrize("gauge", ["landau", "coulomb"])
@pytest.mark.parametrize("every", [1, 7])
def test_fused_fix_loop_matches_oracle_with_lag_one(gfm, gauge, every):
    """gf_fix with the fused monitor ends one sweep after the check that met the tolerance (orc_fix_lag, lag = 1);
    the separate check kernel (gf_set_monitor 0) is the paper's loop (lag = 0); bit-identical fields between the fused
    loop and plain sweeping for the same number of sweeps"""
    dims = (8, 8, 8, 8)
    U = gf_inputs.smooth_random(dims, 0.3, 62)
    og = ORC_GAUGE[gauge]
    fx = gfm.GaugeFixer(dims, precision="fp64", gauge=gauge)
    fx.load(U)
    n, th, F = fx.fix(1e-9, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=every, max_sweeps=3000)
    ref = U.copy()
    n_ref, th_ref, F_ref = oracle.fix(ref, dims, oracle.UPDATE_OVERRELAX2, 1.6, 1e-9, every, 3000, 0, og, lag=1)
    assert n == n_ref and 0 < n < 3000
    assert th == pytest.approx(th_ref, rel=1e-5) and F == pytest.approx(F_ref, rel=1e-10)
    got = fx.download()
    assert np.abs(got - ref).max() < 1e-9
    assert fx.fix(1e-9, check_every=every)[0] == 0  # already fixed: no sweep
    fx.load(U)
    fx.overrelax(1.6, n)
    assert np.array_equal(fx.download(), got)  # the monitor changes no link
    gfm.gf_set_monitor(fx.ctx, 0)
    fx.load(U)
    n0 = fx.fix(1e-9, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=every, max_sweeps=3000)[0]
    ref = U.copy()
    assert n0 == oracle.fix(ref, dims, oracle.UPDATE_OVERRELAX2, 1.6, 1e-9, every, 3000, 0, og, lag=0)[0] == n - 1
    # cut by max_sweeps: the check at the last allowed sweep cannot take place
    gfm.gf_set_monitor(fx.ctx, 1)
    fx.load(U)
    assert fx.fix(1e-9, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=every, max_sweeps=n - 1)[0] == n - 1
    fx.close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_fused_fix_slices_matches_oracle_with_lag_one(gfm, precision):
    """Coulomb gauge, per-timeslice stop rule with the fused monitor: a slice found below the tolerance after sweep n is
    frozen from sweep n + 2 on (orc_fix_slices_lag, lag = 1); with check_every = 1 every slice stops within one sweep of
    meeting the tolerance"""
    dims = (8, 8, 8, 6)
    U = gf_inputs.smooth_random(dims, 0.5, 63)
    fx = gfm.GaugeFixer(dims, precision=precision, gauge="coulomb")
    fx.load(U)
    tol = 1e-9 if precision == "fp64" else 1e-8
    n, th, F, per = fx.fix_slices(tol, gfm.GF_UPDATE_OVERRELAX2, 1.5, check_every=1, max_sweeps=3000)
    ref = U.copy()
    n_ref, th_ref, F_ref, per_ref = oracle.fix_slices(ref, dims, oracle.UPDATE_OVERRELAX2, 1.5, tol, 1, 3000, lag=1)
    sl = fx.theta_slices()
    assert max(sl) < tol and n == max(per) and len(set(per)) > 1
    if precision == "fp64":
        assert per == per_ref.tolist() and n == n_ref
        assert th == pytest.approx(th_ref, rel=1e-5) and F == pytest.approx(F_ref, rel=1e-10)
        assert np.abs(fx.download() - ref).max() < 1e-9
        ref0 = U.copy()
        per0 = oracle.fix_slices(ref0, dims, oracle.UPDATE_OVERRELAX2, 1.5, tol, 1, 3000, lag=0)[3]
        assert per == (per0 + 1).tolist()  # one sweep past the crossing, per slice
    else:
        assert np.abs(np.array(per) - per_ref).max() <= 3 and F == pytest.approx(F_ref, rel=1e-5)
    assert fx.fix_slices(tol, check_every=1)[0] == 0
    fx.close()


def test_fused_monitor_F_counts_slices_frozen_before_the_first_sweep(gfm):
    """gf_monitor_last after gf_fix_slices on a field with one timeslice already fixed at the start (its spatial links
    are unit matrices: theta_t = 0): that slice is never swept, and the monitor's F must still contain its share"""
    dims = (8, 8, 8, 6)
    Vs = dims[0] * dims[1] * dims[2]
    U = gf_inputs.smooth_random(dims, 0.5, 66)
    U[2 * Vs:3 * Vs, :3] = np.eye(3)  # timeslice t = 2, mu = x, y, z
    fx = gfm.GaugeFixer(dims, precision="fp64", gauge="coulomb")
    fx.load(U)
    assert fx.theta_slices()[2] == 0.0
    n, th, F, per = fx.fix_slices(1e-30, gfm.GF_UPDATE_OVERRELAX2, 1.5, check_every=2, max_sweeps=6)
    assert gfm.gf_fix_last_form(fx.ctx) == (1, 1) and n == 6 and per == [6, 6, 0, 6, 6, 6]
    k, th_k, F_k, th_t = gfm.gf_monitor_last(fx.ctx, dims[3])
    assert k == 4  # checks after sweeps 2 and 4; none at the last allowed sweep
    ref = U.copy()
    oracle.fix_slices(ref, dims, oracle.UPDATE_OVERRELAX2, 1.5, 1e-30, 2, 4, lag=1)
    assert F_k == pytest.approx(oracle.functional(ref, dims, oracle.COULOMB), rel=1e-10)
    np.testing.assert_allclose(th_t, oracle.theta_slices(ref, dims, oracle.COULOMB), rtol=1e-6, atol=1e-30)
    assert th_t[2] == 0.0 and th_k == pytest.approx(oracle.theta(ref, dims, oracle.COULOMB), rel=1e-6)
    fx.close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("every", [1, 4, 25])
def test_fix_result_does_not_depend_on_the_launch_shape(gfm, precision, every):
    """gf_fix: the same arguments give the same sweeps_done and the same field whatever gf_set_tuning picked -- with the
    default shape the fused monitor runs (check_every <= 10), with a 96-thread block its blocks straddle timeslices and
    the separate check runs, under the same stop rule (lag 1, from the context's gf_set_monitor setting alone); with
    check_every = 25 both shapes take the separate check.  fp64: bit-identical fields; fp32: the hybrid chain's
    roughness history differs between a 32- and a 1-sweep batch of launches, so fields agree to the fp32 tolerance."""
    dims = (8, 8, 8, 8)
    U = gf_inputs.smooth_random(dims, 0.3, 65)
    tol = 1e-9 if precision == "fp64" else 1e-8
    out = []
    for block in (0, 96, 64):
        fx = gfm.GaugeFixer(dims, precision=precision)
        gfm.gf_set_tuning(fx.ctx, 0, block)
        fx.load(U)
        n, th, F = fx.fix(tol, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=every, max_sweeps=3000)
        out.append((n, gfm.gf_fix_last_form(fx.ctx), fx.download(), th))
        fx.close()
    assert out[0][1] == (1, 1 if every <= 10 else 0) and out[1][1] == (1, 0)
    assert 0 < out[0][0] < 3000 and out[0][3] < tol
    for n, form, field, th in out[1:]:
        assert form[0] == 1
        if precision == "fp64":
            assert n == out[0][0] and np.array_equal(field, out[0][2])
        else:
            assert abs(n - out[0][0]) <= every and th < tol
    ref = U.copy()
    n_ref = oracle.fix(ref, dims, oracle.UPDATE_OVERRELAX2, 1.6, tol, every, 3000, lag=1)[0]
    if precision == "fp64":
        assert out[0][0] == n_ref and np.abs(out[0][2] - ref).max() < 1e-9


def test_fused_monitor_stochastic_and_fallback(gfm):
    """the variants run under the monitor too (stochastic relaxation: decisions continue through the loop, C18); a
    lattice whose blocks straddle timeslices falls back to the separate check and keeps the context's stop rule (lag 1)"""
    dims = (8, 8, 8, 4)
    U = gf_inputs.smooth_random(dims, 0.3, 64)
    fx = gfm.GaugeFixer(dims, precision="fp64")
    fx.load(U)
    n, th, F = fx.fix(1e-8, gfm.GF_UPDATE_STOCHASTIC, 0.5, check_every=2, max_sweeps=3000, seed=5)
    ref = U.copy()
    n_ref, th_ref, F_ref = oracle.fix(ref, dims, oracle.UPDATE_STOCHASTIC, 0.5, 1e-8, 2, 3000, 5, lag=1)
    assert n == n_ref and F == pytest.approx(F_ref, rel=1e-10) and np.abs(fx.download() - ref).max() < 1e-9
    fx.close()
    dims = (6, 6, 6, 4)  # V_s / 2 = 108 sites, two threads per site: 216 threads do not fill 32-thread blocks evenly
    U = gf_inputs.smooth_random(dims, 0.3, 54)
    fx = gfm.GaugeFixer(dims, precision="fp64")
    fx.load(U)
    n = fx.fix(1e-9, gfm.GF_UPDATE_OVERRELAX2, 1.6, check_every=3, max_sweeps=2000)[0]
    ref = U.copy()
    assert n == oracle.fix(ref, dims, oracle.UPDATE_OVERRELAX2, 1.6, 1e-9, 3, 2000, lag=1)[0]
    assert gfm.gf_fix_last_form(fx.ctx) == (1, 0) and np.abs(fx.download() - ref).max() < 1e-9
    with pytest.raises(gfm.GFError):
        gfm.gf_monitor_last(fx.ctx, 4)
    fx.close()


# ---------------------------------------------------------------------------------------------------------
# the fp64 annealing draw's own log / sin / cos (branch-free, for 24-bit uniforms) over their WHOLE domain
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.gpu
def test_kp_double_math_over_all_uniforms(gfm):
    """kp_neglog_word / kp_sincos2pi_word (gf_device.cuh) against numpy on every one of the 2^23 uniforms
    u = (2m + 1) 2^-24: -ln u to 4e-16 relative (also as u -> 1, where it falls to 6e-8), sine and cosine to 5e-16
    absolute.  The reference reduces the angle exactly (4u = q + r) before it calls numpy, so that it carries no
    argument-rounding error of its own."""
    import torch

    m = np.arange(2**23, dtype=np.uint64)
    words = torch.from_numpy((m << 9).astype(np.uint32).view(np.int32)).cuda()  # x >> 9 = m
    nl = torch.empty(m.size, dtype=torch.float64, device="cuda")
    sn, cs = torch.empty_like(nl), torch.empty_like(nl)
    gfm.gf_debug_kp_math(words, nl, sn, cs)
    torch.cuda.synchronize()
    w = 2 * m + 1
    u = w.astype(np.float64) / 2.0**24
    # -ln u: log1p(u - 1) is the accurate form near 1 (u - 1 is exact)
    ref = np.where(u > 0.5, -np.log1p(u - 1.0), -np.log(u))
    rel = np.abs(nl.cpu().numpy() - ref) / ref
    assert rel.max() <= 4e-16, (rel.max(), int(rel.argmax()))
    q = (w + 2**21) >> 22
    r = (w.astype(np.int64) - (q.astype(np.int64) << 22)).astype(np.float64) / 2.0**22
    s0, c0 = np.sin(0.5 * np.pi * r), np.cos(0.5 * np.pi * r)
    qq = (q & 3).astype(np.int64)
    ref_s = np.choose(qq, [s0, c0, -s0, -c0])
    ref_c = np.choose(qq, [c0, -s0, -c0, s0])
    assert np.abs(sn.cpu().numpy() - ref_s).max() <= 5e-16
    assert np.abs(cs.cpu().numpy() - ref_c).max() <= 5e-16
    # a spot check against the plain definition, argument rounding included
    assert np.abs(cs.cpu().numpy()[::4097] - np.cos(2 * np.pi * u[::4097])).max() <= 2e-15
