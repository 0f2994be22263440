"""Pins of the oracle's update variants (readings C17-C19): first-order overrelaxation, stochastic
relaxation, microcanonical sweeps.  Each against a closed form, an invariant or an independent restatement."""
import numpy as np
import pytest

import gf_inputs
import oracle

import np_lattice as npl


def _unit_quat(rng):
    q = rng.normal(size=4)
    return q / np.linalg.norm(q)


def _exact_power(g, w):
    """exact g^w of the SU(2) element g = (cos phi, sin phi n)"""
    phi = np.arccos(np.clip(g[0], -1, 1))
    n = g[1:] / max(np.linalg.norm(g[1:]), 1e-300)
    return np.concatenate([[np.cos(w * phi)], np.sin(w * phi) * n])


def test_first_order_closed_forms():
    """C17: h = g at omega = 1; direction of hvec unchanged; matches exact g^omega to O(phi^2):
    |h - g^w| <= w (w - 1) / 2 * phi^2 (1 + O(phi)) for small rotation angle phi"""
    rng = np.random.default_rng(1)
    for _ in range(50):
        g = _unit_quat(rng)
        assert np.allclose(oracle.su2_overrelax1(g, 1.0), g, atol=1e-15)
        h = oracle.su2_overrelax1(g, 1.6)
        assert abs(np.linalg.norm(h) - 1) < 1e-15
        assert np.allclose(np.cross(h[1:], g[1:]), 0, atol=1e-15) and np.dot(h[1:], g[1:]) > 0
    for phi in (1e-3, 1e-2, 5e-2):
        n = _unit_quat(rng)[1:]
        n /= np.linalg.norm(n)
        g = np.concatenate([[np.cos(phi)], np.sin(phi) * n])
        for w in (1.3, 1.7, 1.9):
            err = np.linalg.norm(oracle.su2_overrelax1(g, w) - _exact_power(g, w))
            # after normalisation the first-order form is a rotation by atan(w tan(phi) / ...) ~ w phi (1 + O(phi^2)):
            # the angle error is cubic, bounded by w (w^2 - 1) / 3 * phi^3
            assert err <= w * (w * w - 1) / 3 * phi**3 * 1.5 + 1e-15
    # explicit value: g0 = 0, omega = 1.5: h = (1 - 1.5, 1.5 gvec) / sqrt(0.25 + 2.25)
    g = np.array([0.0, 0.0, 1.0, 0.0])
    assert np.allclose(oracle.su2_overrelax1(g, 1.5), np.array([-0.5, 0, 1.5, 0]) / np.sqrt(2.5), atol=1e-15)


def test_square_is_exact_double_rotation():
    """C18/C19: g^2 equals the exact power at omega = 2 and the quaternion product g (x) g"""
    rng = np.random.default_rng(2)
    for _ in range(50):
        g = _unit_quat(rng)
        sq = oracle.su2_square(g)
        assert np.allclose(sq, oracle.quat_mul(g, g), atol=1e-15)
        assert np.allclose(sq, _exact_power(g, 2.0), atol=1e-12)
        assert np.allclose(sq, oracle.su2_overrelax(g, 2.0), atol=1e-14)  # the 2nd-order form is exact at omega = 2


@pytest.mark.parametrize("gauge,nd", [(oracle.LANDAU, 4), (oracle.COULOMB, 3)])
def test_microcanonical_sweeps_conserve_F(gauge, nd):
    """C19: g -> g^2 leaves Re tr[g K] at its old value in every subgroup step, so F is unchanged by whole sweeps
    (p = 1 stochastic relaxation); the field does change; plaquette and unitarity are preserved"""
    dims = (4, 6, 4, 4)
    U = gf_inputs.smooth_random(dims, 0.5, 41)
    U0 = U.copy()
    F0, P0 = npl.functional(U, dims, nd), npl.plaquette(U, dims)
    oracle.relax(U, dims, oracle.UPDATE_STOCHASTIC, 1.0, 3, 5, gauge)
    assert np.abs(U - U0).max() > 0.1
    assert abs(npl.functional(U, dims, nd) - F0) < 1e-13
    assert abs(npl.plaquette(U, dims) - P0) < 1e-13
    uu, det = oracle.unitarity_defect(U, dims)
    assert uu < 1e-13 and det < 1e-13


def test_stochastic_limits_and_rate():
    """C18: p = 0 is plain relaxation (omega = 1, up to the renormalisation rounding of the latter); decisions follow the stated Philox recipe and their
    rate is p within 4 sigma; same seed -> same decisions, other seed -> others"""
    dims = (4, 4, 4, 6)
    V = int(np.prod(dims))
    U = gf_inputs.smooth_random(dims, 0.4, 42)
    a, b = U.copy(), U.copy()
    oracle.relax(a, dims, oracle.UPDATE_STOCHASTIC, 0.0, 2, 9)
    oracle.overrelax(b, dims, 1.0, 2)
    assert np.abs(a - b).max() < 1e-13
    p = 0.3
    c = U.copy()
    sq = oracle.relax(c, dims, oracle.UPDATE_STOCHASTIC, p, 1, 9, squared=True)
    n = sq.size
    assert abs(sq.mean() - p) < 4 * np.sqrt(p * (1 - p) / n)
    # the recipe, restated: counter (site, sweep, parity << 2 | subgroup, 0x40000000), key = seed, first word
    for s in (0, 17, V - 1):
        x = s % 4 + (s // 4) % 4 + (s // 16) % 4 + s // 64
        for sub in range(3):
            w = oracle.philox4x32_10([s, 0, ((x & 1) << 2) | sub, 0x40000000], [9, 0])[0]
            u = (2 * (int(w) >> 9) + 1) / 2**24
            assert sq[s, sub] == int(u < p)
    d = U.copy()
    assert np.array_equal(oracle.relax(d, dims, oracle.UPDATE_STOCHASTIC, p, 1, 9, squared=True), sq)
    e = U.copy()
    assert not np.array_equal(oracle.relax(e, dims, oracle.UPDATE_STOCHASTIC, p, 1, 10, squared=True), sq)


def test_variants_converge_on_trivial_orbit():
    """first-order overrelaxation and stochastic relaxation are gauge-fixing algorithms: on the trivial orbit
    (config 1) theta -> 0 and F -> 1 (P1 for the variants)"""
    dims = (4, 4, 4, 4)
    U0 = gf_inputs.trivial_orbit(dims, 1)
    for update, param in ((oracle.UPDATE_OVERRELAX1, 1.3), (oracle.UPDATE_OVERRELAX1, 1.6),
                          (oracle.UPDATE_STOCHASTIC, 0.3), (oracle.UPDATE_STOCHASTIC, 0.7)):
        U = U0.copy()
        oracle.relax(U, dims, update, param, 300, 3)
        assert oracle.theta(U, dims) < 1e-14, (update, param)
        assert abs(oracle.functional(U, dims) - 1) < 1e-12, (update, param)


def test_second_order_variant_is_the_overrelax_call():
    dims = (4, 4, 2, 6)
    U = gf_inputs.smooth_random(dims, 0.4, 43)
    a, b = U.copy(), U.copy()
    oracle.relax(a, dims, oracle.UPDATE_OVERRELAX2, 1.7, 2, 0, oracle.COULOMB)
    oracle.overrelax(b, dims, 1.7, 2, oracle.COULOMB)
    assert np.array_equal(a, b)


def test_anneal_micro_reduces_to_anneal_and_conserves_between_heatbath():
    dims = (4, 4, 4, 4)
    U = gf_inputs.smooth_random(dims, 0.5, 44)
    a, b = U.copy(), U.copy()
    oracle.anneal_micro(a, dims, 1.0, 0.5, 3, 0, 7)
    oracle.anneal(b, dims, 1.0, 0.5, 3, 7)
    assert np.array_equal(a, b)
    # one heatbath sweep then 2 microcanonical sweeps: F equals F after the heatbath sweep alone
    c, d = U.copy(), U.copy()
    oracle.anneal_micro(c, dims, 0.8, 0.8, 1, 2, 7)
    oracle.anneal(d, dims, 0.8, 0.8, 1, 7)
    assert np.abs(c - d).max() > 0.05
    assert abs(npl.functional(c, dims, 4) - npl.functional(d, dims, 4)) < 1e-13


def test_fix_loop_config1_and_cadence():
    """Alg. 1 outer loop: config 1 (golden/config1_expectation.txt) stops below theta_tol with F = 1; the number of
    sweeps is the first multiple of check_every at which a sweep-by-sweep run is below the tolerance; max_sweeps
    cuts the last chunk; an already fixed field needs 0 sweeps"""
    dims = (4, 4, 4, 4)
    U0 = gf_inputs.trivial_orbit(dims, 1)
    U = U0.copy()
    first = None
    for n in range(1, 501):
        oracle.overrelax(U, dims, 1.7, 1)
        if oracle.theta(U, dims) < 1e-14:
            first = n
            break
    assert first is not None
    for every in (1, 7, 100):
        V = U0.copy()
        n, th, F = oracle.fix(V, dims, oracle.UPDATE_OVERRELAX2, 1.7, 1e-14, every, 500)
        assert n == -(-first // every) * every and th < 1e-14 and abs(F - 1) < 1e-12
    V = U0.copy()
    n, th, F = oracle.fix(V, dims, oracle.UPDATE_OVERRELAX2, 1.7, 1e-14, 7, 10)
    assert n == 10 and th == oracle.theta(V, dims) and F == oracle.functional(V, dims)
    n, th, F = oracle.fix(U, dims, oracle.UPDATE_OVERRELAX2, 1.7, 1e-14, 5, 10)
    assert n == 0


def test_fix_slices_freezes_timeslices_independently():
    """C20 (Coulomb, per-timeslice stop rule): every slice ends below the tolerance; slices need different numbers
    of sweeps; the spatial links of slice t are exactly those of plain all-slice sweeping after n_t sweeps (the
    slices decouple, C12); the result is still a gauge transform of the input (plaquette)"""
    dims = (6, 6, 6, 8)
    Vs = 6 * 6 * 6
    U0 = gf_inputs.smooth_random(dims, 0.5, 45)
    U = U0.copy()
    n, th, F, per = oracle.fix_slices(U, dims, oracle.UPDATE_OVERRELAX2, 1.5, 1e-9, 5, 3000)
    sl = oracle.theta_slices(U, dims, oracle.COULOMB)
    assert n == per.max() and n < 3000 and th == sl.max() and (sl < 1e-9).all()
    assert len(set(per.tolist())) > 1 and (per % 5 == 0).all() and per.min() > 0
    assert abs(npl.plaquette(U, dims) - npl.plaquette(U0, dims)) < 1e-12
    ref = U0.copy()
    done = 0
    for nt in sorted(set(per.tolist())):
        oracle.overrelax(ref, dims, 1.5, nt - done, oracle.COULOMB)
        done = nt
        for t in np.nonzero(per == nt)[0]:
            a = U[t * Vs:(t + 1) * Vs, :3]
            b = ref[t * Vs:(t + 1) * Vs, :3]
            assert np.array_equal(a, b), (t, nt)
    # nothing to do on a fixed field
    n2, _, _, per2 = oracle.fix_slices(U, dims, oracle.UPDATE_OVERRELAX2, 1.5, 1e-9, 5, 3000)
    assert n2 == 0 and per2.max() == 0


def test_fix_chunks_continue_the_stochastic_sweep_counter():
    """C18: inside the fixing loop the sweep counter of the stochastic decisions runs on through the chunks, so a
    chunked run is the unchunked run bit for bit (no decision is replayed) -- pinned against orc_relax, and the
    decisions of consecutive sweeps against the stated Philox recipe with counter word 1 = 0, 1, 2"""
    dims = (4, 4, 4, 6)
    V = int(np.prod(dims))
    U0 = gf_inputs.smooth_random(dims, 0.4, 44)
    p, seed, nsw = 0.4, 11, 6
    whole = U0.copy()
    oracle.relax(whole, dims, oracle.UPDATE_STOCHASTIC, p, nsw, seed)
    for every in (1, 2, 4):
        chunked = U0.copy()
        n, th, F = oracle.fix(chunked, dims, oracle.UPDATE_STOCHASTIC, p, 0.0, every, nsw, seed)  # tol 0: never stops
        assert n == nsw and np.array_equal(chunked, whole), every
    # relax_from(sweep0) takes the decisions of sweep sweep0 of the recipe, not those of sweep 0
    for sweep0 in (0, 1, 2):
        c = U0.copy()
        sq = oracle.relax_from(c, dims, oracle.UPDATE_STOCHASTIC, p, 1, sweep0, seed, squared=True)
        for s in (3, 40, V - 2):
            x = s % 4 + (s // 4) % 4 + (s // 16) % 4 + s // 64
            for sub in range(3):
                w = oracle.philox4x32_10([s, sweep0, ((x & 1) << 2) | sub, 0x40000000], [seed, 0])[0]
                assert sq[s, sub] == int((2 * (int(w) >> 9) + 1) / 2**24 < p)
    a, b = U0.copy(), U0.copy()
    sa = oracle.relax_from(a, dims, oracle.UPDATE_STOCHASTIC, p, 1, 0, seed, squared=True)
    sb = oracle.relax_from(b, dims, oracle.UPDATE_STOCHASTIC, p, 1, 1, seed, squared=True)
    assert not np.array_equal(sa, sb)


def test_heatbath_half_is_the_annealing_half_sweep():
    """orc_heatbath_half on RED then BLACK is one annealing step (same field, same trial counts); a half-sweep
    touches the trial counts of its own sublattice only and, by C6, no link twice"""
    dims = (4, 4, 2, 6)
    V = int(np.prod(dims))
    U0 = gf_inputs.smooth_random(dims, 0.5, 45)
    a = U0.copy()
    ta = oracle.anneal(a, dims, 0.9, 0.9, 1, 7, trials=True)
    b = U0.copy()
    tb = np.full((V, 3), -1, dtype=np.int32)
    oracle.heatbath_half(b, dims, 0.9, 7, 0, 0, trials=tb)
    s = np.arange(V)
    par = (s % 4 + (s // 4) % 4 + (s // 16) % 2 + s // 32) & 1
    assert (tb[par == 1] == -1).all() and (tb[par == 0] >= 1).all()
    # every link has exactly one RED end: after the RED half-sweep every link differs from its input
    assert (np.abs(b - U0).reshape(V * 4, -1).max(axis=1) > 1e-6).all()
    oracle.heatbath_half(b, dims, 0.9, 7, 0, 1, trials=tb)
    assert np.array_equal(a, b) and np.array_equal(ta, tb)


def test_fix_lag_one_stops_one_sweep_after_the_check():
    """C21: orc_fix_lag(lag = 1) ends one sweep after the first checked sweep below the tolerance; its field is plain
    sweeping for that many sweeps; lag = 0 is orc_fix; no check takes place at the last allowed sweep (lag = 1)"""
    dims = (4, 4, 4, 4)
    U0 = gf_inputs.smooth_random(dims, 0.3, 46)
    tol = 1e-8
    scan, th = U0.copy(), []
    for n in range(1, 400):
        oracle.overrelax(scan, dims, 1.6, 1)
        th.append(oracle.theta(scan, dims))
        if th[-1] < 1e-10:
            break
    for every in (1, 3, 10):
        first = next(n for n in range(every, len(th) + 1, every) if th[n - 1] < tol)  # first checked sweep below tol
        for lag in (0, 1):
            V = U0.copy()
            n, thn, F = oracle.fix(V, dims, oracle.UPDATE_OVERRELAX2, 1.6, tol, every, 1000, lag=lag)
            assert n == first + lag, (every, lag)
            W = U0.copy()
            oracle.overrelax(W, dims, 1.6, n)
            assert np.array_equal(V, W)
            assert thn == oracle.theta(W, dims) and F == oracle.functional(W, dims)
        V = U0.copy()  # the check at sweep `first` cannot take place if that is the last allowed sweep
        assert oracle.fix(V, dims, oracle.UPDATE_OVERRELAX2, 1.6, tol, every, first, lag=1)[0] == first
        V = U0.copy()
        assert oracle.fix(V, dims, oracle.UPDATE_OVERRELAX2, 1.6, tol, every, first + 5, lag=1)[0] == first + 1
    assert oracle.fix(scan, dims, oracle.UPDATE_OVERRELAX2, 1.6, tol, 1, 50, lag=1)[0] == 0  # already fixed


def test_fix_slices_lag():
    """orc_fix_slices_lag: lag = 0 is orc_fix_slices (sweep by sweep instead of chunk by chunk); lag = 1 gives every
    slice exactly one more sweep than lag = 0 at check_every = 1 (unless it was fixed from the start)"""
    dims = (4, 4, 4, 6)
    U0 = gf_inputs.smooth_random(dims, 0.5, 47)
    a, b = U0.copy(), U0.copy()
    na, tha, Fa, pa = oracle.fix_slices(a, dims, oracle.UPDATE_OVERRELAX2, 1.5, 1e-9, 4, 3000)
    lib = oracle._load()
    import ctypes
    N, V = oracle._dims(dims)
    th, F = ctypes.c_double(), ctypes.c_double()
    per = np.zeros(dims[3], dtype=np.int32)
    nb = lib.orc_fix_slices_lag(N, oracle.COULOMB, b.ctypes.data, 0, 1.5, 1e-9, 4, 3000, 0, 0, per.ctypes.data,
                                ctypes.byref(th), ctypes.byref(F))
    assert nb == na and np.array_equal(per, pa) and np.array_equal(a, b) and th.value == tha
    c, d = U0.copy(), U0.copy()
    n0, _, _, p0 = oracle.fix_slices(c, dims, oracle.UPDATE_OVERRELAX2, 1.5, 1e-9, 1, 3000, lag=0)
    n1, th1, _, p1 = oracle.fix_slices(d, dims, oracle.UPDATE_OVERRELAX2, 1.5, 1e-9, 1, 3000, lag=1)
    assert np.array_equal(p1, p0 + 1) and n1 == n0 + 1 and th1 < 1e-9


def test_black_sites_keep_K_of_the_finished_sweep_in_the_chain():
    """What the fused monitor rests on (C21): after its three subgroup steps the K <- G K chain of a BLACK site IS
    K(x) of the state after the sweep -- no later update of the half-sweep touches its links (C6) -- so
    sum over BLACK sites of tr[Delta Delta^dagger] from the chain plus the sum over RED sites from K built before
    the next sweep's RED update equals orc_theta of the state in between."""
    dims = (4, 4, 2, 4)
    V = int(np.prod(dims))
    U = gf_inputs.smooth_random(dims, 0.4, 48)
    omega = 1.7
    oracle.overrelax_half(U, dims, omega, 0)
    before_black = U.copy()
    oracle.overrelax_half(U, dims, omega, 1)  # U is now S_1
    s = np.arange(V)
    par = (s % 4 + (s // 4) % 4 + (s // 16) % 2 + s // 32) & 1

    def delta2(K):
        D = (K - K.conj().T) / 2j
        D = D - np.trace(D) / 3 * np.eye(3)
        return float((np.abs(D) ** 2).sum())

    total = 0.0
    for x in range(V):
        if par[x] == 1:  # the chain of the BLACK update, restated with the oracle's pieces on the state before it
            K = oracle.build_K(before_black, dims, x)
            for i, j in ((0, 1), (0, 2), (1, 2)):
                g = oracle.su2_maximiser(oracle.su2_project(K, i, j))
                K = oracle.su2_embed(oracle.su2_overrelax(g, omega), i, j) @ K
            assert delta2(K) == pytest.approx(oracle.site_theta(U, dims, x), rel=1e-9, abs=1e-26)
            total += delta2(K)
        else:            # what the RED half-sweep of the next sweep builds before it updates
            total += delta2(oracle.build_K(U, dims, x))
    assert total / (3 * V) == pytest.approx(oracle.theta(U, dims), rel=1e-12)
