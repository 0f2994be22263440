"""Pins of the CPU oracle against what the paper and the mathematics fix (P1..P13).

Each test compares oracle/ with something that is not the oracle: a value the paper prints, a closed form,
an invariant, brute force, or an independent whole-lattice numpy restatement (tests/np_lattice.py).
"""
import os

import numpy as np
import pytest
from scipy import special

import gf_inputs
import oracle

import np_lattice as npl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
SUBGROUPS = ((0, 1), (0, 2), (1, 2))


def _golden_kv(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, *vals = line.split()
            out[key] = vals
    return out


# ---------------------------------------------------------------------------------------------------------
# P11: Philox4x32-10 known answers (both the oracle's copy and the input generator's copy)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("impl", [oracle.philox4x32_10, gf_inputs.philox4x32_10])
def test_philox_known_answers(impl):
    rows = 0
    with open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            w = [int(v, 16) for v in line.split()]
            out = impl(w[0:4], w[4:6])
            assert [int(v) for v in out] == w[6:10]
            rows += 1
    assert rows == 3


# ---------------------------------------------------------------------------------------------------------
# P10: flop bookkeeping of Alg. 1
# ---------------------------------------------------------------------------------------------------------
def test_paper_flop_model():
    g = {k: int(v[0]) for k, v in _golden_kv("paper_flop_model.txt").items()}
    assert (oracle.FLOP_PROJECT, oracle.FLOP_OMEGA, oracle.FLOP_LEFT, oracle.FLOP_RIGHT) == (
        g["project_flop"], g["omega_flop"], g["left_mult_flop"], g["right_mult_flop"])
    per_sub = g["project_flop"] + g["omega_flop"] + g["directions"] * (g["left_mult_flop"] + g["right_mult_flop"])
    assert per_sub == g["per_subgroup_total"] == oracle.FLOP_PER_SUBGROUP == 751
    assert g["subgroups"] * per_sub == g["per_site_total"] == oracle.FLOP_PER_SITE == 2253
    assert g["links_per_site"] * g["reals_per_link"] == g["reals_per_site"] == 144


# ---------------------------------------------------------------------------------------------------------
# P1: trivial orbit relaxes to F = 1, theta -> 0 (north_star; BASELINE.json configs[0])
# ---------------------------------------------------------------------------------------------------------
def test_trivial_orbit_config1():
    g = _golden_kv("config1_expectation.txt")
    dims = tuple(int(v) for v in g["dims"])
    U = gf_inputs.trivial_orbit(dims, int(g["seed"][0]))
    assert abs(npl.plaquette(U, dims) - 1.0) < 1e-13  # a pure gauge
    assert oracle.theta(U, dims) > 1.0  # far from fixed to begin with
    tol, omega = float(g["theta_tol"][0]), float(g["omega"][0])
    sweeps = 0
    while oracle.theta(U, dims) >= tol and sweeps < int(g["max_sweeps"][0]):
        oracle.overrelax(U, dims, omega, 1)
        sweeps += 1
    assert oracle.theta(U, dims) < tol, "theta did not reach 1e-14 within 500 sweeps"
    assert sweeps < 200
    assert abs(oracle.functional(U, dims) - float(g["F_final"][0])) < float(g["F_abs_tol"][0])
    # the fixed field of a trivial orbit at the global maximum is the unit field up to a constant centre-free
    # gauge rotation: every link must be (numerically) the same constant matrix with Re tr = 3
    assert np.abs(U - np.eye(3)).max() < 1e-6


# ---------------------------------------------------------------------------------------------------------
# independent restatements: F, theta (P8), K, plaquette, per-site quantities
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 2, 8)])
@pytest.mark.parametrize("gauge,nd", [(oracle.LANDAU, 4), (oracle.COULOMB, 3)])
def test_reductions_match_numpy_definitions(dims, gauge, nd):
    U = gf_inputs.smooth_random(dims, 0.4, 11)
    V = int(np.prod(dims))
    assert oracle.functional(U, dims, gauge) == pytest.approx(npl.functional(U, dims, nd), rel=1e-13, abs=1e-15)
    th_sites = npl.theta_from_A(U, dims, nd)  # P8: Delta from A_mu differences
    assert oracle.theta_mean(U, dims, gauge) == pytest.approx(th_sites.sum() / (3 * V), rel=1e-12)
    for s in (0, 5, V - 1, V // 2 + 3):
        x, y, z, t = npl.site_coords(s, dims)
        assert oracle.site_theta(U, dims, s, gauge) == pytest.approx(th_sites[t, z, y, x], rel=1e-11)
        np.testing.assert_allclose(oracle.build_K(U, dims, s, gauge), npl.K_field(U, dims, nd)[t, z, y, x],
                                   rtol=0, atol=1e-13)
    if gauge == oracle.COULOMB:
        sl = oracle.theta_slices(U, dims)
        Vs = dims[0] * dims[1] * dims[2]
        np.testing.assert_allclose(sl, th_sites.reshape(dims[3], -1).sum(axis=1) / (3 * Vs), rtol=1e-12)
        assert oracle.theta(U, dims, gauge) == pytest.approx(sl.max(), rel=1e-15)
    assert oracle.plaquette(U, dims) == pytest.approx(npl.plaquette(U, dims), rel=1e-13)


# ---------------------------------------------------------------------------------------------------------
# P9: constant diagonal field: theta = 0, F closed form, a sweep leaves it unchanged
# ---------------------------------------------------------------------------------------------------------
def test_constant_diagonal_fixed_point():
    dims = (4, 4, 2, 6)
    V = int(np.prod(dims))
    phi = np.array([0.3, -0.7, 1.1, 0.45])
    U = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    for mu in range(4):
        U[:, mu] = np.diag([np.exp(1j * phi[mu]), np.exp(-1j * phi[mu]), 1.0])
    U0 = U.copy()
    assert oracle.theta(U, dims) < 1e-30
    assert oracle.functional(U, dims) == pytest.approx(np.sum(2 * np.cos(phi) + 1) / 12, rel=1e-14)
    assert oracle.functional(U, dims, oracle.COULOMB) == pytest.approx(np.sum(2 * np.cos(phi[:3]) + 1) / 9, rel=1e-14)
    oracle.overrelax(U, dims, 1.7, 2)
    assert np.abs(U - U0).max() < 1e-14


# ---------------------------------------------------------------------------------------------------------
# P3/P4 + C4/C7: the SU(2) maximiser, against explicit Pauli matrices and brute force
# ---------------------------------------------------------------------------------------------------------
def test_embedding_matches_pauli_matrices():
    rng = np.random.default_rng(5)
    for (i, j) in SUBGROUPS:
        q = rng.normal(size=4)
        q /= np.linalg.norm(q)
        G = oracle.su2_embed(q, i, j)
        np.testing.assert_allclose(G, npl.embed(q, i, j), atol=1e-16)
        np.testing.assert_allclose(G @ G.conj().T, np.eye(3), atol=1e-15)
        assert abs(np.linalg.det(G) - 1) < 1e-15
        # quaternion product is the matrix product under the embedding
        p = rng.normal(size=4)
        p /= np.linalg.norm(p)
        np.testing.assert_allclose(npl.quat_to_su2(oracle.quat_mul(p, q)), npl.quat_to_su2(p) @ npl.quat_to_su2(q),
                                   atol=1e-15)


def test_projection_is_linear_functional_of_g():
    """C7: Re tr[G K] = const + g0 k0 - g1 k1 - g2 k2 - g3 k3 for any K and any unit g."""
    rng = np.random.default_rng(6)
    K = rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3))
    for (i, j) in SUBGROUPS:
        k = oracle.su2_project(K, i, j)
        rest = [r for r in range(3) if r not in (i, j)][0]
        for _ in range(20):
            g = rng.normal(size=4)
            g /= np.linalg.norm(g)
            lhs = np.trace(npl.embed(g, i, j) @ K).real
            rhs = K[rest, rest].real + g[0] * k[0] - g[1] * k[1] - g[2] * k[2] - g[3] * k[3]
            assert lhs == pytest.approx(rhs, abs=1e-13)


def test_maximiser_beats_brute_force_and_diagonalises_block():
    dims = (2, 2, 2, 2)
    U = gf_inputs.hot(dims, 21)
    rng = np.random.default_rng(7)
    cand = rng.normal(size=(100000, 4))
    cand /= np.linalg.norm(cand, axis=1, keepdims=True)
    for s in (0, 7, 13):
        K = oracle.build_K(U, dims, s)
        for (i, j) in SUBGROUPS:
            k = oracle.su2_project(K, i, j)
            g = oracle.su2_maximiser(k)
            n = np.linalg.norm(k)
            assert np.linalg.norm(g) == pytest.approx(1.0, abs=1e-15)
            best = np.trace(npl.embed(g, i, j) @ K).real
            # P4: brute force over 1e5 random SU(2) elements, evaluated with explicit 2x2 matrices
            blk = K[np.ix_([i, j], [i, j])]
            vals = np.einsum("nab,ba->n", npl.quat_to_su2(cand), blk).real
            rest = [r for r in range(3) if r not in (i, j)][0]
            assert best >= vals.max() + K[rest, rest].real
            assert best - (vals.max() + K[rest, rest].real) < 0.05 * n  # and the brute force gets close
            # P3: the projected block of G K is (n, 0, 0, 0)
            k_new = oracle.su2_project(npl.embed(g, i, j) @ K, i, j)
            np.testing.assert_allclose(k_new, [n, 0, 0, 0], atol=1e-13)


# ---------------------------------------------------------------------------------------------------------
# P7: second-order g^omega (C9)
# ---------------------------------------------------------------------------------------------------------
def test_overrelax_formula_closed_forms():
    rng = np.random.default_rng(8)
    for _ in range(50):
        g = rng.normal(size=4)
        g /= np.linalg.norm(g)
        np.testing.assert_allclose(oracle.su2_overrelax(g, 1.0), g, atol=1e-15)
        m2 = npl.quat_to_su2(g) @ npl.quat_to_su2(g)
        np.testing.assert_allclose(npl.quat_to_su2(oracle.su2_overrelax(g, 2.0)), m2, atol=1e-14)
    # against the exact power (cos(w phi), sin(w phi) n) for small rotation angles: error <= |w(w-1)(w-2)/6| phi^3
    for omega in (1.3, 1.7, 1.9):
        for phi in (0.01, 0.05, 0.2):
            axis = rng.normal(size=3)
            axis /= np.linalg.norm(axis)
            g = np.concatenate([[np.cos(phi)], np.sin(phi) * axis])
            exact = np.concatenate([[np.cos(omega * phi)], np.sin(omega * phi) * axis])
            h = oracle.su2_overrelax(g, omega)
            assert np.linalg.norm(h) == pytest.approx(1.0, abs=1e-15)
            bound = abs(omega * (omega - 1) * (omega - 2) / 6) * phi ** 3
            err = np.linalg.norm(h - exact)
            assert err <= 1.1 * bound
            assert err >= 0.5 * bound  # and it is genuinely second order, not better
    # the series is in (g-1): first and second derivative in omega at the identity direction
    g = np.array([np.cos(0.3), np.sin(0.3), 0, 0])
    d = g[0] - 1
    w = 1.7
    h = oracle.su2_overrelax(g, w)
    raw = np.array([1 + w * d + w * (w - 1) / 2 * (d * d - np.sin(0.3) ** 2), (w + w * (w - 1) * d) * np.sin(0.3), 0, 0])
    np.testing.assert_allclose(h, raw / np.linalg.norm(raw), atol=1e-15)


def test_overrelax_guards():
    # singular point: g0 = -1 and omega = 1 + 1/sqrt2 -> |h| = 0 -> falls back to g (C9)
    g = np.array([-1.0, 0.0, 0.0, 0.0])
    np.testing.assert_array_equal(oracle.su2_overrelax(g, 1 + 1 / np.sqrt(2)), g)
    np.testing.assert_array_equal(oracle.su2_maximiser(np.zeros(4)), [1, 0, 0, 0])


# ---------------------------------------------------------------------------------------------------------
# site update: what it does to the links is a gauge transformation at x, and F_raw changes by Re tr[(g-1) K]
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge,nd", [(oracle.LANDAU, 4), (oracle.COULOMB, 3)])
def test_site_update_is_local_gauge_transformation(gauge, nd):
    dims = (4, 4, 4, 4)
    V = 256
    U = gf_inputs.smooth_random(dims, 0.4, 12)
    s = 77
    K = npl.K_field(U, dims, nd)[npl.site_coords(s, dims)[::-1]]
    U1 = U.copy()
    oracle.site_overrelax(U1, dims, s, 1.7, gauge)
    g = U1[s, 0] @ U[s, 0].conj().T  # read g(x) off one forward link
    np.testing.assert_allclose(g @ g.conj().T, np.eye(3), atol=1e-14)
    gfield = np.tile(np.eye(3, dtype=np.complex128), (V, 1, 1))
    gfield[s] = g
    np.testing.assert_allclose(U1, npl.gauge_transform(U, dims, gfield), atol=1e-14)  # all 8 links, nothing else
    dF = (npl.functional(U1, dims, nd) - npl.functional(U, dims, nd)) * 3 * nd * V
    assert dF == pytest.approx(np.trace((g - np.eye(3)) @ K).real, abs=1e-11)
    # omega = 1: three exact subgroup maximisations, each raising Re tr[gK] by n - k0 >= 0 (P2); the last
    # subgroup's block of the new K is diagonalised (P3)
    U2 = U.copy()
    oracle.site_overrelax(U2, dims, s, 1.0, gauge)
    Kc, gain = K.copy(), 0.0
    for (i, j) in SUBGROUPS:
        k = oracle.su2_project(Kc, i, j)
        gain += np.linalg.norm(k) - k[0]
        Kc = npl.embed(oracle.su2_maximiser(k), i, j) @ Kc
    dF1 = (npl.functional(U2, dims, nd) - npl.functional(U, dims, nd)) * 3 * nd * V
    assert dF1 == pytest.approx(gain, abs=1e-11) and gain > 0
    K_new = npl.K_field(U2, dims, nd)[npl.site_coords(s, dims)[::-1]]
    k_last = oracle.su2_project(K_new, 1, 2)
    np.testing.assert_allclose(k_last[1:], 0, atol=1e-13)
    assert k_last[0] > 0


def test_omega_two_is_microcanonical():
    """h = g^2 reflects g about the maximum: Re tr[gK] and hence F are exactly conserved (unit test of C9 + a5)."""
    dims = (4, 4, 4, 4)
    U = gf_inputs.smooth_random(dims, 0.4, 13)
    F0 = npl.functional(U, dims)
    for s in range(0, 256, 7):
        oracle.site_overrelax(U, dims, s, 2.0)
    assert npl.functional(U, dims) == pytest.approx(F0, abs=1e-13)
    assert np.abs(U - gf_inputs.smooth_random(dims, 0.4, 13)).max() > 0.1  # but the links did move


# ---------------------------------------------------------------------------------------------------------
# P2: omega = 1 -> F non-decreasing after every half-sweep (hot field)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge,nd", [(oracle.LANDAU, 4), (oracle.COULOMB, 3)])
def test_relaxation_monotone(gauge, nd):
    dims = (4, 4, 4, 4)
    U = gf_inputs.hot(dims, 31)
    F_prev = npl.functional(U, dims, nd)
    for it in range(60):
        oracle.overrelax_half(U, dims, 1.0, it & 1, gauge)
        F = npl.functional(U, dims, nd)
        assert F > F_prev
        F_prev = F
    assert F_prev > 0.4


# ---------------------------------------------------------------------------------------------------------
# P5/P6: gauge invariance (plaquette) and unitarity under sweeps of every kind
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("gauge", [oracle.LANDAU, oracle.COULOMB])
def test_plaquette_and_unitarity_invariant(gauge):
    dims = (4, 4, 4, 6)
    U = gf_inputs.smooth_random(dims, 0.5, 14)
    U0 = U.copy()
    p0 = npl.plaquette(U, dims)
    oracle.overrelax(U, dims, 1.7, 40, gauge)
    assert abs(npl.plaquette(U, dims) - p0) < 1e-12
    oracle.anneal(U, dims, 1.4, 0.01, 10, 7, gauge)
    assert abs(npl.plaquette(U, dims) - p0) < 1e-12
    np.testing.assert_allclose(U @ npl.dag(U), np.broadcast_to(np.eye(3), U.shape), atol=1e-12)
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-12
    uu, dd = oracle.unitarity_defect(U, dims)
    assert uu < 1e-12 and dd < 1e-12
    # every gauge-invariant loop is preserved: compare the plaquette field site by site via Re tr of all 1x1 loops
    G0, G1 = npl.as_grid(U0, dims), npl.as_grid(U, dims)
    for mu, nu in ((0, 3), (1, 2)):
        def loop(G):
            return np.trace(G[..., mu, :, :] @ npl.shift(G[..., nu, :, :], mu, 1)
                            @ npl.dag(npl.shift(G[..., mu, :, :], nu, 1)) @ npl.dag(G[..., nu, :, :]),
                            axis1=-2, axis2=-1)
        np.testing.assert_allclose(loop(G1), loop(G0), atol=1e-12)


def test_coulomb_timeslices_decouple_and_converge():
    dims = (4, 4, 4, 4)
    U = gf_inputs.smooth_random(dims, 0.5, 15)
    oracle.overrelax(U, dims, 1.7, 150, oracle.COULOMB)
    sl = oracle.theta_slices(U, dims)
    assert sl.max() < 1e-10
    assert oracle.theta(U, dims, oracle.COULOMB) == sl.max()
    assert npl.theta_from_A(U, dims, 3).max() < 1e-9
    assert oracle.theta_mean(U, dims, oracle.LANDAU) > 1e-3  # Coulomb-fixed is not Landau-fixed


def test_results_independent_of_thread_count():
    dims = (4, 4, 4, 4)
    U1 = gf_inputs.smooth_random(dims, 0.4, 16)
    U8 = U1.copy()
    nthr = oracle.max_threads()
    try:
        oracle.set_threads(1)
        oracle.overrelax(U1, dims, 1.7, 3)
        oracle.anneal(U1, dims, 1.0, 0.5, 2, 3)
        oracle.set_threads(4)
        oracle.overrelax(U8, dims, 1.7, 3)
        oracle.anneal(U8, dims, 1.0, 0.5, 2, 3)
    finally:
        oracle.set_threads(nthr)
    np.testing.assert_array_equal(U1, U8)  # C6: race-free, order-independent


def test_gauge_covariance_of_fixing():
    """Fixing g-transformed links with a constant g gives the constant-g transform of the fixed links (eq. 1.1)."""
    dims = (4, 4, 4, 4)
    U = gf_inputs.smooth_random(dims, 0.4, 17)
    g = gf_inputs.haar_su3(99, 0)
    Ug = np.ascontiguousarray(g @ U @ g.conj().T)
    assert oracle.functional(Ug, dims) == pytest.approx(oracle.functional(U, dims), abs=1e-14)
    assert oracle.theta(Ug, dims) == pytest.approx(oracle.theta(U, dims), rel=1e-12)


# ---------------------------------------------------------------------------------------------------------
# P12/P13: heatbath (C13/C14)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("alpha", [0.5, 2.0, 8.0, 40.0])
def test_kennedy_pendleton_law(alpha):
    n = 40000
    hs = np.empty((n, 4))
    trials = np.empty(n, dtype=int)
    for c0 in range(n):
        hs[c0], trials[c0] = oracle.kp_draw(alpha, (7, 0), c0, 3, 1)
    np.testing.assert_allclose(np.linalg.norm(hs, axis=1), 1.0, atol=1e-14)
    # density sqrt(1-h0^2) exp(alpha h0) on [-1,1]  =>  <h0> = I_2(alpha)/I_1(alpha)
    h0 = hs[:, 0]
    assert abs(h0.mean() - special.ive(2, alpha) / special.ive(1, alpha)) < 4 * h0.std() / np.sqrt(n)
    # second moment by quadrature of the density
    x = np.linspace(-1, 1, 200001)
    w = np.sqrt(1 - x * x) * np.exp(alpha * (x - 1))
    m2 = np.sum(w * x * x) / np.sum(w)
    assert abs((h0 ** 2).mean() - m2) < 4 * (h0 ** 2).std() / np.sqrt(n)
    # isotropy of hvec / |hvec|
    dirs = hs[:, 1:] / np.linalg.norm(hs[:, 1:], axis=1, keepdims=True)
    assert np.abs(dirs.mean(axis=0)).max() < 4 / np.sqrt(3 * n)
    np.testing.assert_allclose((dirs ** 2).mean(axis=0), 1 / 3, atol=4 * 0.3 / np.sqrt(n))
    assert trials.min() >= 1 and trials.max() < 4096
    if alpha >= 8:
        assert trials.mean() < 1.1


def test_kp_draw_follows_stated_recipe():
    """One draw, re-derived from the Philox words by hand (numpy), including the reject/accept decisions."""
    key, c0, c1, c2, alpha = (123, 45), 1000, 9, 6, 0.7

    def u24(x):
        return (2 * (int(x) >> 9) + 1) / 2.0 ** 24

    t = 0
    while True:
        x = gf_inputs.philox4x32_10([c0, c1, c2, t], key)  # the generator module's independent Philox copy
        u1, u2, u3, u4 = (u24(v) for v in x)
        delta = (-np.log(u1) / alpha) * np.cos(2 * np.pi * u3) ** 2 + (-np.log(u2) / alpha)
        if u4 * u4 <= 1 - 0.5 * delta:
            break
        t += 1
    h, ntr = oracle.kp_draw(alpha, key, c0, c1, c2)
    assert ntr == t + 1 and t >= 1  # this counter needs at least one rejection
    assert h[0] == pytest.approx(1 - delta, abs=1e-15)
    x = gf_inputs.philox4x32_10([c0, c1, c2, 0x80000000], key)
    ct, ph = 1 - 2 * u24(x[0]), 2 * np.pi * u24(x[1])
    r = np.sqrt(1 - h[0] ** 2)
    np.testing.assert_allclose(h[1:], [r * np.sqrt(1 - ct * ct) * np.cos(ph), r * np.sqrt(1 - ct * ct) * np.sin(ph), r * ct],
                               atol=1e-15)


def test_heatbath_site_update_block_is_n_times_h():
    dims = (4, 4, 4, 4)
    U = gf_inputs.smooth_random(dims, 0.5, 18)
    s, T, seed, step = 100, 0.8, 7 + (5 << 32), 3
    U1 = U.copy()
    ntr = oracle.site_heatbath(U1, dims, s, T, seed, step)
    assert (ntr >= 1).all()
    # still a local gauge transformation
    g = U1[s, 2] @ U[s, 2].conj().T
    gfield = np.tile(np.eye(3, dtype=np.complex128), (256, 1, 1))
    gfield[s] = g
    np.testing.assert_allclose(U1, npl.gauge_transform(U, dims, gfield), atol=1e-14)
    # last subgroup: the projected (1,2) block of the new K equals n * h with h the KP draw at alpha = n / T
    K_new = npl.K_field(U1, dims)[npl.site_coords(s, dims)[::-1]]
    k = oracle.su2_project(K_new, 1, 2)
    n = np.linalg.norm(k)
    parity = sum(npl.site_coords(s, dims)) & 1
    h, ntr_last = oracle.kp_draw(n / T, (seed & 0xFFFFFFFF, seed >> 32), s, step, (parity << 2) | 2)
    np.testing.assert_allclose(k / n, h, atol=1e-12)
    assert ntr_last == ntr[2]


def test_annealing_heats_and_freezes():
    dims = (4, 4, 4, 4)
    U = gf_inputs.smooth_random(dims, 0.4, 19)
    p0 = npl.plaquette(U, dims)
    Uh = U.copy()
    oracle.anneal(Uh, dims, 1.4, 1.4, 20, 7)
    F_hot = oracle.functional(Uh, dims)
    Uc = U.copy()
    oracle.anneal(Uc, dims, 1.4, 0.01, 100, 7)
    F_cold = oracle.functional(Uc, dims)
    assert F_hot < 0.3 < 0.6 < F_cold  # exp(+F_raw/T): hot = disordered gauge, cold = close to a maximum
    assert abs(npl.plaquette(Uc, dims) - p0) < 1e-12
    # schedule: nsteps = 1 runs at T_start; different seeds give different fields; same seed reproduces
    Ua, Ub, Uc2 = U.copy(), U.copy(), U.copy()
    oracle.anneal(Ua, dims, 0.7, 0.1, 1, 5)
    oracle.anneal(Ub, dims, 0.7, 0.7, 1, 5)
    oracle.anneal(Uc2, dims, 0.7, 0.1, 1, 6)
    np.testing.assert_array_equal(Ua, Ub)
    assert np.abs(Ua - Uc2).max() > 1e-3
    # linear schedule: two steps 0.9 -> 0.3 equal one step at 0.9 followed by... the step index keys the RNG, so
    # compare with two single-site-free runs through site_heatbath over the whole lattice
    Ud = U.copy()
    oracle.anneal(Ud, dims, 0.9, 0.3, 3, 11)
    Ue = U.copy()
    for step, T in enumerate((0.9, 0.6, 0.3)):
        for parity in (0, 1):
            for s in range(256):
                if sum(npl.site_coords(s, dims)) & 1 == parity:
                    oracle.site_heatbath(Ue, dims, s, T, 11, step)
    np.testing.assert_allclose(Ud, Ue, atol=1e-13)


def test_sweep_order_red_then_black():
    """C5: RED = even sites first.  A full sweep equals the half-sweeps applied in that order and differs otherwise."""
    dims = (4, 4, 4, 4)
    U = gf_inputs.smooth_random(dims, 0.4, 20)
    Ua, Ub, Uc = U.copy(), U.copy(), U.copy()
    oracle.overrelax(Ua, dims, 1.7, 1)
    oracle.overrelax_half(Ub, dims, 1.7, 0)
    oracle.overrelax_half(Ub, dims, 1.7, 1)
    np.testing.assert_array_equal(Ua, Ub)
    oracle.overrelax_half(Uc, dims, 1.7, 1)
    oracle.overrelax_half(Uc, dims, 1.7, 0)
    assert np.abs(Ua - Uc).max() > 1e-3
    # a RED half-sweep is the site updates of the even sites in any order
    Ud = U.copy()
    for s in reversed(range(256)):
        if sum(npl.site_coords(s, dims)) % 2 == 0:
            oracle.site_overrelax(Ud, dims, s, 1.7)
    Ue = U.copy()
    oracle.overrelax_half(Ue, dims, 1.7, 0)
    np.testing.assert_array_equal(Ud, Ue)


def test_unitarity_defect_of_known_matrices():
    """orc_unitarity_defect is the checker of several GPU tests: pin it on matrices with a known defect.
    diag(1+e, 1, 1): U U^dagger - 1 = diag(2e + e^2, 0, 0), det - 1 = e; a unitary matrix with det = exp(i a):
    U U^dagger = 1 and |det - 1| = 2 sin(a/2); an SU(3) field: both ~ 1e-16."""
    dims = (2, 2, 2, 2)
    U = gf_inputs.hot(dims, 5)
    uu, det = oracle.unitarity_defect(U, dims)
    assert uu < 1e-14 and det < 1e-14
    eps = 3e-4
    V = U.copy()
    V[5, 2] = np.diag([1 + eps, 1.0, 1.0])
    uu, det = oracle.unitarity_defect(V, dims)
    assert uu == pytest.approx(2 * eps + eps * eps, rel=1e-10) and det == pytest.approx(eps, rel=1e-10)
    a = 0.02
    W = U.copy()
    W[7, 1] = W[7, 1] * np.exp(1j * a / 3)  # unitary, det = exp(i a)
    uu, det = oracle.unitarity_defect(W, dims)
    assert uu < 1e-14 and det == pytest.approx(2 * np.sin(a / 2), rel=1e-9)
    X = U.copy()
    X[0, 0, 0, 1] += 1e-3  # one off-diagonal entry of one link: (U U^dagger - 1) picks up terms of that size
    uu, det = oracle.unitarity_defect(X, dims)
    assert 5e-4 < uu < 3e-3


def test_reunitarise_projects_back_to_su3():
    """orc_reunitarise (the definition of the CUDA path's re-orthonormalisation on load, C15): a sheared and scaled
    link comes back unitary with det 1; row 0 keeps its direction, row 1 keeps its component orthogonal to row 0,
    row 2 = conj(row0 x row1); an SU(3) link is left unchanged to rounding."""
    dims = (2, 2, 2, 2)
    U = gf_inputs.hot(dims, 6)
    V = U.copy()
    oracle.reunitarise(V, dims)
    assert np.abs(V - U).max() < 1e-14
    rng = np.random.default_rng(3)
    D = U.copy()
    D *= 1.0 + 0.05 * rng.standard_normal((D.shape[0], 4, 3, 1))  # every row scaled
    D[:, :, 1, :] += 0.1 * D[:, :, 0, :]                          # row 1 sheared towards row 0
    D[:, :, 2, :] = rng.standard_normal(D[:, :, 2, :].shape)      # row 2 destroyed
    W = D.copy()
    oracle.reunitarise(W, dims)
    uu, det = oracle.unitarity_defect(W, dims)
    assert uu < 1e-14 and det < 1e-14
    r0 = D[:, :, 0, :] / np.linalg.norm(D[:, :, 0, :], axis=-1, keepdims=True)
    assert np.abs(W[:, :, 0, :] - r0).max() < 1e-14
    r1 = D[:, :, 1, :] - (np.conj(r0) * D[:, :, 1, :]).sum(-1, keepdims=True) * r0
    r1 /= np.linalg.norm(r1, axis=-1, keepdims=True)
    assert np.abs(W[:, :, 1, :] - r1).max() < 1e-14
    assert np.abs(W[:, :, 2, :] - np.conj(np.cross(r0, r1))).max() < 1e-14
    # the shear and the scaling did not change the SU(3) matrix the first two rows span: it is the original link
    assert np.abs(W - U).max() < 1e-13
