"""ctypes front end of the fp64 CPU oracle (oracle/gf_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, ``__graft_entry__.smoke()`` and bench.py's cpu_baseline /
``--impl reference`` legs.  Nothing under ``paper_1209_4008_b200`` imports this package and this package
imports nothing from it.

All fields are numpy complex128 arrays ``U[s, mu, row, col]`` in the canonical layout,
updated IN PLACE.  Function names mirror the ``gf_*`` C-ABI calls: overrelax / anneal / functional / theta.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

LANDAU, COULOMB = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gf_oracle.c")
_LIB = os.path.join(_HERE, "liborc.so")
_lib = None

_c_int4 = ctypes.c_int * 4
_vp = ctypes.c_void_p
_dbl = ctypes.c_double
_int = ctypes.c_int


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 -fopenmp (as it stands; never tuned)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    N = ctypes.POINTER(ctypes.c_int)
    sig = {
        "orc_build_K": (None, [N, _int, _vp, ctypes.c_long, _vp]),
        "orc_su2_project": (None, [_vp, _int, _int, _vp]),
        "orc_su2_maximiser": (None, [_vp, _vp]),
        "orc_su2_overrelax": (None, [_vp, _dbl, _vp]),
        "orc_quat_mul": (None, [_vp, _vp, _vp]),
        "orc_su2_embed": (None, [_vp, _int, _int, _vp]),
        "orc_site_overrelax": (None, [N, _int, _vp, ctypes.c_long, _dbl]),
        "orc_overrelax_half": (None, [N, _int, _vp, _dbl, _int]),
        "orc_overrelax": (None, [N, _int, _vp, _dbl, _int]),
        "orc_functional": (_dbl, [N, _int, _vp]),
        "orc_site_theta": (_dbl, [N, _int, _vp, ctypes.c_long]),
        "orc_theta": (_dbl, [N, _int, _vp, _vp]),
        "orc_theta_report": (_dbl, [N, _int, _vp]),
        "orc_plaquette": (_dbl, [N, _vp]),
        "orc_unitarity_defect": (None, [N, _vp, _vp, _vp]),
        "orc_reunitarise": (None, [N, _vp]),
        "orc_philox4x32_10": (None, [_vp, _vp, _vp]),
        "orc_kp_draw": (_int, [_dbl, _vp, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32, _vp]),
        "orc_site_heatbath": (None, [N, _int, _vp, ctypes.c_long, _dbl, ctypes.c_uint64, ctypes.c_uint32, _vp]),
        "orc_anneal": (None, [N, _int, _vp, _dbl, _dbl, _int, ctypes.c_uint64, _vp]),
        "orc_su2_overrelax1": (None, [_vp, _dbl, _vp]),
        "orc_su2_square": (None, [_vp, _vp]),
        "orc_site_relax": (None, [N, _int, _vp, ctypes.c_long, _int, _dbl, ctypes.c_uint64, ctypes.c_uint32, _vp]),
        "orc_relax": (None, [N, _int, _vp, _int, _dbl, _int, ctypes.c_uint64, _vp]),
        "orc_relax_from": (None, [N, _int, _vp, _int, _dbl, _int, _int, ctypes.c_uint64, _vp]),
        "orc_heatbath_half": (None, [N, _int, _vp, _dbl, ctypes.c_uint64, ctypes.c_uint32, _int, _vp]),
        "orc_fix": (_int, [N, _int, _vp, _int, _dbl, _dbl, _int, _int, ctypes.c_uint64, _vp, _vp]),
        "orc_fix_lag": (_int, [N, _int, _vp, _int, _dbl, _dbl, _int, _int, ctypes.c_uint64, _int, _vp, _vp]),
        "orc_fix_slices_lag": (_int, [N, _int, _vp, _int, _dbl, _dbl, _int, _int, ctypes.c_uint64, _int, _vp, _vp, _vp]),
        "orc_fix_slices": (_int, [N, _int, _vp, _int, _dbl, _dbl, _int, _int, ctypes.c_uint64, _vp, _vp, _vp]),
        "orc_anneal_micro": (None, [N, _int, _vp, _dbl, _dbl, _int, _int, ctypes.c_uint64, _vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _dims(dims):
    dims = tuple(int(d) for d in dims)
    assert len(dims) == 4
    return _c_int4(*dims), dims[0] * dims[1] * dims[2] * dims[3]


def _field(U, V):
    assert isinstance(U, np.ndarray) and U.dtype == np.complex128 and U.flags.c_contiguous
    assert U.shape == (V, 4, 3, 3), U.shape
    return U.ctypes.data


def set_threads(n: int) -> None:
    """OpenMP thread count for the oracle (results do not depend on it, C6)."""
    os.environ["OMP_NUM_THREADS"] = str(n)
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
    except OSError:
        pass


def max_threads() -> int:
    try:
        return int(ctypes.CDLL("libgomp.so.1").omp_get_max_threads())
    except OSError:
        return 1


# ---- the five calls ------------------------------------------------------------------------------------
def overrelax(U, dims, omega: float, nsweeps: int, gauge: int = LANDAU) -> None:
    N, V = _dims(dims)
    _load().orc_overrelax(N, gauge, _field(U, V), float(omega), int(nsweeps))


def overrelax_half(U, dims, omega: float, parity: int, gauge: int = LANDAU) -> None:
    N, V = _dims(dims)
    _load().orc_overrelax_half(N, gauge, _field(U, V), float(omega), int(parity))


def anneal(U, dims, T_start: float, T_end: float, nsteps: int, seed: int, gauge: int = LANDAU,
           trials: bool = False):
    N, V = _dims(dims)
    tr = np.zeros((V, 3), dtype=np.int32) if trials else None
    _load().orc_anneal(N, gauge, _field(U, V), float(T_start), float(T_end), int(nsteps), int(seed),
                       tr.ctypes.data if trials else None)
    return tr


UPDATE_OVERRELAX2, UPDATE_OVERRELAX1, UPDATE_STOCHASTIC = 0, 1, 2


def relax(U, dims, update: int, param: float, nsweeps: int, seed: int = 0, gauge: int = LANDAU, squared: bool = False):
    """update variants (C17, C18): second / first order overrelaxation (param = omega), stochastic relaxation
    (param = p).  squared=True returns the (V, 3) array of g^2 decisions of the last sweep."""
    N, V = _dims(dims)
    sq = np.zeros((V, 3), dtype=np.int32) if squared else None
    _load().orc_relax(N, gauge, _field(U, V), int(update), float(param), int(nsweeps), int(seed),
                      sq.ctypes.data if squared else None)
    return sq


def relax_from(U, dims, update: int, param: float, nsweeps: int, sweep0: int, seed: int = 0, gauge: int = LANDAU,
               squared: bool = False):
    """as relax with the sweep counter of the stochastic decisions starting at sweep0 (the chunks of fix)"""
    N, V = _dims(dims)
    sq = np.zeros((V, 3), dtype=np.int32) if squared else None
    _load().orc_relax_from(N, gauge, _field(U, V), int(update), float(param), int(nsweeps), int(sweep0), int(seed),
                           sq.ctypes.data if squared else None)
    return sq


def heatbath_half(U, dims, T: float, seed: int, step: int, parity: int, gauge: int = LANDAU, trials=None):
    """one heatbath half-sweep over one sublattice; trials: optional (V, 3) int32 array receiving the trial counts
    of the updated sites (other entries untouched)"""
    N, V = _dims(dims)
    if trials is not None:
        assert trials.shape == (V, 3) and trials.dtype == np.int32 and trials.flags.c_contiguous
    _load().orc_heatbath_half(N, gauge, _field(U, V), float(T), int(seed), int(step), int(parity),
                              trials.ctypes.data if trials is not None else None)
    return trials


def fix(U, dims, update: int, param: float, theta_tol: float, check_every: int, max_sweeps: int, seed: int = 0,
        gauge: int = LANDAU, lag: int = 0):
    """Alg. 1 outer loop: returns (sweeps done, theta, F).  lag = 0: the paper's loop; lag = 1:
    the loop ends one sweep after the check that met the tolerance (C21)"""
    N, V = _dims(dims)
    th, F = ctypes.c_double(), ctypes.c_double()
    n = _load().orc_fix_lag(N, gauge, _field(U, V), int(update), float(param), float(theta_tol), int(check_every),
                            int(max_sweeps), int(seed), int(lag), ctypes.byref(th), ctypes.byref(F))
    return int(n), th.value, F.value


def fix_slices(U, dims, update: int, param: float, theta_tol: float, check_every: int, max_sweeps: int, seed: int = 0,
               gauge: int = COULOMB, lag: int = 0):
    """Alg. 1 with the stop rule per timeslice (C20): returns (max sweeps, theta = max_t theta_t, F, sweeps per slice)"""
    N, V = _dims(dims)
    th, F = ctypes.c_double(), ctypes.c_double()
    per = np.zeros(int(dims[3]), dtype=np.int32)
    if lag == 0:
        n = _load().orc_fix_slices(N, gauge, _field(U, V), int(update), float(param), float(theta_tol), int(check_every),
                                   int(max_sweeps), int(seed), per.ctypes.data, ctypes.byref(th), ctypes.byref(F))
    else:
        n = _load().orc_fix_slices_lag(N, gauge, _field(U, V), int(update), float(param), float(theta_tol),
                                       int(check_every), int(max_sweeps), int(seed), int(lag), per.ctypes.data,
                                       ctypes.byref(th), ctypes.byref(F))
    return int(n), th.value, F.value, per


def anneal_micro(U, dims, T_start: float, T_end: float, nsteps: int, n_micro: int, seed: int, gauge: int = LANDAU,
                 trials: bool = False):
    """annealing with n_micro microcanonical (g -> g^2) sweeps after every heatbath sweep (C19)"""
    N, V = _dims(dims)
    tr = np.zeros((V, 3), dtype=np.int32) if trials else None
    _load().orc_anneal_micro(N, gauge, _field(U, V), float(T_start), float(T_end), int(nsteps), int(n_micro),
                             int(seed), tr.ctypes.data if trials else None)
    return tr


def su2_overrelax1(g, omega: float) -> np.ndarray:
    g = np.ascontiguousarray(g, dtype=np.float64)
    h = np.zeros(4)
    _load().orc_su2_overrelax1(g.ctypes.data, float(omega), h.ctypes.data)
    return h


def su2_square(g) -> np.ndarray:
    g = np.ascontiguousarray(g, dtype=np.float64)
    h = np.zeros(4)
    _load().orc_su2_square(g.ctypes.data, h.ctypes.data)
    return h


def functional(U, dims, gauge: int = LANDAU) -> float:
    N, V = _dims(dims)
    return float(_load().orc_functional(N, gauge, _field(U, V)))


def theta(U, dims, gauge: int = LANDAU) -> float:
    """Landau: eq. 2.5.  Coulomb: max over timeslices (C12)."""
    N, V = _dims(dims)
    return float(_load().orc_theta_report(N, gauge, _field(U, V)))


def theta_slices(U, dims, gauge: int = COULOMB) -> np.ndarray:
    N, V = _dims(dims)
    out = np.zeros(int(dims[3]), dtype=np.float64)
    _load().orc_theta(N, gauge, _field(U, V), out.ctypes.data)
    return out


def theta_mean(U, dims, gauge: int = LANDAU) -> float:
    """eq. 2.5 over the whole lattice for either gauge."""
    N, V = _dims(dims)
    return float(_load().orc_theta(N, gauge, _field(U, V), None))


# ---- pieces, exposed for the pins ----------------------------------------------------------------------
def site_overrelax(U, dims, s: int, omega: float, gauge: int = LANDAU) -> None:
    N, V = _dims(dims)
    _load().orc_site_overrelax(N, gauge, _field(U, V), int(s), float(omega))


def site_heatbath(U, dims, s: int, T: float, seed: int, step: int, gauge: int = LANDAU, buf=None) -> np.ndarray:
    """buf: optional (V, 3) int32 scratch for the trial counts, reused between calls on large lattices"""
    N, V = _dims(dims)
    tr = np.zeros((V, 3), dtype=np.int32) if buf is None else buf
    assert tr.shape == (V, 3) and tr.dtype == np.int32 and tr.flags.c_contiguous
    _load().orc_site_heatbath(N, gauge, _field(U, V), int(s), float(T), int(seed), int(step), tr.ctypes.data)
    return tr[s].copy()


def build_K(U, dims, s: int, gauge: int = LANDAU) -> np.ndarray:
    N, V = _dims(dims)
    K = np.zeros((3, 3), dtype=np.complex128)
    _load().orc_build_K(N, gauge, _field(U, V), int(s), K.ctypes.data)
    return K


def site_theta(U, dims, s: int, gauge: int = LANDAU) -> float:
    N, V = _dims(dims)
    return float(_load().orc_site_theta(N, gauge, _field(U, V), int(s)))


def su2_project(K, i: int, j: int) -> np.ndarray:
    K = np.ascontiguousarray(K, dtype=np.complex128)
    k = np.zeros(4)
    _load().orc_su2_project(K.ctypes.data, i, j, k.ctypes.data)
    return k


def su2_maximiser(k) -> np.ndarray:
    k = np.ascontiguousarray(k, dtype=np.float64)
    g = np.zeros(4)
    _load().orc_su2_maximiser(k.ctypes.data, g.ctypes.data)
    return g


def su2_overrelax(g, omega: float) -> np.ndarray:
    g = np.ascontiguousarray(g, dtype=np.float64)
    h = np.zeros(4)
    _load().orc_su2_overrelax(g.ctypes.data, float(omega), h.ctypes.data)
    return h


def quat_mul(p, q) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.float64)
    q = np.ascontiguousarray(q, dtype=np.float64)
    out = np.zeros(4)
    _load().orc_quat_mul(p.ctypes.data, q.ctypes.data, out.ctypes.data)
    return out


def su2_embed(q, i: int, j: int) -> np.ndarray:
    q = np.ascontiguousarray(q, dtype=np.float64)
    G = np.zeros((3, 3), dtype=np.complex128)
    _load().orc_su2_embed(q.ctypes.data, i, j, G.ctypes.data)
    return G


def plaquette(U, dims) -> float:
    N, V = _dims(dims)
    return float(_load().orc_plaquette(N, _field(U, V)))


def unitarity_defect(U, dims):
    N, V = _dims(dims)
    a, b = ctypes.c_double(), ctypes.c_double()
    _load().orc_unitarity_defect(N, _field(U, V), ctypes.byref(a), ctypes.byref(b))
    return a.value, b.value


def reunitarise(U, dims) -> None:
    N, V = _dims(dims)
    _load().orc_reunitarise(N, _field(U, V))


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    _load().orc_philox4x32_10(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


def kp_draw(alpha: float, key, c0: int, c1: int, c2: int):
    k = np.asarray(key, dtype=np.uint32)
    h = np.zeros(4)
    n = _load().orc_kp_draw(float(alpha), k.ctypes.data, int(c0), int(c1), int(c2), h.ctypes.data)
    return h, int(n)


# paper flop model, Alg. 1
FLOP_PROJECT, FLOP_OMEGA, FLOP_LEFT, FLOP_RIGHT = 60, 19, 84, 84
FLOP_PER_SUBGROUP = FLOP_PROJECT + FLOP_OMEGA + 4 * (FLOP_LEFT + FLOP_RIGHT)
FLOP_PER_SITE = 3 * FLOP_PER_SUBGROUP
