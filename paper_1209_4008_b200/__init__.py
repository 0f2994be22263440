"""paper_1209_4008_b200 -- thin Python binding of libgf.so (include/gf.h).

Lattice gauge fixing of SU(3) gauge fields by checkerboard overrelaxation and SU(2)-heatbath simulated annealing
(Schroeck & Vogt, arXiv:1209.4008) on one NVIDIA B200.  Every step of the method runs in the CUDA kernels of
``csrc/``; this module only marshals arguments.  PyTorch supplies device memory and streams, nothing else.
There is no CPU path: without the compiled library or without a CUDA device the calls raise.

The functions carry the names of the C ABI: ``gf_create, gf_overrelax, gf_anneal, gf_functional, gf_theta`` (plus
``gf_pack / gf_unpack / gf_theta_slices / gf_overrelax_host`` and the tuning calls).  :class:`GaugeFixer` is a
small convenience wrapper that owns a context and a native field.
"""
from __future__ import annotations

import ctypes
import os

GF_FP32, GF_FP64 = 0, 1
GF_LANDAU, GF_COULOMB = 0, 1
GF_OK, GF_EINVAL, GF_ECUDA, GF_ENOMEM = 0, -1, -2, -3
GF_UPDATE_OVERRELAX2, GF_UPDATE_OVERRELAX1, GF_UPDATE_STOCHASTIC = 0, 1, 2

# paper flop model, Alg. 1: 60 + 19 + 4*(84+84) = 751 per subgroup, 2253 per site
FLOP_PER_SITE = 3 * (60 + 19 + 4 * (84 + 84))

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgf.so")

# every symbol include/gf.h declares: name -> (restype, argtypes)
_vp, _i, _d, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
_ull = ctypes.c_ulonglong
_pd, _pi = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
SIGNATURES = {
    "gf_create": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _i, _i, _i]),
    "gf_destroy": (None, [_vp]),
    "gf_last_error": (ctypes.c_char_p, [_vp]),
    "gf_set_storage": (_i, [_vp, _i]),
    "gf_field_bytes": (_sz, [_vp]),
    "gf_pack": (_i, [_vp, _vp, _vp, _vp]),
    "gf_unpack": (_i, [_vp, _vp, _vp, _vp]),
    "gf_convert": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "gf_overrelax": (_i, [_vp, _vp, _d, _i, _vp]),
    "gf_anneal": (_i, [_vp, _vp, _d, _d, _i, _ull, _vp]),
    "gf_relax": (_i, [_vp, _vp, _i, _d, _i, _ull, _vp]),
    "gf_anneal_micro": (_i, [_vp, _vp, _d, _d, _i, _i, _ull, _vp]),
    "gf_fix": (_i, [_vp, _vp, _i, _d, _d, _i, _i, _ull, _pi, _pd, _pd, _vp]),
    "gf_fix_slices": (_i, [_vp, _vp, _i, _d, _d, _i, _i, _ull, _pi, _pi, _pd, _pd, _vp]),
    "gf_functional": (_i, [_vp, _vp, _pd]),
    "gf_theta": (_i, [_vp, _vp, _pd]),
    "gf_theta_slices": (_i, [_vp, _vp, _pd]),
    "gf_overrelax_host": (_i, [_vp, _vp, _d, _i, _pd, _pd]),
    "gf_overrelax_host_f32": (_i, [_vp, _vp, _d, _i, _pd, _pd]),
    "gf_overrelax_host_batch": (_i, [_vp, ctypes.POINTER(_vp), _i, _i, _d, _i, _pd, _pd]),
    "gf_set_tuning": (_i, [_vp, _i, _i]),
    "gf_set_reunit": (_i, [_vp, _i]),
    "gf_set_l2_reversal": (_i, [_vp, _i]),
    "gf_set_l2_policy": (_i, [_vp, _i, _i]),
    "gf_set_pdl": (_i, [_vp, _i]),
    "gf_set_prefetch": (_i, [_vp, _i]),
    "gf_set_coulomb_reading": (_i, [_vp, _i]),
    "gf_create_slab": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _i, _i, _i, _i, _i]),
    "gf_slab_face_bytes": (_sz, [_vp]),
    "gf_slab_pack_face": (_i, [_vp, _vp, _i, _i, _vp, _vp]),
    "gf_slab_unpack_face": (_i, [_vp, _vp, _i, _i, _vp, _vp]),
    "gf_begin_sweeps": (_i, [_vp, _vp]),
    "gf_relax_half": (_i, [_vp, _vp, _i, _d, _i, _i, _ull, _i, _i, _vp]),
    "gf_anneal_half": (_i, [_vp, _vp, _d, _i, _i, _ull, _i, _i, _vp]),
    "gf_raw_sums": (_i, [_vp, _vp, _pd, _pd]),
    "gf_set_monitor": (_i, [_vp, _i]),
    "gf_monitor_last": (_i, [_vp, _pi, _pd, _pd, _pd]),
    "gf_fix_last_form": (_i, [_vp, _pi, _pi]),
    "gf_set_chain": (_i, [_vp, _i, _d, _d]),
    "gf_chain_count": (_i, [_vp, ctypes.POINTER(_ull), ctypes.POINTER(_ull)]),
    "gf_set_trial_buffer": (_i, [_vp, _vp]),
    "gf_launch_count": (_ull, [_vp]),
    "gf_kernel_info": (_i, [_vp, _i, _pi, _pi]),
    "gf_debug_kp_math": (_i, [_vp, _i, _vp, _vp, _vp, _vp]),
    "gf_theta_static": (_i, [_i, _i, _i, _i, _i, _i, _i, _vp, _vp, _vp, ctypes.c_char_p, _sz]),
    "gf_theta_static_max_partials": (_sz, []),
}

_lib = None


class GFError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"libgf error {code}: {message}")
        self.code = code


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree libgf.so (build it with ``python -m paper_1209_4008_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1209_4008_b200.build` "
                "(there is no CPU fallback)"
            )
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(ctx, rc: int) -> None:
    if rc != GF_OK:
        msg = load_library().gf_last_error(ctx)
        raise GFError(rc, msg.decode() if msg else "")


def _ptr(t) -> int:
    """device (or host) address of a torch tensor / numpy array / int"""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _stream(stream) -> int:
    if stream is None:
        import torch

        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


# ---- the C ABI, one Python function per call -------------------------------------------------------------
def gf_create(Nx: int, Ny: int, Nz: int, Nt: int, precision: int = GF_FP64, gauge: int = GF_LANDAU):
    lib = load_library()
    ctx = _vp()
    rc = lib.gf_create(ctypes.byref(ctx), Nx, Ny, Nz, Nt, precision, gauge)
    _check(None, rc)
    return ctx


def gf_create_slab(Nx: int, Ny: int, Nz: int, Nt_global: int, t_begin: int, t_end: int, precision: int = GF_FP64,
                   gauge: int = GF_LANDAU):
    lib = load_library()
    ctx = _vp()
    _check(None, lib.gf_create_slab(ctypes.byref(ctx), Nx, Ny, Nz, Nt_global, t_begin, t_end, precision, gauge))
    return ctx


def gf_slab_face_bytes(ctx) -> int:
    return int(load_library().gf_slab_face_bytes(ctx))


def gf_slab_pack_face(ctx, U, which: int, block_parity: int, buf, stream=None) -> None:
    _check(ctx, load_library().gf_slab_pack_face(ctx, _ptr(U), int(which), int(block_parity), _ptr(buf), _stream(stream)))


def gf_slab_unpack_face(ctx, U, which: int, block_parity: int, buf, stream=None) -> None:
    _check(ctx, load_library().gf_slab_unpack_face(ctx, _ptr(U), int(which), int(block_parity), _ptr(buf), _stream(stream)))


def gf_begin_sweeps(ctx, stream=None) -> None:
    _check(ctx, load_library().gf_begin_sweeps(ctx, _stream(stream)))


def gf_relax_half(ctx, U, update: int, param: float, parity: int, sweep: int, seed: int, t_first: int, t_count: int,
                  stream=None) -> None:
    _check(ctx, load_library().gf_relax_half(ctx, _ptr(U), int(update), float(param), int(parity), int(sweep), int(seed),
                                            int(t_first), int(t_count), _stream(stream)))


def gf_anneal_half(ctx, U, T: float, parity: int, step: int, seed: int, t_first: int, t_count: int, stream=None) -> None:
    _check(ctx, load_library().gf_anneal_half(ctx, _ptr(U), float(T), int(parity), int(step), int(seed), int(t_first),
                                             int(t_count), _stream(stream)))


def gf_raw_sums(ctx, U):
    """(F_raw, theta_raw) over the owned sites"""
    a, b = ctypes.c_double(), ctypes.c_double()
    _check(ctx, load_library().gf_raw_sums(ctx, _ptr(U), ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


def gf_destroy(ctx) -> None:
    load_library().gf_destroy(ctx)


def gf_set_storage(ctx, reals_per_link: int) -> None:
    _check(ctx, load_library().gf_set_storage(ctx, reals_per_link))


def gf_field_bytes(ctx) -> int:
    return int(load_library().gf_field_bytes(ctx))


def gf_pack(ctx, U_canon_dev, U_native_dev, stream=None) -> None:
    _check(ctx, load_library().gf_pack(ctx, _ptr(U_canon_dev), _ptr(U_native_dev), _stream(stream)))


def gf_unpack(ctx, U_native_dev, U_canon_dev, stream=None) -> None:
    _check(ctx, load_library().gf_unpack(ctx, _ptr(U_native_dev), _ptr(U_canon_dev), _stream(stream)))


def gf_convert(src_ctx, U_src, dst_ctx, U_dst, stream=None) -> None:
    _check(dst_ctx, load_library().gf_convert(src_ctx, _ptr(U_src), dst_ctx, _ptr(U_dst), _stream(stream)))


def gf_overrelax(ctx, U, omega: float, nsweeps: int, stream=None) -> None:
    _check(ctx, load_library().gf_overrelax(ctx, _ptr(U), float(omega), int(nsweeps), _stream(stream)))


def gf_anneal(ctx, U, T_start: float, T_end: float, nsteps: int, seed: int, stream=None) -> None:
    _check(ctx, load_library().gf_anneal(ctx, _ptr(U), float(T_start), float(T_end), int(nsteps), int(seed),
                                        _stream(stream)))


def gf_relax(ctx, U, update: int, param: float, nsweeps: int, seed: int = 0, stream=None) -> None:
    _check(ctx, load_library().gf_relax(ctx, _ptr(U), int(update), float(param), int(nsweeps), int(seed),
                                       _stream(stream)))


def gf_anneal_micro(ctx, U, T_start: float, T_end: float, nsteps: int, n_micro: int, seed: int, stream=None) -> None:
    _check(ctx, load_library().gf_anneal_micro(ctx, _ptr(U), float(T_start), float(T_end), int(nsteps), int(n_micro),
                                              int(seed), _stream(stream)))


def gf_fix(ctx, U, update: int, param: float, theta_tol: float, check_every: int, max_sweeps: int, seed: int = 0,
           stream=None):
    """Alg. 1 with its stop rule; returns (sweeps done, theta, F)"""
    n, th, F = ctypes.c_int(), ctypes.c_double(), ctypes.c_double()
    _check(ctx, load_library().gf_fix(ctx, _ptr(U), int(update), float(param), float(theta_tol), int(check_every),
                                     int(max_sweeps), int(seed), ctypes.byref(n), ctypes.byref(th), ctypes.byref(F),
                                     _stream(stream)))
    return n.value, th.value, F.value


def gf_fix_slices(ctx, U, Nt: int, update: int, param: float, theta_tol: float, check_every: int, max_sweeps: int,
                  seed: int = 0, stream=None):
    """Coulomb gauge, stop rule per timeslice; returns (max sweeps, theta, F, list of sweeps per slice)"""
    n, th, F = ctypes.c_int(), ctypes.c_double(), ctypes.c_double()
    per = (ctypes.c_int * Nt)()
    _check(ctx, load_library().gf_fix_slices(ctx, _ptr(U), int(update), float(param), float(theta_tol),
                                            int(check_every), int(max_sweeps), int(seed), ctypes.byref(n), per,
                                            ctypes.byref(th), ctypes.byref(F), _stream(stream)))
    return n.value, th.value, F.value, list(per)


def gf_functional(ctx, U) -> float:
    out = ctypes.c_double()
    _check(ctx, load_library().gf_functional(ctx, _ptr(U), ctypes.byref(out)))
    return out.value


def gf_theta(ctx, U) -> float:
    out = ctypes.c_double()
    _check(ctx, load_library().gf_theta(ctx, _ptr(U), ctypes.byref(out)))
    return out.value


def gf_theta_slices(ctx, U, Nt: int):
    out = (ctypes.c_double * Nt)()
    _check(ctx, load_library().gf_theta_slices(ctx, _ptr(U), out))
    return list(out)


def gf_theta_static(dims, precision: int, gauge: int, reals_per_link: int, U, out_dev, stream=None) -> None:
    """theta without a context and without any allocation inside the library (include/gf.h, gf_theta_static): for host
    programs that own all of the GPU's memory themselves or must not stall the device on an allocation.  ``U``: native
    field (device), ``out_dev``: Nt + 2 doubles on the device, written asynchronously on ``stream``: [0] theta of the
    lattice, [1] max over timeslices, [2 + t] theta_t.  The scratch is one fixed 1 MiB array per GPU shared by all
    calls: lattices needing more than ``gf_theta_static_max_partials()`` block partials raise GFError(GF_EINVAL), and
    calls that overlap on the GPU race.  Make the first call on a device at set-up, before any stream capture."""
    err = ctypes.create_string_buffer(512)
    rc = load_library().gf_theta_static(int(dims[0]), int(dims[1]), int(dims[2]), int(dims[3]), int(precision), int(gauge),
                                        int(reals_per_link), _ptr(U), _ptr(out_dev), _stream(stream), err, len(err))
    if rc != GF_OK:
        raise GFError(rc, err.value.decode())


def gf_theta_static_max_partials() -> int:
    return int(load_library().gf_theta_static_max_partials())


def gf_overrelax_host(ctx, U_canon_host, omega: float, nsweeps: int):
    """U_canon_host: host array (numpy complex128 (V,4,3,3) or a pinned torch tensor), updated in place.
    Returns (F, theta) after the last sweep."""
    F, th = ctypes.c_double(), ctypes.c_double()
    _check(ctx, load_library().gf_overrelax_host(ctx, _ptr(U_canon_host), float(omega), int(nsweeps),
                                                ctypes.byref(F), ctypes.byref(th)))
    return F.value, th.value


def gf_overrelax_host_f32(ctx, U_canon_host, omega: float, nsweeps: int):
    """as gf_overrelax_host with the canonical field held as float32 (numpy complex64 (V,4,3,3) or pinned tensor)"""
    F, th = ctypes.c_double(), ctypes.c_double()
    _check(ctx, load_library().gf_overrelax_host_f32(ctx, _ptr(U_canon_host), float(omega), int(nsweeps),
                                                    ctypes.byref(F), ctypes.byref(th)))
    return F.value, th.value


def gf_overrelax_host_batch(ctx, U_canon_hosts, omega: float, nsweeps: int):
    """U_canon_hosts: list of host arrays (numpy complex128 / complex64 (V,4,3,3), or pinned torch tensors of float64 /
    float32), all of one element type, each updated in place.  Returns ([F], [theta])."""
    n = len(U_canon_hosts)
    if n == 0:
        return [], []
    first = U_canon_hosts[0]
    itemsize = first.element_size() if hasattr(first, "element_size") else first.dtype.itemsize
    elem = 4 if itemsize in (4,) or str(getattr(first, "dtype", "")) in ("complex64", "torch.float32") else 8
    ptrs = (_vp * n)(*[_ptr(u) for u in U_canon_hosts])
    F, th = (ctypes.c_double * n)(), (ctypes.c_double * n)()
    _check(ctx, load_library().gf_overrelax_host_batch(ctx, ptrs, n, elem, float(omega), int(nsweeps), F, th))
    return list(F), list(th)


def gf_set_tuning(ctx, threads_per_site: int = 0, block: int = 0) -> None:
    _check(ctx, load_library().gf_set_tuning(ctx, threads_per_site, block))


def gf_set_reunit(ctx, every: int) -> None:
    _check(ctx, load_library().gf_set_reunit(ctx, every))


def gf_set_l2_reversal(ctx, on: bool) -> None:
    _check(ctx, load_library().gf_set_l2_reversal(ctx, int(bool(on))))


def gf_set_l2_policy(ctx, load_policy: int, store_policy: int) -> None:
    _check(ctx, load_library().gf_set_l2_policy(ctx, int(load_policy), int(store_policy)))


def gf_set_pdl(ctx, on: bool) -> None:
    _check(ctx, load_library().gf_set_pdl(ctx, int(bool(on))))


def gf_set_prefetch(ctx, sites: int) -> None:
    _check(ctx, load_library().gf_set_prefetch(ctx, int(sites)))


def gf_set_coulomb_reading(ctx, reading_b: bool) -> None:
    _check(ctx, load_library().gf_set_coulomb_reading(ctx, -1 if reading_b is None else int(bool(reading_b))))


def gf_set_monitor(ctx, fused: int) -> None:
    """0: separate check kernel, 1: fused where it applies and pays (default), 2: fused wherever it applies"""
    _check(ctx, load_library().gf_set_monitor(ctx, int(fused)))


def gf_monitor_last(ctx, Nt: int):
    """last check of a fused fixing loop: (sweep n, theta, F, [theta_t]) of the state after sweep n"""
    n, th, F = ctypes.c_int(), ctypes.c_double(), ctypes.c_double()
    sl = (ctypes.c_double * Nt)()
    _check(ctx, load_library().gf_monitor_last(ctx, ctypes.byref(n), ctypes.byref(th), ctypes.byref(F), sl))
    return n.value, th.value, F.value, list(sl)


def gf_fix_last_form(ctx):
    """(lag, fused) of the last gf_fix / gf_fix_slices on this context: lag 0 = the paper's stop rule, 1 = one sweep
    after the check that met the tolerance (C21); fused 1 = the sweep kernels monitored theta themselves, 0 = separate
    check kernel.  (-1, -1) before the first call."""
    lag, fused = ctypes.c_int(), ctypes.c_int()
    _check(ctx, load_library().gf_fix_last_form(ctx, ctypes.byref(lag), ctypes.byref(fused)))
    return lag.value, fused.value


def gf_set_chain(ctx, chain: int, watch_threshold: float = 0.0, fix_threshold: float = 0.0) -> None:
    """fp32 contexts: 0 = fp32 site chain, 1 = double, 2 = hybrid (default); thresholds of 0 keep the current values"""
    _check(ctx, load_library().gf_set_chain(ctx, int(chain), float(watch_threshold), float(fix_threshold)))


def gf_chain_count(ctx):
    """(half-sweep launches that ran the double chain, site updates redone in double) since gf_create"""
    a, b = _ull(), _ull()
    _check(ctx, load_library().gf_chain_count(ctx, ctypes.byref(a), ctypes.byref(b)))
    return int(a.value), int(b.value)


def gf_set_trial_buffer(ctx, d_trials) -> None:
    _check(ctx, load_library().gf_set_trial_buffer(ctx, _ptr(d_trials)))


def gf_debug_kp_math(words_dev, neglog_dev=None, sin_dev=None, cos_dev=None, stream=None) -> None:
    """-ln u, sin(2 pi u), cos(2 pi u) of the uniforms of the given Philox words (device uint32 / float64 tensors)"""
    rc = load_library().gf_debug_kp_math(_ptr(words_dev), int(words_dev.numel()), _ptr(neglog_dev) if neglog_dev is not None else None,
                                         _ptr(sin_dev) if sin_dev is not None else None,
                                         _ptr(cos_dev) if cos_dev is not None else None, _stream(stream))
    if rc != GF_OK:
        raise GFError(rc, "gf_debug_kp_math")


def gf_launch_count(ctx) -> int:
    return int(load_library().gf_launch_count(ctx))


def gf_kernel_info(ctx, mode: int = 0):
    regs, loc = ctypes.c_int(), ctypes.c_int()
    _check(ctx, load_library().gf_kernel_info(ctx, mode, ctypes.byref(regs), ctypes.byref(loc)))
    return regs.value, loc.value


# ---- convenience wrapper ---------------------------------------------------------------------------------
class GaugeFixer:
    """Owns a gf_ctx and one native field on the current CUDA device.

    >>> gf = GaugeFixer((32, 32, 32, 32), precision="fp32", reals_per_link=12)
    >>> gf.load(U)                      # numpy complex128 (V,4,3,3), canonical layout
    >>> gf.overrelax(1.7, 100); gf.theta(), gf.functional()
    >>> U_fixed = gf.download()
    """

    def __init__(self, dims, precision="fp64", gauge="landau", reals_per_link: int = 18):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1209_4008_b200 needs a CUDA device (there is no CPU path)")
        self.dims = tuple(int(d) for d in dims)
        self.V = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        self.precision = {"fp32": GF_FP32, "fp64": GF_FP64}[precision] if isinstance(precision, str) else precision
        self.gauge = {"landau": GF_LANDAU, "coulomb": GF_COULOMB}[gauge] if isinstance(gauge, str) else gauge
        self.R = int(reals_per_link)
        self.ctx = gf_create(*self.dims, self.precision, self.gauge)
        gf_set_storage(self.ctx, self.R)
        self.nbytes = gf_field_bytes(self.ctx)
        self.U = torch.empty(self.nbytes, dtype=torch.uint8, device="cuda")
        self._torch = torch

    def close(self):
        if self.ctx is not None:
            gf_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # field transfer
    def load(self, U_canon):
        """host numpy complex128 (V,4,3,3) or device float64 tensor with V*72 elements -> native field"""
        torch = self._torch
        if not isinstance(U_canon, torch.Tensor):
            U_canon = torch.from_numpy(U_canon.view("float64").reshape(-1))
        dev = U_canon.to("cuda", non_blocking=False).contiguous()
        assert dev.dtype == torch.float64 and dev.numel() == self.V * 72
        gf_pack(self.ctx, dev, self.U)
        torch.cuda.current_stream().synchronize()

    def download(self):
        """native field -> host numpy complex128 (V,4,3,3)"""
        torch = self._torch
        dev = torch.empty(self.V * 72, dtype=torch.float64, device="cuda")
        gf_unpack(self.ctx, self.U, dev)
        return dev.cpu().numpy().view("complex128").reshape(self.V, 4, 3, 3)

    def convert_to(self, precision=None, gauge=None, reals_per_link=None) -> "GaugeFixer":
        """a new GaugeFixer holding this field in another precision / storage (mixed-precision fixing)"""
        other = GaugeFixer(self.dims, self.precision if precision is None else precision,
                           self.gauge if gauge is None else gauge,
                           self.R if reals_per_link is None else reals_per_link)
        gf_convert(self.ctx, self.U, other.ctx, other.U)
        return other

    # the method
    def overrelax(self, omega: float, nsweeps: int, stream=None):
        gf_overrelax(self.ctx, self.U, omega, nsweeps, stream)

    def anneal(self, T_start: float, T_end: float, nsteps: int, seed: int, stream=None, n_micro: int = 0):
        gf_anneal_micro(self.ctx, self.U, T_start, T_end, nsteps, n_micro, seed, stream)

    def fix(self, theta_tol: float, update: int = GF_UPDATE_OVERRELAX2, param: float = 1.7, check_every: int = 100,
            max_sweeps: int = 100000, seed: int = 0, stream=None):
        return gf_fix(self.ctx, self.U, update, param, theta_tol, check_every, max_sweeps, seed, stream)

    def fix_slices(self, theta_tol: float, update: int = GF_UPDATE_OVERRELAX2, param: float = 1.7,
                   check_every: int = 100, max_sweeps: int = 100000, seed: int = 0, stream=None):
        return gf_fix_slices(self.ctx, self.U, self.dims[3], update, param, theta_tol, check_every, max_sweeps, seed,
                             stream)

    def relax(self, update: int, param: float, nsweeps: int, seed: int = 0, stream=None):
        gf_relax(self.ctx, self.U, update, param, nsweeps, seed, stream)

    def functional(self) -> float:
        return gf_functional(self.ctx, self.U)

    def theta(self) -> float:
        return gf_theta(self.ctx, self.U)

    def theta_slices(self):
        return gf_theta_slices(self.ctx, self.U, self.dims[3])
