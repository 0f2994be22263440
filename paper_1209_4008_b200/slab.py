"""One configuration sharded in t over several slab contexts (the
checkerboard layout "opens the door to an efficient future multi-GPU parallelization").

No arithmetic of the method lives here: the half-sweeps, the face gather / scatter and the reductions run in the kernels
of libgf.so (``gf_create_slab, gf_relax_half, gf_anneal_half, gf_slab_pack_face, gf_slab_unpack_face, gf_raw_sums``); this
module is the schedule of one half-sweep and the transport of the face messages.

Decomposition: slab r owns the timeslices [t_r, t_{r+1}) (even bounds, so that its checkerboard is the global one) and
keeps a ghost copy of the temporal links of slice t_r - 1.  These are the only links a site update of slab r shares
with another slab: U_t(x - t) of the sites of its first slice, read for K(x) and multiplied by g(x)^dagger.  In a
half-sweep of parity p every link has exactly one active end (C6); the ghost links whose upper end is active start at
sites of parity 1 - p.  One half-sweep is therefore

    1. up:    slab r-1 sends the temporal links of its LAST slice, parity block 1-p  ->  ghost of slab r
    2. sweep: every slab updates the active sites of its slices (the first slice uses, and updates, the ghost)
    3. down:  slab r sends its ghost back                                           ->  last slice of slab r-1

(Nx Ny Nz / 2) * reals_per_link * sizeof(real) bytes per message: 1.18 MB at 32^3 fp32 R18, i.e. 1.5 us of an NVLink-5
direction (770 GB/s measured peer copy) against ~11 us for the half-sweep of a 32^3 x 4 slab.  With ``overlap`` the
interior slices are swept while the up message is in flight and only the first slice waits for it.

Transports: :class:`LocalRing` (all slabs in one process on one GPU: device-to-device copies stand in for the link -- the
form the one-GPU tests run) and :class:`DistRing` (one slab per rank, ``torch.distributed`` point-to-point: NCCL over
NVLink on a multi-GPU node, gloo in the CPU tests).  The engine behind a slab is anything with the methods of
:class:`GpuSlab`; tests drive the same schedule with a CPU engine built on the oracle.
"""
from __future__ import annotations

from typing import Dict, List, Sequence

UP, DOWN = +1, -1


def slab_bounds(Nt: int, nslabs: int) -> List[tuple]:
    """even-sized t-slabs, as equal as the evenness allows"""
    if nslabs < 1 or Nt % 2 or Nt < 2 * nslabs:
        raise ValueError(f"cannot cut {Nt} timeslices into {nslabs} slabs of an even number (>= 2) of slices")
    pairs = Nt // 2
    cuts = [2 * ((pairs * r) // nslabs) for r in range(nslabs + 1)]
    return [(cuts[r], cuts[r + 1]) for r in range(nslabs)]


# ---------------------------------------------------------------------------------------------------------
# transports: a message from every local slab to its upper (UP) or lower (DOWN) neighbour, periodic in t
# ---------------------------------------------------------------------------------------------------------
class LocalRing:
    """all slabs live in this process; a message is a device-to-device copy"""

    def __init__(self, nslabs: int):
        self.n = nslabs
        self.local_ranks = list(range(nslabs))

    def start(self, msgs: Dict[int, object], direction: int, recv_like: Dict[int, object]):
        out = {}
        for src, buf in msgs.items():
            dst = (src + direction) % self.n
            recv_like[dst].copy_(buf)
            out[dst] = recv_like[dst]
        return out

    def finish(self, handle):
        return handle

    def allreduce_sum(self, values: Dict[int, Sequence[float]]):
        keys = sorted(values)
        return [sum(values[k][i] for k in keys) for i in range(len(values[keys[0]]))]

    def allreduce_max(self, values: Dict[int, float]):
        return max(values.values())


class StreamRing(LocalRing):
    """all slabs live in this process, EACH ON ITS OWN CUDA STREAM (engines with a `.stream`): the copy that stands for a
    message runs on the receiver's stream behind an event the sender records after packing, so the interior launches of
    one slab really do overlap the face traffic and the launches of the others, and only the events order them -- what
    DistRing does across processes.  The sender then waits for the copy before it may reuse its send buffer."""

    def __init__(self, engines: Dict[int, object]):
        import torch

        super().__init__(len(engines))
        self.torch = torch
        self.stream = {r: e.stream for r, e in engines.items()}

    def start(self, msgs: Dict[int, object], direction: int, recv_like: Dict[int, object]):
        torch = self.torch
        out = {}
        for src, buf in msgs.items():
            dst = (src + direction) % self.n
            packed = torch.cuda.Event()
            packed.record(self.stream[src])
            self.stream[dst].wait_event(packed)
            with torch.cuda.stream(self.stream[dst]):
                recv_like[dst].copy_(buf)
            copied = torch.cuda.Event()
            copied.record(self.stream[dst])
            self.stream[src].wait_event(copied)
            out[dst] = recv_like[dst]
        return out


class DistRing:
    """one slab per rank of an initialised torch.distributed group; messages are point-to-point sends"""

    def __init__(self, group=None):
        import torch.distributed as dist

        self.dist = dist
        self.group = group
        self.rank = dist.get_rank(group)
        self.n = dist.get_world_size(group)
        self.local_ranks = [self.rank]

    def start(self, msgs: Dict[int, object], direction: int, recv_like: Dict[int, object]):
        dist = self.dist
        buf, recv = msgs[self.rank], recv_like[self.rank]
        if self.n == 1:
            recv.copy_(buf)
            return (None, recv)
        dst, src = (self.rank + direction) % self.n, (self.rank - direction) % self.n
        ops = [dist.P2POp(dist.isend, buf, dst, self.group), dist.P2POp(dist.irecv, recv, src, self.group)]
        return (dist.batch_isend_irecv(ops), recv)

    def finish(self, handle):
        reqs, recv = handle
        if reqs is not None:
            for r in reqs:
                r.wait()
        return {self.rank: recv}

    def allreduce_sum(self, values: Dict[int, Sequence[float]]):
        import torch

        v = values[self.rank]
        t = torch.tensor(list(v), dtype=torch.float64, device=self._device())
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return [float(x) for x in t.cpu()]

    def allreduce_max(self, values: Dict[int, float]):
        import torch

        t = torch.tensor([values[self.rank]], dtype=torch.float64, device=self._device())
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX, group=self.group)
        return float(t.cpu()[0])

    def _device(self):
        import torch

        return "cuda" if self.dist.get_backend(self.group) == "nccl" else "cpu"


# ---------------------------------------------------------------------------------------------------------
# the engine of one slab on the GPU: argument marshalling around the C ABI
# ---------------------------------------------------------------------------------------------------------
class GpuSlab:
    def __init__(self, dims, t_begin: int, t_end: int, precision="fp64", gauge="landau", reals_per_link: int = 18,
                 own_stream: bool = False):
        import torch

        import paper_1209_4008_b200 as gfm

        self.gfm, self.torch = gfm, torch
        self.stream = torch.cuda.Stream() if own_stream else None  # None: whatever stream is current at each call
        self.dims = tuple(int(d) for d in dims)
        self.t_begin, self.t_end, self.Nt = int(t_begin), int(t_end), int(t_end - t_begin)
        prec = {"fp32": gfm.GF_FP32, "fp64": gfm.GF_FP64}[precision]
        self.ctx = gfm.gf_create_slab(*self.dims[:3], self.dims[3], t_begin, t_end, prec,
                                      {"landau": gfm.GF_LANDAU, "coulomb": gfm.GF_COULOMB}[gauge])
        gfm.gf_set_storage(self.ctx, reals_per_link)
        self.U = torch.zeros(gfm.gf_field_bytes(self.ctx), dtype=torch.uint8, device="cuda")
        self.face_bytes = gfm.gf_slab_face_bytes(self.ctx)
        self.Vs = self.dims[0] * self.dims[1] * self.dims[2]

    def close(self):
        if self.ctx is not None:
            self.gfm.gf_destroy(self.ctx)
            self.ctx = None

    def new_face(self):
        return self.torch.empty(self.face_bytes, dtype=self.torch.uint8, device="cuda")

    def _on_stream(self):
        """context manager: the slab's own stream current (a no-op without one)"""
        import contextlib

        return self.torch.cuda.stream(self.stream) if self.stream is not None else contextlib.nullcontext()

    def load(self, U_canon_slab):
        """host numpy complex128 (Nt_local * Vs, 4, 3, 3): the owned slices in the canonical layout"""
        torch = self.torch
        dev = torch.from_numpy(U_canon_slab.view("float64").reshape(-1)).to("cuda")
        assert dev.numel() == self.Nt * self.Vs * 72
        torch.cuda.current_stream().synchronize()
        with self._on_stream():
            self.gfm.gf_pack(self.ctx, dev, self.U)
            torch.cuda.current_stream().synchronize()

    def download(self):
        torch = self.torch
        dev = torch.empty(self.Nt * self.Vs * 72, dtype=torch.float64, device="cuda")
        with self._on_stream():
            self.gfm.gf_unpack(self.ctx, self.U, dev)
            torch.cuda.current_stream().synchronize()
        return dev.cpu().numpy().view("complex128").reshape(self.Nt * self.Vs, 4, 3, 3)

    # the five methods of an engine
    def pack_face(self, which: int, block_parity: int, buf):
        with self._on_stream():
            self.gfm.gf_slab_pack_face(self.ctx, self.U, which, block_parity, buf)
        return buf

    def unpack_face(self, which: int, block_parity: int, buf):
        with self._on_stream():
            self.gfm.gf_slab_unpack_face(self.ctx, self.U, which, block_parity, buf)

    def half_sweep(self, kind, parity: int, sweep: int, t_first: int, t_count: int):
        with self._on_stream():
            if kind[0] == "anneal":
                self.gfm.gf_anneal_half(self.ctx, self.U, kind[1], parity, sweep, kind[2], t_first, t_count)
            else:
                self.gfm.gf_relax_half(self.ctx, self.U, kind[1], kind[2], parity, sweep, kind[3], t_first, t_count)

    def begin(self):
        with self._on_stream():
            self.gfm.gf_begin_sweeps(self.ctx)

    def raw_sums(self):
        with self._on_stream():
            return self.gfm.gf_raw_sums(self.ctx, self.U)

    def theta_slices(self):
        with self._on_stream():
            return self.gfm.gf_theta_slices(self.ctx, self.U, self.Nt)


# ---------------------------------------------------------------------------------------------------------
# the schedule
# ---------------------------------------------------------------------------------------------------------
class SlabRunner:
    """Runs sweeps on the local slabs of a ring.  engines: {rank: engine} for the ranks the transport calls local."""

    def __init__(self, engines: Dict[int, object], transport, dims, gauge: str = "landau", overlap: bool = True):
        self.eng, self.tr = engines, transport
        assert sorted(engines) == sorted(transport.local_ranks)
        self.dims = tuple(dims)
        self.V = dims[0] * dims[1] * dims[2] * dims[3]
        self.nd = 3 if gauge == "coulomb" else 4
        self.coulomb = gauge == "coulomb"
        self.overlap = overlap
        self.send = {r: e.new_face() for r, e in engines.items()}
        self.recv = {r: e.new_face() for r, e in engines.items()}

    def _shift(self, which_from: int, which_to: int, block_parity: int, direction: int, between=None):
        for r, e in self.eng.items():
            e.pack_face(which_from, block_parity, self.send[r])
        handle = self.tr.start(self.send, direction, self.recv)
        if between is not None:
            between()
        got = self.tr.finish(handle)
        for r, e in self.eng.items():
            e.unpack_face(which_to, block_parity, got[r])

    def half_sweep(self, kind, parity: int, sweep: int):
        bp = 1 - parity
        interior = None
        if self.overlap:  # the interior does not see the ghost: sweep it while the up message travels
            def interior():
                for e in self.eng.values():
                    e.half_sweep(kind, parity, sweep, 1, e.Nt - 1)
        self._shift(0, 1, bp, UP, interior)                       # last slice of r-1 -> ghost of r
        for e in self.eng.values():
            if self.overlap:
                e.half_sweep(kind, parity, sweep, 0, 1)
            else:
                e.half_sweep(kind, parity, sweep, 0, e.Nt)
        self._shift(1, 0, bp, DOWN)                               # ghost of r -> last slice of r-1

    def sweep(self, kind, sweep: int):
        self.half_sweep(kind, 0, sweep)  # RED, BLACK
        self.half_sweep(kind, 1, sweep)

    def begin(self):
        for e in self.eng.values():
            e.begin()

    def overrelax(self, omega: float, nsweeps: int, update: int = 0, seed: int = 0):
        self.begin()
        for s in range(nsweeps):
            self.sweep(("relax", update, omega, seed), s)

    def anneal(self, T_start: float, T_end: float, nsteps: int, seed: int):
        self.begin()
        for i in range(nsteps):
            T = T_start + (T_end - T_start) * i / (nsteps - 1) if nsteps > 1 else T_start  # C13
            self.sweep(("anneal", T, seed), i)

    def refresh_ghosts(self):
        """both parity blocks of the ghost, for theta of the first owned slice"""
        self._shift(0, 1, 0, UP)
        self._shift(0, 1, 1, UP)

    def functional_theta(self):
        """(F, theta) of the whole configuration: raw sums added over the slabs, normalised by the whole volume; Coulomb:
        theta = max over all timeslices (C12)"""
        self.refresh_ghosts()
        sums = self.tr.allreduce_sum({r: e.raw_sums() for r, e in self.eng.items()})
        F = sums[0] / (3.0 * self.nd * self.V)
        if self.coulomb:
            theta = self.tr.allreduce_max({r: max(e.theta_slices()) for r, e in self.eng.items()})
        else:
            theta = sums[1] / (3.0 * self.V)
        return F, theta

    def fix(self, omega: float, theta_tol: float, check_every: int = 100, max_sweeps: int = 100000, update: int = 0,
            seed: int = 0):
        """Alg. 1 with its stop rule (orc_fix): returns (sweeps, theta, F)"""
        done = 0
        self.begin()
        F, th = self.functional_theta()
        while th >= theta_tol and done < max_sweeps:
            n = min(check_every, max_sweeps - done)
            for s in range(done, done + n):
                self.sweep(("relax", update, omega, seed), s)
            done += n
            F, th = self.functional_theta()
        return done, th, F


def local_slabs(dims, nslabs: int, precision="fp64", gauge="landau", reals_per_link: int = 18, overlap: bool = True,
                streams: bool = False):
    """nslabs slab contexts of one configuration in this process (one GPU), wired into a :class:`SlabRunner`.
    streams = False: every launch and copy on the current stream (:class:`LocalRing`; the schedule's order only).
    streams = True: one CUDA stream per slab, face copies ordered by events (:class:`StreamRing`): the interior launches
    of a slab overlap the face traffic and the other slabs' launches, as they would across GPUs."""
    bounds = slab_bounds(dims[3], nslabs)
    engines = {r: GpuSlab(dims, b[0], b[1], precision, gauge, reals_per_link, own_stream=streams)
               for r, b in enumerate(bounds)}
    ring = StreamRing(engines) if streams else LocalRing(nslabs)
    return SlabRunner(engines, ring, dims, gauge, overlap), bounds


def dist_slab(dims, precision="fp64", gauge="landau", reals_per_link: int = 18, overlap: bool = True, group=None):
    """this rank's slab of one configuration sharded over the ranks of a torch.distributed group"""
    ring = DistRing(group)
    b = slab_bounds(dims[3], ring.n)[ring.rank]
    eng = GpuSlab(dims, b[0], b[1], precision, gauge, reals_per_link)
    return SlabRunner({ring.rank: eng}, ring, dims, gauge, overlap), b
