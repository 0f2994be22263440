#!/usr/bin/env python
"""bench.py -- throughput of the gauge-fixing hot path on B200, one JSON line on stdout (rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A STEP is one pass of the whole path at the paper's cadence (F and theta are evaluated after every
100th iteration): `--sweeps-per-step` (default 100) checkerboard overrelaxation sweeps (RED + BLACK half-sweeps,
Alg. 1) at omega, then gf_functional and gf_theta with their scalar read-back.
Metric: site-updates/s (one site-update = the full SU(3) update of one site: 3 SU(2) subgroups, 8 links);
GFlop/s = site-updates/s x 2253 (paper flop model).

Workloads (BASELINE.json configs; seeded synthetic fields, recipe in DESIGN.md "Inputs"):
    32^4-f32-r18 (default, the headline config), 32^4-f32-r12, 32^4-f64-r18, 32^4-f64-r12, 64^4-f64-r18, 64^4-f32-r18,
    16^3x32-f32-r18, 16^3x32-f64-r18, 48^3x64-f32-r18-coulomb, and the annealing sweeps 48^3x64-f32-r18-coulomb-anneal,
    48^3x64-f64-r18-coulomb-anneal, 32^4-f64-r18-anneal, 32^4-f32-r12-anneal
N > 1 (torchrun): by default every rank runs an independent replica of the workload on its own GPU ("replicas": the
shape of production gauge fixing, ensembles of configurations; no data-path collective); --shard t runs ONE
configuration cut into t-slabs over the ranks (paper_1209_4008_b200/slab.py: one face message up and one down per
half-sweep and slab boundary, strong scaling -- never run on more than one GPU so far: unmeasured).
value = site-updates of the whole job / max-over-ranks time.

--impl reference times the fp64 CPU oracle (oracle/, as it stands) on the host cores on the same config.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_SITE = 2253
L2_BYTES = 126 * 2**20

# name -> dims, precision, R, gauge, omega, generator (eps, seed), mode
WORKLOADS = {
    "32^4-f32-r18": dict(dims=(32, 32, 32, 32), precision="fp32", R=18, gauge="landau", omega=1.7, eps=0.4, seed=3),
    "32^4-f32-r12": dict(dims=(32, 32, 32, 32), precision="fp32", R=12, gauge="landau", omega=1.7, eps=0.4, seed=3),
    "32^4-f64-r18": dict(dims=(32, 32, 32, 32), precision="fp64", R=18, gauge="landau", omega=1.7, eps=0.4, seed=3),
    "32^4-f64-r12": dict(dims=(32, 32, 32, 32), precision="fp64", R=12, gauge="landau", omega=1.7, eps=0.4, seed=3),
    "64^4-f64-r18": dict(dims=(64, 64, 64, 64), precision="fp64", R=18, gauge="landau", omega=1.8, eps=0.4, seed=4),
    "64^4-f32-r18": dict(dims=(64, 64, 64, 64), precision="fp32", R=18, gauge="landau", omega=1.8, eps=0.4, seed=4),
    "16^3x32-f32-r18": dict(dims=(16, 16, 16, 32), precision="fp32", R=18, gauge="landau", omega=1.7, eps=0.3, seed=2),
    "16^3x32-f64-r18": dict(dims=(16, 16, 16, 32), precision="fp64", R=18, gauge="landau", omega=1.7, eps=0.3, seed=2),
    "48^3x64-f32-r18-coulomb": dict(dims=(48, 48, 48, 64), precision="fp32", R=18, gauge="coulomb", omega=1.7,
                                    eps=0.5, seed=5),
    "48^3x64-f32-r18-coulomb-anneal": dict(dims=(48, 48, 48, 64), precision="fp32", R=18, gauge="coulomb",
                                           omega=1.7, eps=0.5, seed=5, anneal=True),
    "48^3x64-f64-r18-coulomb-anneal": dict(dims=(48, 48, 48, 64), precision="fp64", R=18, gauge="coulomb",
                                           omega=1.7, eps=0.5, seed=5, anneal=True),
    "32^4-f64-r18-anneal": dict(dims=(32, 32, 32, 32), precision="fp64", R=18, gauge="landau", omega=1.7, eps=0.4, seed=3,
                                anneal=True),
    "32^4-f32-r12-anneal": dict(dims=(32, 32, 32, 32), precision="fp32", R=12, gauge="landau", omega=1.7, eps=0.4, seed=3,
                                anneal=True),
}
# further workloads timed after the main one in the default run (lattices above 32^4: at most 3 steps each)
ALSO_DEFAULT = ["32^4-f32-r12", "32^4-f64-r18", "32^4-f64-r12", "64^4-f32-r18", "64^4-f64-r18",
                "48^3x64-f32-r18-coulomb", "48^3x64-f32-r18-coulomb-anneal", "48^3x64-f64-r18-coulomb-anneal",
                "32^4-f64-r18-anneal", "32^4-f32-r12-anneal", "16^3x32-f32-r18", "16^3x32-f64-r18"]


def volume(dims):
    return dims[0] * dims[1] * dims[2] * dims[3]


def model_bytes_per_site_update(R: int, precision: str, gauge: str = "landau", anneal: bool = False) -> int:
    """every half-sweep reads and writes every link once (C6): 16 R s bytes per site-update.  Coulomb relaxation
    and annealing sweeps in fp32 run reading B (C12): 6 of the 8 links plus the 18-real g(x) field, (12 R + 36) s."""
    s = 8 if precision == "fp64" else 4
    if gauge == "coulomb" and precision == "fp32":
        return (12 * R + 36) * s  # annealing sweeps run reading B too
    return 16 * R * s


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------------------
# inputs: seeded synthetic fields from gf_inputs (host, canonical fp64).  Lattices above 32^4 sites are built
# by generating the field of half the extents and repeating it twice per direction (still a periodic gauge
# field of the same smoothness; keeps the default run's host time and memory bounded) -- named in `config`.
# ---------------------------------------------------------------------------------------------------------
def base_field(w):
    import gf_inputs

    dims = w["dims"]
    tiled = volume(dims) > 32**4
    gdims = tuple(d // 2 for d in dims) if tiled else dims
    U = gf_inputs.smooth_random(gdims, w["eps"], w["seed"])
    return U, gdims, tiled


def device_canonical(U, gdims, dims, tiled):
    """host canonical (numpy complex128 (V,4,3,3)) -> device float64 tensor of V*72 reals (tiled if asked)"""
    import torch

    t = torch.from_numpy(U.view("float64").reshape(-1)).to("cuda")
    if tiled:
        Nx, Ny, Nz, Nt = gdims
        t = t.view(Nt, Nz, Ny, Nx, 72).repeat(2, 2, 2, 2, 1).contiguous().view(-1)
    assert t.numel() == volume(dims) * 72
    return t


class ClockSampler:
    """SM clock, power and throttle reasons polled through NVML from a thread of this process (10 ms period), started
    before the warm-up; summary() reports the samples that fall inside the timed region (B200_PROFILING.md)"""

    def __init__(self, index: int):
        self.index = index
        self.samples = []  # (time.perf_counter(), sm MHz, power W, reasons bitmask)
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        self._err = None

    def start(self):
        try:
            import pynvml

            pynvml.nvmlInit()
            uuid_env = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            h = None
            if uuid_env and not uuid_env.split(",")[0].isdigit():
                try:
                    h = pynvml.nvmlDeviceGetHandleByUUID(uuid_env.split(",")[self.index].encode())
                except Exception:
                    h = None
            if h is None:
                phys = int(uuid_env.split(",")[self.index]) if uuid_env and uuid_env.split(",")[0].isdigit() else self.index
                h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
        except Exception as exc:  # NVML missing: report it, the run itself does not depend on it
            self._err = f"NVML unavailable: {exc}"
            return

        def poll():
            while not self._stop.is_set():
                try:
                    self.samples.append((time.perf_counter(), float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)),
                                         pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0,
                                         int(pynvml.nvmlDeviceGetCurrentClocksEventReasons(h))))
                except Exception:
                    pass
                self._stop.wait(0.01)

        self._thread = threading.Thread(target=poll, daemon=True)
        self._thread.start()

    def stop(self):
        self._stop.set()
        if self._thread is not None:
            self._thread.join(timeout=2)

    def summary(self, t0: float, t1: float):
        if self._err is not None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [self._err], "samples": 0}
        inside = [x for x in self.samples if t0 <= x[0] <= t1]
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}
        reasons = sorted({n for x in inside for bit, n in names.items() if x[3] & bit})
        sm = sorted(x[1] for x in inside)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.max_mhz,
                "power_w_max": max((x[2] for x in inside), default=None), "samples": len(inside),
                "samples_with_sw_power_cap": sum(1 for x in inside if x[3] & 0x4), "reasons": reasons,
                "how": "NVML polled every 10 ms in-process, samples inside the timed region"}


# ---------------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------------
def make_fixer(gfm, w, canon_dev):
    fx = gfm.GaugeFixer(w["dims"], precision=w["precision"], gauge=w["gauge"], reals_per_link=w["R"])
    gfm.gf_pack(fx.ctx, canon_dev, fx.U)
    return fx


def run_step(gfm, fx, w, sweeps, stream, ev=None):
    """one step: `sweeps` sweeps, then F and theta with their read-back.  ev = (start, stop) CUDA events recorded
    on `stream` around the sweep launches alone (roofline of the half-sweep kernel)."""
    if ev is not None:
        ev[0].record(stream)
    if w.get("anneal"):
        gfm.gf_anneal(fx.ctx, fx.U, 1.4, 0.01, sweeps, 7, stream)
    else:
        gfm.gf_overrelax(fx.ctx, fx.U, w["omega"], sweeps, stream)
    if ev is not None:
        ev[1].record(stream)
    return gfm.gf_functional(fx.ctx, fx.U), gfm.gf_theta(fx.ctx, fx.U)


def time_device(gfm, fx, w, sweeps, steps, warmup, stream, barrier=None, sampler=None):
    """W untimed steps, then K steps timed with CUDA events on the launching stream.
    Returns (seconds for K steps, seconds inside the sweep launches, launches, last F, last theta, clocks)."""
    import torch

    if sampler is not None:
        sampler.start()  # before the warm-up: the timed region of a fast workload is shorter than a sampler's start-up
    for _ in range(warmup):
        run_step(gfm, fx, w, sweeps, stream)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    if barrier is not None:
        barrier()
    launches0 = gfm.gf_launch_count(fx.ctx)
    fp32 = w["precision"] == "fp32"
    dc0 = gfm.gf_chain_count(fx.ctx) if fp32 else (0, 0)  # synchronises; outside the timed region
    h0 = time.perf_counter()
    t0.record(stream)
    for k in range(steps):
        F, th = run_step(gfm, fx, w, sweeps, stream, evs[k])
    t1.record(stream)
    torch.cuda.synchronize()
    h1 = time.perf_counter()
    clocks = None
    if sampler is not None:
        sampler.stop()
        clocks = sampler.summary(h0, h1)
    if barrier is not None:
        barrier()
    total = t0.elapsed_time(t1) * 1e-3
    in_sweeps = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
    dc1 = gfm.gf_chain_count(fx.ctx) if fp32 else (0, 0)
    # hybrid chain (fp32): launches / site updates of the TIMED region that ran in double
    time_device.double_chain = (dc1[0] - dc0[0], dc1[1] - dc0[1])
    return total, in_sweeps, gfm.gf_launch_count(fx.ctx) - launches0, F, th, clocks


def l2_copy_peak(nbytes: int) -> float:
    """GB/s (read + write) of a device copy whose source and destination together are the size of the field and stay in
    L2: the roof of a workload whose field is L2-resident (its half-sweep reads and writes the field once)"""
    import torch

    n = max(1, nbytes // 2 // 4)
    a = torch.empty(n, dtype=torch.float32, device="cuda").normal_()
    b = torch.empty_like(a)
    for _ in range(5):
        b.copy_(a)
    best = 0.0
    for _ in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(20):
            b.copy_(a)
        e1.record()
        torch.cuda.synchronize()
        best = max(best, 20 * 2 * n * 4 / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    return best


def roofline_entry(w, sweeps, steps, in_sweeps_s, traffic=None, total_s=None, l2_peak=None):
    """dominant kernel = the half-sweep kernel: algorithmic bytes per launch = (V/2) * 16 R s.
    achieved / frac: ALGORITHMIC bytes over the live CUDA-event duration, against the measured copy peak (for a field
    that fits L2: against a measured L2-resident copy of the same size).  dram_*: the same duration with the DRAM bytes
    one launch moved under ncu (profiles/r2_traffic.csv) -- below the algorithmic figure wherever L2 keeps part of the
    field between half-sweeps (32^4: 0.87 of the bytes; 64^4 and 48^3x64: 0.98-1.0)."""
    peak, which = measured_peaks()
    per_launch_bytes = (volume(w["dims"]) // 2) * model_bytes_per_site_update(w["R"], w["precision"], w["gauge"],
                                                                              bool(w.get("anneal")))
    nlaunch = 2 * sweeps * steps
    avg_s = in_sweeps_s / nlaunch
    achieved = per_launch_bytes / avg_s / 1e9
    out = {"bound": "hbm", "kernel": "gf_half_sweep_kernel", "achieved": round(achieved, 1), "peak": peak,
           "unit": "GB/s", "frac": round(achieved / peak, 4), "traffic": traffic,
           "bytes_per_launch": per_launch_bytes, "avg_launch_us": round(avg_s * 1e6, 3), "peak_source": which,
           "achieved_kind": "effective: algorithmic bytes / CUDA-event time",
           "frac_of_nominal_8TBs": round(achieved / 8000.0, 4),
           "share_of_step": round(in_sweeps_s / total_s, 4) if total_s else None}
    if traffic:
        dram = traffic / avg_s / 1e9
        out.update({"dram_achieved": round(dram, 1), "dram_frac": round(dram / peak, 4),
                    "dram_frac_of_nominal_8TBs": round(dram / 8000.0, 4),
                    "dram_kind": "ncu dram__bytes_read.sum + dram__bytes_write.sum of one launch / the live CUDA-event time"})
    if l2_peak:
        out.update({"bound": "l2", "peak": round(l2_peak, 1), "frac": round(achieved / l2_peak, 4),
                    "peak_source": "measured in this run: device copy with source + destination = field size, L2-resident "
                                   "(torch b.copy_(a), best of 5 x 20)", "hbm_peak": peak})
    return out


def max_over_ranks(seconds: float, device) -> float:
    """N > 1: the timed region of the job is the slowest rank's (the only collective on this path: replicas only)"""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return seconds
    tt = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def whole_job_value(world: int, V: int, sweeps: int, steps: int, seconds: float) -> float:
    """site-updates/s of the whole job: every rank sweeps its own replica (weak scaling, no data-path collective)"""
    return world * V * sweeps * steps / seconds


def time_e2e(gfm, w, hosts, sweeps, steps, warmup):
    """the host-buffer C-ABI call on an ensemble: gf_overrelax_host_batch -- H2D of every canonical field, pack, sweeps,
    F, theta, unpack, D2H, all inside the timed region; the copies of neighbouring configurations overlap the sweeps"""
    import torch

    prec = gfm.GF_FP64 if w["precision"] == "fp64" else gfm.GF_FP32
    ctx = gfm.gf_create(*w["dims"], prec, gfm.GF_COULOMB if w["gauge"] == "coulomb" else gfm.GF_LANDAU)
    gfm.gf_set_storage(ctx, w["R"])
    for _ in range(warmup):
        gfm.gf_overrelax_host_batch(ctx, hosts, w["omega"], sweeps)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        gfm.gf_overrelax_host_batch(ctx, hosts, w["omega"], sweeps)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    # the same through the single-configuration call (gf_overrelax_host / _f32): nothing overlaps the copies -- the
    # figure round 1 reported, kept so that the end-to-end numbers of the rounds stay comparable
    one = gfm.gf_overrelax_host_f32 if hosts[0].element_size() == 4 else gfm.gf_overrelax_host
    one(ctx, hosts[0], w["omega"], sweeps)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        one(ctx, hosts[0], w["omega"], sweeps)
    torch.cuda.synchronize()
    dt_single = time.perf_counter() - t0
    gfm.gf_destroy(ctx)
    nbytes = hosts[0].numel() * hosts[0].element_size()
    return dt, nbytes, nbytes + 16, dt_single


def time_oracle(w, U, sweeps, reps):
    """the oracle as it stands (gcc -O2 -fopenmp), fp64, on the host cores; returns seconds per repetition"""
    import oracle

    gauge = oracle.COULOMB if w["gauge"] == "coulomb" else oracle.LANDAU
    dims = w["dims"]
    oracle.overrelax(U, dims, w["omega"], 1, gauge)  # warm-up (page in, thread pool)
    t0 = time.perf_counter()
    for _ in range(reps):
        oracle.overrelax(U, dims, w["omega"], sweeps, gauge)
        oracle.functional(U, dims, gauge)
        oracle.theta(U, dims, gauge)
    return (time.perf_counter() - t0) / reps


def oracle_sample_dims(w):
    """lattice of the CPU legs: the workload's own lattice up to 32^4 sites (the oracle sweeps 32^4 in ~0.1 s on 16
    cores, so the reference arm runs the config it names); beyond that a bounded sample, the same generator on 16^3x32"""
    dims = w["dims"]
    if volume(dims) <= 32**4:
        return dims
    return (16, 16, 16, 32)


def main_reference(args, w, rank):
    """--impl reference: the oracle timed on the host cores, same config / metric / unit (rank 0 only)"""
    if rank != 0:
        return
    import gf_inputs
    import oracle

    sdims = oracle_sample_dims(w)
    ws = dict(w, dims=sdims)
    U = gf_inputs.smooth_random(sdims, w["eps"], w["seed"])
    sweeps = args.ref_sweeps
    for _ in range(args.warmup):
        time_oracle(ws, U, sweeps, 1)
    sec = time_oracle(ws, U, sweeps, args.steps)
    cores = oracle.max_threads()
    value = volume(sdims) * sweeps / sec
    sample = (f"{sweeps} sweeps + F + theta per step on " +
              ("the workload's own " if tuple(sdims) == tuple(w["dims"]) else "a bounded sample: a ") +
              f"{'x'.join(map(str, sdims))} lattice from the same generator (eps={w['eps']}, seed={w['seed']}), fp64")
    line = {
        "impl": "reference", "metric": "site-updates/s", "value": value, "unit": "site-updates/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "dims": list(w["dims"]), "gauge": w["gauge"], "omega": w["omega"],
                   "sample": sample, "sample_dims": list(sdims), "same_lattice": tuple(sdims) == tuple(w["dims"])},
        "gflops_paper_model": value * FLOP_PER_SITE / 1e9,
        "cpu_baseline": {"value": value, "unit": "site-updates/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "site-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    _print_json(line)


_JSON_FD = None


def _reserve_stdout():
    """Libraries (NCCL prints its version banner) write to stdout: keep fd 1 for the ONE JSON line by pointing it at
    stderr for the rest of the run and writing the line to the saved descriptor."""
    global _JSON_FD
    if _JSON_FD is None:
        sys.stdout.flush()
        _JSON_FD = os.dup(1)
        os.dup2(2, 1)


def _print_json(line: dict) -> None:
    data = (json.dumps(line) + "\n").encode()
    if _JSON_FD is None:
        sys.stdout.write(data.decode())
        sys.stdout.flush()
    else:
        os.write(_JSON_FD, data)


def field_bytes_of(wl):
    return 4 * volume(wl["dims"]) * wl["R"] * (8 if wl["precision"] == "fp64" else 4)


def main_shard(args, w, gfm, rank, world, local_rank, barrier, sweeps, steps, warmup):
    """--shard t: ONE configuration cut into t-slabs over the ranks (strong scaling).  Each rank holds
    its slab and a ghost slice; per half-sweep one face message goes up and one comes down per slab boundary
    (torch.distributed point-to-point over NCCL).  Unmeasured on multi-GPU hardware in this run (no such node)."""
    import numpy as np
    import torch

    import gf_inputs
    from paper_1209_4008_b200 import slab

    dims = w["dims"]
    if w.get("anneal"):
        raise SystemExit("bench.py --shard t: overrelaxation workloads only")
    gdims = tuple(d // 2 for d in dims) if volume(dims) > 32**4 else dims
    tiled = gdims != dims
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized():
        run, (t0, t1) = slab.dist_slab(dims, w["precision"], w["gauge"], w["R"], overlap=True)
    else:  # a plain one-GPU run: the whole lattice as one slab whose ghost is its own last slice
        run, bounds = slab.local_slabs(dims, 1, w["precision"], w["gauge"], w["R"])
        t0, t1 = bounds[0]
    U = gf_inputs.smooth_random(gdims, w["eps"], w["seed"])
    Vs = dims[0] * dims[1] * dims[2]
    if tiled:
        Nx, Ny, Nz, Nt = gdims
        U = np.tile(U.reshape(Nt, Nz, Ny, Nx, 4, 3, 3), (2, 2, 2, 2, 1, 1, 1)).reshape(-1, 4, 3, 3)
    eng = next(iter(run.eng.values()))
    eng.load(np.ascontiguousarray(U[t0 * Vs: t1 * Vs]))
    del U
    kind = ("relax", 0, w["omega"], 0)

    def step(s0):
        for s in range(s0, s0 + sweeps):
            run.sweep(kind, s)
        return run.functional_theta()

    run.begin()
    done = 0
    for _ in range(warmup):
        step(done)
        done += sweeps
    torch.cuda.synchronize()
    if barrier is not None:
        barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        F, th = step(done)
        done += sweeps
    e1.record()
    torch.cuda.synchronize()
    if barrier is not None:
        barrier()
    total = max_over_ranks(e0.elapsed_time(e1) * 1e-3, "cuda")
    if rank != 0:
        return
    V = volume(dims)
    value = V * sweeps * steps / total
    face = gfm.gf_slab_face_bytes(eng.ctx)
    _print_json({
        "metric": "site-updates/s", "value": value, "unit": "site-updates/s", "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": total / steps * 1e3, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64" if w["precision"] == "fp64" else "f32", "data": "synthetic",
        "config": {"workload": args.workload, "dims": list(dims), "gauge": w["gauge"], "reals_per_link": w["R"], "omega": w["omega"],
                   "step": f"{sweeps} overrelaxation sweeps + F + theta (all-reduce of two sums)",
                   "parallelism": f"one configuration in {world} t-slabs of {t1 - t0} timeslices; per half-sweep and slab boundary "
                                  f"one face of {face} bytes up and one down (torch.distributed P2P), interior swept meanwhile"},
        "gflops_paper_model": value * FLOP_PER_SITE / 1e9, "F": F, "theta": th, "gpu_launches": gfm.gf_launch_count(eng.ctx),
        "e2e": None, "roofline": None, "cpu_baseline": None,
    })


def main():
    _reserve_stdout()
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="32^4-f32-r18", choices=sorted(WORKLOADS))
    ap.add_argument("--sweeps-per-step", type=int, default=100)
    ap.add_argument("--ref-sweeps", type=int, default=5, help="sweeps per step of the --impl reference arm")
    ap.add_argument("--also", default=",".join(ALSO_DEFAULT), help="comma list of further workloads timed after "
                    "the main one and reported under 'also' ('' = none)")
    ap.add_argument("--tps", type=int, default=0, help="threads per site override (0 = library default)")
    ap.add_argument("--block", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-configs", type=int, default=12, help="configurations per step of the end-to-end (host buffer) leg")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "t"],
                    help="N > 1: independent replicas (default) or one configuration in t-slabs over the ranks")
    ap.add_argument("--traffic-csv", default=os.path.join(ROOT, "profiles", "r2_traffic.csv"),
                    help="ncu dram__bytes_read.sum / dram__bytes_write.sum per launch of the half-sweep kernel, per "
                         "workload (profiles/r2_traffic.md)")
    args = ap.parse_args()
    w = WORKLOADS[args.workload]

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        main_reference(args, w, rank)
        return

    import torch
    import paper_1209_4008_b200 as gfm

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path (use --impl reference for the oracle)")
    gfm.load_library()
    torch.cuda.set_device(local_rank)
    barrier = None
    under_torchrun = "RANK" in os.environ and "MASTER_ADDR" in os.environ
    if world > 1 or under_torchrun:  # one rank per GPU over NCCL; a 1-rank torchrun launch takes the same path
        import torch.distributed as dist

        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")  # NCCL logs to stdout by default: keep it to the JSON line
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        barrier = dist.barrier
    stream = torch.cuda.Stream()
    sweeps, steps, warmup = args.sweeps_per_step, args.steps, max(args.warmup, 3)

    if args.shard == "t":
        main_shard(args, w, gfm, rank, world, local_rank, barrier, sweeps, steps, warmup)
        if world > 1 or under_torchrun:
            dist.barrier()
            dist.destroy_process_group()
        return

    traffic = {}
    if os.path.exists(args.traffic_csv):
        import csv

        acc = {}
        with open(args.traffic_csv) as fh:
            for row in csv.DictReader(fh):
                acc.setdefault(row["workload"], []).append(float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]))
        traffic = {k: int(sum(v) / len(v)) for k, v in acc.items()}

    def measure(name, wl, sampler=None, bar=None, steps=steps):
        U, gdims, tiled = base_field(wl)
        canon = device_canonical(U, gdims, wl["dims"], tiled)
        fx = make_fixer(gfm, wl, canon)
        gfm.gf_set_tuning(fx.ctx, args.tps, args.block)
        del canon
        torch.cuda.synchronize()
        fits = field_bytes_of(wl) <= L2_BYTES
        total, in_sw, launches, F, th, clocks = time_device(gfm, fx, wl, sweeps, steps, warmup, stream, bar, sampler)
        regs, spill = gfm.gf_kernel_info(fx.ctx, 1 if wl.get("anneal") else 0)
        dc_launches, dc_sites = time_device.double_chain  # over the timed region only
        fx.close()
        del fx
        torch.cuda.empty_cache()
        l2_peak = l2_copy_peak(field_bytes_of(wl)) if fits else None
        return dict(U=U if not tiled else None, total=total, in_sweeps=in_sw, launches=launches, F=F, theta=th,
                    clocks=clocks, regs=regs, spill=spill, tiled=tiled, gdims=gdims, fits_l2=fits,
                    double_chain_launches=dc_launches, double_sites=dc_sites,
                    roofline=roofline_entry(wl, sweeps, steps, in_sw, None if fits else traffic.get(name), total, l2_peak))

    sampler = ClockSampler(local_rank) if rank == 0 else None
    m = measure(args.workload, w, sampler, barrier)
    total = max_over_ranks(m["total"], "cuda")
    V = volume(w["dims"])
    value = whole_job_value(world, V, sweeps, steps, total)

    if world > 1 or under_torchrun:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return

    # ---- rank 0, N = 1 extras: end-to-end through the host-buffer call, further workloads, the CPU baseline ----
    e2e = None
    if not args.no_e2e and not w.get("anneal"):
        import numpy as np

        U = m["U"] if m["U"] is not None else base_field(dict(w, dims=m["gdims"]))[0]
        if m["tiled"]:
            Nx, Ny, Nz, Nt = m["gdims"]
            U = np.tile(U.reshape(Nt, Nz, Ny, Nx, 4, 3, 3), (2, 2, 2, 2, 1, 1, 1)).reshape(-1, 4, 3, 3)
        # an ensemble of nconf configurations in pinned host memory; an fp32 context takes them as float, an fp64 one as double
        nconf = max(1, args.e2e_configs if field_bytes_of(w) < (2 << 30) else 2)
        base = torch.from_numpy(U.view("float64").reshape(-1))
        if w["precision"] == "fp32":
            base = base.to(torch.float32)
        hosts = [base.clone().pin_memory() for _ in range(nconf)]
        del base
        e_steps = max(1, min(steps, 3))
        dt, h2d, d2h, dt_single = time_e2e(gfm, w, hosts, sweeps, e_steps, 1)
        e2e = {"value": world * nconf * V * sweeps * e_steps / dt, "unit": "site-updates/s", "h2d_bytes_per_step": nconf * h2d,
               "d2h_bytes_per_step": nconf * d2h, "steps": e_steps, "ms_per_step": dt / e_steps * 1e3,
               "configurations_per_step": nconf, "ms_per_configuration": dt / e_steps / nconf * 1e3,
               "call": f"gf_overrelax_host_batch: {nconf} canonical configurations in pinned host memory in, the fixed fields + "
                       "F + theta out; upload of configuration i+1 and download of i-1 overlap the sweeps of i (three slots, "
                       "three streams); element type = the context's precision",
               "single_configuration": {
                   "value": world * V * sweeps * e_steps / dt_single, "unit": "site-updates/s",
                   "ms_per_step": dt_single / e_steps * 1e3, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "call": "gf_overrelax_host" + ("_f32" if w["precision"] == "fp32" else "") +
                           ": ONE configuration per step, copies not overlapped with the sweeps (round 1's e2e figure)"}}
        del hosts

    also = []
    for name in [n for n in args.also.split(",") if n and n != args.workload]:
        wl = WORKLOADS[name]
        Va = volume(wl["dims"])
        a_steps = min(steps, 5) if Va <= 32**4 else min(steps, 2)
        a = measure(name, wl, steps=a_steps)
        va = Va * sweeps * a_steps / a["total"]
        also.append({"workload": name, "value": va, "unit": "site-updates/s", "gflops_paper_model": va * FLOP_PER_SITE / 1e9,
                     "steps": a_steps, "ms_per_step": a["total"] / a_steps * 1e3,
                     "fits_l2": a["fits_l2"], "roofline": a["roofline"], "F": a["F"], "theta": a["theta"],
                     "regs_per_thread": a["regs"], "spill_bytes": a["spill"],
                     "gpu_launches": a["launches"], "double_chain_launches": a["double_chain_launches"],
                     "double_chain_fraction": a["double_chain_launches"] / max(1, 2 * sweeps * a_steps),
                     "sites_redone_in_double": a["double_sites"]})

    cpu = None
    if not args.no_cpu_baseline:
        import gf_inputs
        import oracle

        sdims = oracle_sample_dims(w)
        ws = dict(w, dims=sdims)
        Us = gf_inputs.smooth_random(sdims, w["eps"], w["seed"])
        probe = time_oracle(ws, Us, 1, 1)
        n = max(1, min(200, int(15.0 / max(probe, 1e-3))))  # about 15 s of CPU work
        sec = time_oracle(ws, Us, n, 1)
        cpu = {"value": volume(sdims) * n / sec, "unit": "site-updates/s", "cores": oracle.max_threads(), "kind": "oracle",
               "sample": f"{n} sweeps + F + theta on " + ("the workload's own " if tuple(sdims) == tuple(w["dims"]) else "a ") +
                         f"{'x'.join(map(str, sdims))} lattice from the same generator "
                         f"(eps={w['eps']}, seed={w['seed']}), fp64, gcc -O2 -fopenmp"}

    field_bytes = field_bytes_of(w)
    if field_bytes <= L2_BYTES:
        l2_note = f"field {field_bytes / 2**20:.0f} MiB fits L2 (126 MiB): roofline against a measured L2-resident copy, not HBM"
    elif field_bytes <= 4 * L2_BYTES:
        l2_note = (f"inputs larger than L2: field {field_bytes / 2**20:.0f} MiB vs 126 MiB L2, no flush; L2-ASSISTED: the "
                   "evict-last stores keep part of the field dirty in L2 between half-sweeps, the DRAM bytes of a launch are "
                   "~0.87 of the algorithmic ones (roofline.dram_*); the 64^4 workloads in `also` are the L2-free figures")
    else:
        l2_note = f"inputs larger than L2: field {field_bytes / 2**20:.0f} MiB vs 126 MiB L2, no flush"
    line = {
        "metric": "site-updates/s", "value": value, "unit": "site-updates/s", "n_gpus": world, "steps": steps,
        "warmup": warmup, "ms_per_step": total / steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64" if w["precision"] == "fp64" else "f32", "data": "synthetic",
        "config": {
            "workload": args.workload, "dims": list(w["dims"]), "gauge": w["gauge"], "reals_per_link": w["R"],
            "omega": w["omega"], "step": f"{sweeps} {'annealing' if w.get('anneal') else 'overrelaxation'} sweeps + "
                                         "gf_functional + gf_theta",
            "input": f"smooth-random eps={w['eps']} seed={w['seed']}" + (" on half extents, repeated 2x per direction"
                                                                          if m["tiled"] else ""),
            "l2": l2_note,
            "parallelism": "replicas only" if world > 1 else "single GPU",
        },
        "gflops_paper_model": value * FLOP_PER_SITE / 1e9,
        "paper_context": "300 GFlops on GTX 580 (PAPER.md:13), another machine: context, not the target",
        "F": m["F"], "theta": m["theta"],
        "regs_per_thread": m["regs"], "spill_bytes": m["spill"],
        "double_chain_launches": m["double_chain_launches"],  # of the 2 * sweeps * steps half-sweep launches timed
        "double_chain_fraction": m["double_chain_launches"] / max(1, 2 * sweeps * steps),
        "roofline": m["roofline"], "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": m["launches"],
        "clocks": m["clocks"], "also": also,
    }
    _print_json(line)


if __name__ == "__main__":
    main()
