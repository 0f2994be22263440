"""N > 1 path of bench.py ("replicas only") on CPU: two gloo ranks, the max-over-ranks timing and
the whole-job value; plus the --impl reference arm's contract (rank 0 alone prints one JSON line)."""
import json
import os
import socket
import subprocess
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, out):
    import torch.distributed as dist

    import bench

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    local = 1.0 + 0.5 * rank  # rank 1 is the slow one
    total = bench.max_over_ranks(local, "cpu")
    out.put((rank, total, bench.whole_job_value(world, 256, 10, 3, total)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo_world2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    for rank, total, value in got:
        assert total == 1.5  # the slowest rank's time on every rank
        assert value == 2 * 256 * 10 * 3 / 1.5  # both replicas' site-updates over that time


def test_single_process_is_identity():
    import bench

    assert bench.max_over_ranks(0.25, "cpu") == 0.25
    assert bench.whole_job_value(1, 1048576, 100, 10, 0.2) == 1048576 * 100 * 10 / 0.2


def test_reference_arm_prints_one_json_line_rank0_only():
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
           "--ref-sweeps", "1", "--workload", "16^3x32-f64-r18"]
    res = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=600)
    assert res.returncode == 0, res.stderr
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["impl"] == "reference" and line["unit"] == "site-updates/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    env["RANK"] = "1"
    env["WORLD_SIZE"] = "2"
    res = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=600)
    assert res.returncode == 0 and res.stdout.strip() == ""
