"""World-size-2 gloo test (CPU) of bench.py's multi-rank host logic: request sharding (disjoint cover, no exchange),
max-over-ranks timing, whole-job sums, and that only rank 0 runs the `--impl reference` arm."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class _HostClock:
    """Stands in for bench.DeviceClock (CUDA events) where there is no GPU: same interface, host time."""

    def mark(self):
        import time
        return time.perf_counter()

    def ms(self, a, b):
        return (b - a) * 1e3

    def sync(self):
        pass


class _StubWorkload:
    """What bench.run() needs of a workload: step(i, mark) with four phase boundaries, launches(), bytes per phase.  The
    phases just sleep - rank 1 twice as long as rank 0 - so the max-over-ranks reductions have something to choose."""

    def __init__(self, rank, world):
        import bench
        self.ids = bench.rank_requests(rank, world, per_gpu=5)
        self.rank, self.n = rank, 0
        self.bytes_a, self.bytes_b, self.bytes_c = 1000.0 * (rank + 1), 10.0, 100.0

    def launches(self):
        return 3 * self.n

    def step(self, i, mark=None):
        import time
        mark = mark or (lambda k: None)
        mark(0)
        for k in (1, 2, 3):
            time.sleep(0.004 * (self.rank + 1))
            mark(k)
        self.n += 1


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import argparse
    import contextlib
    import io

    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    mine = bench.rank_requests(rank, world, per_gpu=5)
    gathered = [None] * world
    dist.all_gather_object(gathered, mine)
    t_max = bench.max_over_ranks(1.5 + rank, world)              # device time of the slowest rank
    b_sum = bench.sum_over_ranks(100.0 * (rank + 1), world)      # whole-job bytes
    # the rank-aware part of bench.main() itself - timed region between barriers, reductions, rank-0 line - on a stub workload
    wl = _StubWorkload(rank, world)
    info = {"n_layers": 2, "n_req": 5, "n_chunks": 8, "window_tokens": 64, "bytes_a": wl.bytes_a, "bytes_b": wl.bytes_b, "bytes_c": wl.bytes_c,
            "decode_launch": "stub"}
    buf = io.StringIO()
    with contextlib.redirect_stdout(buf):
        line = bench.run(argparse.Namespace(steps=4, warmup=1), world, rank, wl, _HostClock(), info)
    dist.barrier()
    q.put((rank, mine, gathered, t_max, b_sum, line, buf.getvalue(), wl.n))
    dist.destroy_process_group()


def test_world_size_2_sharding_and_reductions():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mine, gathered, t_max, b_sum, line, printed, n_steps in res:
        assert gathered[rank] == mine
        flat = [x for g in gathered for x in g]
        assert sorted(flat) == list(range(world * 5)) and len(set(flat)) == len(flat)     # disjoint cover
        assert t_max == 2.5                     # max over ranks, identical on every rank
        assert b_sum == 300.0
        assert n_steps == 5                     # 1 warm-up + exactly 4 timed steps on every rank
        if rank != 0:
            assert line is None and printed == ""                  # only rank 0 prints
            continue
        assert json.loads(printed.strip()) == line
        assert line["n_gpus"] == 2 and line["steps"] == 4 and line["scaling"] == "weak" and line["gpu_launches"] == 3
        # value = ALL ranks' phase-A bytes (1000 + 2000) / the SLOWEST rank's phase-A time (rank 1: >= 8 ms per step)
        ms_a = line["phases_ms"]["relocate_patch_batch"]
        assert ms_a >= 8.0 and abs(line["value"] - 3000.0 / (ms_a * 1e-3) / 1e9) < 1e-9 * line["value"]
        assert line["ms_per_step"] >= 3 * 8.0 and line["decode_tok_per_s"] == 2 * 5 / (line["phases_ms"]["decode_all_layers"] * 1e-3)
        # the per-kernel roofline entries are this rank's own (bytes and time of rank 0), not the job's
        assert line["roofline_all"]["kam_relocate_patch_kernel"]["ms_per_launch"] < ms_a
    assert torch.distributed.is_available()


def test_single_rank_reductions_are_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.25, 1) == 3.25 and bench.sum_over_ranks(7.0, 1) == 7.0
    assert bench.rank_requests(0, 1, per_gpu=4) == [0, 1, 2, 3]


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env["RANK"] = "0"; env["LOCAL_RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "GB/s"
