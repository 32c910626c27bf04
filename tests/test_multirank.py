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


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    mine = bench.rank_requests(rank, world, per_gpu=5)
    gathered = [None] * world
    dist.all_gather_object(gathered, mine)
    t_max = bench.max_over_ranks(1.5 + rank, world)              # device time of the slowest rank
    b_sum = bench.sum_over_ranks(100.0 * (rank + 1), world)      # whole-job bytes
    dist.barrier()
    q.put((rank, mine, gathered, t_max, b_sum))
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
    for rank, mine, gathered, t_max, b_sum in res:
        assert gathered[rank] == mine
        flat = [x for g in gathered for x in g]
        assert sorted(flat) == list(range(world * 5)) and len(set(flat)) == len(flat)     # disjoint cover
        assert t_max == 2.5                     # max over ranks, identical on every rank
        assert b_sum == 300.0
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
