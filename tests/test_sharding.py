"""Host logic of the one-process-per-GPU layout, on CPU: sample ranges tile the batch, and the
cross-rank reductions (max of device times, sums of tallies) work over a real 2-rank gloo group."""
import json
import os
import socket
import subprocess
import sys

import pytest

from paper_2311_17189_b200 import sharding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("n,world", [(0, 1), (1, 2), (10, 3), (1_000_003, 8), (7, 8)])
def test_shard_range_tiles_the_batch(n, world):
    nxt = 0
    sizes = []
    for r in range(world):
        first, cnt = sharding.shard_range(n, r, world)
        assert first == nxt and cnt >= 0
        nxt += cnt
        sizes.append(cnt)
    assert nxt == n and max(sizes) - min(sizes) <= 1


def test_weak_range_is_the_single_process_stream():
    assert [sharding.weak_range(1000, r, 4) for r in range(4)] == [(0, 1000), (1000, 1000), (2000, 1000), (3000, 1000)]
    with pytest.raises(ValueError):
        sharding.weak_range(10, 4, 4)
    with pytest.raises(ValueError):
        sharding.shard_range(10, -1, 2)


def test_reductions_without_a_group():
    assert sharding.max_over_ranks(1.5) == 1.5
    assert sharding.sum_over_ranks([1, 2.5]) == [1.0, 2.5]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        t = sharding.max_over_ranks(10.0 + rank, dist)
        first, cnt = sharding.shard_range(1001, rank, world)
        tot = sharding.sum_over_ranks([cnt, first * 0.5], dist)
        q.put((rank, t, tot))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_group():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, tot in got:
        assert t == 11.0                       # max over ranks
        assert tot == [1001.0, 0.5 * 501]      # counts add up to the batch; rank 1 starts at 501


def test_bench_reference_arm_two_ranks_prints_one_line():
    """bench.py --impl reference under torchrun (2 ranks, CPU): rank 0 alone runs the oracle and prints
    the JSON line; the other rank exits 0 without work."""
    env = dict(os.environ, OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference",
           "--gpus", "2", "--steps", "1", "--warmup", "0", "--cpu-seconds", "0.3", "--workload", "cfg1"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0


def test_bench_reference_arm_single_process():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                          "--warmup", "1", "--cpu-seconds", "0.3"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "impl"):
        assert key in d, key
    assert d["config"]["workload"] == "cfg3" and d["metric"] == "ami_term_evaluations_per_s" and d["steps"] == 2
