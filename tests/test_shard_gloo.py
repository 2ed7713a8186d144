"""The N>1 path of bench.py on CPU: world_size-2 gloo.  The PLIC path has no exchange step --
cells are independent -- so multi-GPU is contiguous range sharding with no data-path
collective; the only collective is the MAX-over-ranks reduction of the timing."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import gen


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        N = 100000 + 37
        lo, hi = gen.shard_range(N, rank, world)
        shard = gen.random_sphere(hi - lo, seed=1, start=lo)
        # weak-scaling plan of bench.py: rank r owns cells [r*per, (r+1)*per) of the stream
        wlo, whi = bench.rank_cells(per_rank=5000, rank=rank)
        t = bench.max_over_ranks(10.0 + rank, device="cpu")
        total = bench.sum_over_ranks(hi - lo, device="cpu")
        q.put((rank, lo, hi, shard[1][:5].tolist(), float(np.sum(shard[0], dtype=np.float64)),
               wlo, whi, t, total))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_and_timing_reduction():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    N = 100000 + 37
    full = gen.random_sphere(N, seed=1)
    (r0, lo0, hi0, head0, sum0, wlo0, whi0, t0, tot0), (r1, lo1, hi1, head1, sum1, wlo1, whi1, t1, tot1) = res
    assert (lo0, hi1) == (0, N) and hi0 == lo1 and hi0 % 32 == 0
    assert head0 == full[1][:5].tolist() and head1 == full[1][lo1:lo1 + 5].tolist()
    assert abs((sum0 + sum1) - float(np.sum(full[0], dtype=np.float64))) < 1e-6
    assert (wlo0, whi0, wlo1, whi1) == (0, 5000, 5000, 10000)
    assert t0 == t1 == 11.0                     # MAX over ranks
    assert tot0 == tot1 == N


def test_bench_gpus_2_spawns_two_ranks():
    """`python bench.py --gpus 2` without torchrun re-launches itself with two ranks;
    --plumbing-only keeps the run on CPU (gloo): rendezvous, per-rank cell ranges, MAX / SUM reductions."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--plumbing-only"],
                         capture_output=True, text=True, timeout=300, env=env)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                  # rank 0 alone prints
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["ranks"] == 2 and out["cells"] == 2 * 4096
    assert out["max_over_ranks"] == 2.0                     # MAX over the ranks' timings 1.0, 2.0
    full = gen.random_sphere(2 * 4096, seed=1)
    assert abs(out["checksum"] - float(np.sum(full[0], dtype=np.float64))) < 1e-6   # contiguous ranges, no overlap
