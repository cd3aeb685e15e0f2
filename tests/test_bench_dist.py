"""N > 1 plumbing of bench.py on CPU (gloo, world size 2): the path does not shard in this build
(replicas only), so the only cross-rank step is the MAX of the per-rank
times; the reference arm runs on rank 0 alone."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert bench.dist_env() == (rank, rank, world)
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, torch.device("cpu"))
        q.put((rank, ms))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert out == [(0, 15.0), (1, 15.0)]  # every rank sees the slowest rank's time


def test_reference_arm_runs_on_rank0_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 1 exits 0 silently, rank 0 prints the line."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--config", "0", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--config", "0", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0, r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "builds/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


def _shard_worker(rank, world, port, q):
    import ctypes as C
    import types

    import numpy as np
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2004_10811_b200 import binding as B
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # the scalar all-reduce the library calls once per mu step of a sharded plan
        cb = B.make_allreduce(device="cpu")
        vals = (C.c_double * 2)(1.0 + rank, 10.0 * rank)
        cb(None, vals, 2)
        # every rank derives the same chunks from the same sizes (host function of the C-ABI)
        dims = np.arange(1, 41, dtype=np.int32) * 7
        first = B.sm_partition_groups(dims, world)
        # all-gather of D~: unequal contiguous value ranges, one per rank
        bounds = [0, 3, 8]
        info = types.SimpleNamespace(shard_val_begin=bounds[rank], shard_val_end=bounds[rank + 1])
        t = torch.full((8,), -1.0, dtype=torch.float64)
        t[bounds[rank]:bounds[rank + 1]] = rank + 1.0
        B.allgather_result(t, info)
        q.put((rank, list(vals), first.tolist(), t.tolist()))
    finally:
        dist.destroy_process_group()


def test_sharded_reduction_and_allgather_gloo_world2():
    """SURVEY 8(f)4 plumbing on CPU: the library's all-reduce callback, the partition and the all-gather of
    the result columns, two ranks over gloo."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, vals, first, t in out:
        assert vals == [3.0, 10.0]
        assert first == out[0][2] and first[0] == 0 and first[-1] == 40 and 0 < first[1] < 40
        assert t == [1.0, 1.0, 1.0, 2.0, 2.0, 2.0, 2.0, 2.0]
