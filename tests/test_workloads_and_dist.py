"""Seeded input recipes (determinism, shapes, value ranges) and the multi-process host logic of
bench.py on the CPU (gloo, world_size 2): replicas only, max-over-ranks timing."""
import os
import sys

import numpy as np
import pytest

from paper_1306_5076_b200 import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_workloads_are_deterministic_and_prefix_stable():
    a = workloads.cfg3_sort_u32(n=4096)
    b = workloads.cfg3_sort_u32(n=8192)
    assert a.dtype == np.uint32 and np.array_equal(a, b[:4096])
    assert np.array_equal(a, workloads.cfg3_sort_u32(n=4096))
    assert not np.array_equal(a, workloads.cfg1_tiles_u32(num_tiles=4))


def test_config_shapes_and_ranges():
    k, v = workloads.cfg2_tiles_u32_u32(num_tiles=4)
    assert k.max() < 16 and np.array_equal(v, np.arange(4096, dtype=np.uint32))
    n = 1 << 14
    assert np.array_equal(workloads.cfg4_sort_u32("sorted", n), np.arange(n, dtype=np.uint32))
    assert np.array_equal(workloads.cfg4_sort_u32("reverse", n), np.arange(n, dtype=np.uint32)[::-1])
    assert np.unique(workloads.cfg4_sort_u32("dup256", 1 << 16)).size == 256
    z = workloads.cfg4_sort_u32("zipf", 1 << 18)
    assert z.max() < (1 << 20)
    assert 0.10 < (z == 0).mean() < 0.15          # key 0 is ~12.4 % of a Zipf(1.1) input over 2^20 ranks
    assert 0.34 < (z < 16).mean() < 0.41          # keys < 16 are ~37.5 %
    k, v = workloads.cfg5a_sort_u64_u32(n=1 << 16)
    assert k.dtype == np.uint64 and np.unique(k).size < (1 << 16) * 0.55 + 1024
    keys, run_len = workloads.cfg5b_merge_runs_u32(64, n=1 << 14)
    runs = keys.reshape(64, run_len)
    assert np.all(runs[:, :-1] <= runs[:, 1:])


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 * (rank + 1), world)
    keys = bench.replica_keys(workloads.cfg3_sort_u32(n=4096), rank)
    gathered = [None] * world
    dist.all_gather_object(gathered, (int(keys[0]), int(keys.astype(np.uint64).sum())))
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ms, gathered))


def test_bench_host_logic_world_size_2_gloo():
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, gathered in res:
        assert ms == 20.0                              # the slowest rank's time, on every rank
        assert gathered[0] != gathered[1]              # replicas sort different inputs


def test_bench_reference_arm_runs_on_rank0_only():
    sys.path.insert(0, ROOT)
    import bench

    class A:
        workload, log2n, steps, warmup, gpus = "cfg3", 12, 1, 0, 2
    assert bench.run_reference(A, rank=1, world=2) is None   # other ranks exit without work
