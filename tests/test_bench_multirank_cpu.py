"""The N > 1 path on CPU: world_size-2 gloo.  What N > 1 adds to the single-GPU path is the
rendezvous, the barrier, the max-over-ranks of the per-rank step time, the target-slice bookkeeping and the
all-gather of the acceleration slices; those are exercised here without a GPU."""
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist          # noqa: E402
import torch.multiprocessing as mp        # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert bench._env_rank() == (rank, rank, world)
        dist.barrier()
        mine = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
        got = bench.reduce_max_ms(mine, world, device="cpu")
        out[rank] = got
        # one rank reports: the others print nothing (bench.py prints on rank 0 only)
        assert bench.reduce_max_ms(3.0, 1, device="cpu") == 3.0
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    world, port = 2, _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    assert dict(out) == {0: 15.0, 1: 15.0}


def test_config_is_shared_by_both_arms():
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    from paper_1807_08116_b200 import workloads as wl
    w = wl.make_workload(0, scale=0.125)
    a = argparse.Namespace(config=0)
    c1 = bench.workload_config(a, w, [3, 4, 5], 60, 1)
    c2 = bench.workload_config(a, w, [3, 4, 5], 60, 2)
    assert c1["workload"] == c2["workload"] and "configs[0]" in c1["workload"]
    assert c1["parallelism"] == "single GPU" and "N/2 per GPU" in c2["parallelism"]


# ---------------------------------------------------------------- NEXT-4: slices and the exchange (host logic)
def test_slice_bounds_cover_and_align():
    sys.path.insert(0, ROOT)
    from paper_1807_08116_b200.sharded import slice_bounds, SLICE_ALIGN
    for n in (0, 1, 1023, 1024, 1025, 8192, 2 ** 20, 2 ** 20 + 7, 4194304):
        for world in (1, 2, 3, 4, 8):
            covered, chunk0 = 0, None
            for r in range(world):
                i0, i1, chunk = slice_bounds(n, r, world)
                chunk0 = chunk0 or chunk
                assert chunk == chunk0 and chunk % SLICE_ALIGN == 0 and world * chunk >= n
                assert i0 == min(r * chunk, n) and i0 <= i1 <= n and i1 - i0 <= chunk
                assert i0 == covered                     # contiguous, in rank order, no gaps, no overlap
                covered = i1
            assert covered == n
    with pytest.raises(ValueError):
        slice_bounds(10, 2, 2)


def _gather_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    from paper_1807_08116_b200.sharded import slice_bounds, allgather_rows
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n = 2500                                          # ragged: rank 1's slice is short
        i0, i1, chunk = slice_bounds(n, rank, world)
        full = torch.full((world * chunk, 4), -1.0)       # stale values everywhere
        rows = torch.arange(i0, i1, dtype=torch.float32)
        full[i0:i1] = torch.stack([rows, 2 * rows, 3 * rows, torch.zeros_like(rows)], 1)   # "my slice of acc_grav"
        allgather_rows(full, rank, world, chunk)
        out[rank] = full[:n].clone().numpy()
    finally:
        dist.destroy_process_group()


def test_allgather_rows_gloo_world2():
    import numpy as np
    world, port = 2, _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_gather_worker, args=(world, port, out), nprocs=world, join=True)
    rows = np.arange(2500, dtype=np.float32)
    expect = np.stack([rows, 2 * rows, 3 * rows, np.zeros_like(rows)], 1)
    assert np.array_equal(out[0], expect) and np.array_equal(out[1], expect)     # every rank holds every row


def _reduce_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    from paper_1807_08116_b200.sharded import allreduce_sums
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # "my share of the fixed-point sums": values near +-2^62 so that a float detour would lose bits, and
        # wrap-around (two's complement) must behave like the device's unsigned adds
        base = torch.arange(3 * 2048, dtype=torch.int64)
        mine = (base * 1315423911 + (2 ** 61 + 12345) * (1 if rank == 0 else -1)) * (rank + 1)
        allreduce_sums(mine, world)
        out[rank] = mine.clone().numpy()
    finally:
        dist.destroy_process_group()


def test_allreduce_sums_gloo_world2():
    """The exchange of the pair-symmetric path: an exact int64 SUM, identical on every rank."""
    import numpy as np
    world, port = 2, _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_reduce_worker, args=(world, port, out), nprocs=world, join=True)
    base = np.arange(3 * 2048, dtype=np.int64)
    with np.errstate(over="ignore"):
        expect = (base * 1315423911 + (2 ** 61 + 12345)) * 1 + (base * 1315423911 - (2 ** 61 + 12345)) * 2
    assert np.array_equal(out[0], expect) and np.array_equal(out[1], expect)
