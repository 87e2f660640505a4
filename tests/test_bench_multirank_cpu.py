"""The N > 1 path of bench.py on CPU: world_size-2 gloo.  The path does not shard (DESIGN.md §10,
"replicas only"), so what N > 1 adds is the rendezvous, the barrier and the max-over-ranks of the
per-rank step time; those are exercised here without a GPU."""
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
    assert c1["parallelism"] == "single GPU" and c2["parallelism"] == "replicas only"
