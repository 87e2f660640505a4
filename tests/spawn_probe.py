"""Helper of tests/test_bench_multirank_cpu.py::test_bench_launch_ranks_world2_gloo (not a test itself): what one rank
of `bench.py --gpus N` does, with the GPU parts replaced — gloo for NCCL and the recording stand-in for the library —
so that the launch path (bench.launch_ranks -> torch.distributed.run -> RANK / WORLD_SIZE from the environment ->
rendezvous -> sharded steps -> barrier -> max over ranks -> one JSON line from rank 0) runs on CPU."""
import argparse
import json
import os
import sys
from types import SimpleNamespace

import numpy as np
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import bench                                                    # noqa: E402
from paper_1807_08116_b200.sharded import ShardedSimulation     # noqa: E402
from test_bench_multirank_cpu import _StubBinding               # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", required=True)
    args = ap.parse_args()
    rank, local_rank, world = bench._env_rank()
    dist.init_process_group("gloo")                             # env:// rendezvous, as under the driver's torchrun
    n = 2500
    w = SimpleNamespace(n_gas=1000, n_halo=1500, n_total=n, h=0.1, dt=1e-3, posm=np.zeros((n, 4), np.float32),
                        vele=np.zeros((n, 4), np.float32))
    stub = _StubBinding(True)
    sim = ShardedSimulation(w, rank, world, binding=stub, device="cpu")
    sim.step()
    dist.barrier()
    ms = bench.reduce_max_ms(10.0 + 5.0 * rank, world, device="cpu")
    seen = [None] * world
    dist.all_gather_object(seen, rank)
    if rank == 0:
        with open(args.out, "a") as f:
            f.write(json.dumps({"n_gpus": world, "value": ms, "ranks_seen": seen, "calls": stub.calls,
                                "parallelism": bench.parallelism_text(world, sim.path)}) + "\n")
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
