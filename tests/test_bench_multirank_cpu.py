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
    assert c1["parallelism"] == "single GPU" and "one collective per evaluation" in c2["parallelism"]
    # the text follows the path the device chose: work items + int64 all-reduce, or target slices + all-gather
    sym = bench.workload_config(a, w, [3, 4, 5], 60, 2, "pair_symmetric")["parallelism"]
    one = bench.workload_config(a, w, [3, 4, 5], 60, 2, "one_sided_uniform")["parallelism"]
    assert "int64 SUM all-reduce" in sym and "all-gather" not in sym
    assert "all-gather" in one and "int64" not in one and "N/2 per GPU" in one
    assert "no gravity collective" in bench.workload_config(a, w, [3, 4, 5], 60, 2, "none")["parallelism"]
    # the SPH passes are shared as well: tiles of the sorted order + an all-reduce of rho and of acc_sph per pass
    assert "int32 SUM all-reduce of rho" in sym and "int32 SUM all-reduce of rho" in one


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


class _StubBinding:
    """Stands in for the C-ABI face in the world-2 test of ShardedSimulation's exchange: no arithmetic of the method —
    each share call writes rank-tagged values where the library would (the fixed-point sums, the rank's acceleration
    rows), the finish call records what it was handed."""

    class sph_params:                                   # noqa: N801 (mirrors binding.sph_params)
        G = 1.0

        @classmethod
        def from_workload(cls, w):
            return cls()

    def __init__(self, pair_symmetric):
        self.pair_symmetric, self.calls, self.seen = pair_symmetric, [], None

    def sph_grid_from_bbox(self, posm, n_gas, h):
        return "grid"

    def sph_gravity_path(self, ws, n_gas, n, grid):
        self.calls.append("path")
        return "pair_symmetric" if self.pair_symmetric else "one_sided"

    def alloc_workspace(self, n_gas, n, grid):
        return torch.zeros(64 + 24 * 4096, dtype=torch.uint8)

    def gravity_sums_view(self, ws, n_gas, n, grid):
        return ws[64:].view(torch.int64)

    def sph_position_share(self, posm, hsml, sigma, n_gas, n_halo, rank, world, i0, i1, params, grid, rho, acc_grav, ws):
        self.calls.append("share")
        sums = ws[64:].view(torch.int64)
        sums.zero_()
        if self.pair_symmetric:                         # this rank's part of the integer sums
            sums += (rank + 1) * (torch.arange(sums.numel(), dtype=torch.int64) - 2 ** 40)
        else:                                           # this rank's acceleration rows
            acc_grav[i0:i1] = float(rank + 1)

    def nbody_pp_gravity_finish(self, posm, n_gas, n_halo, grid, G, acc_grav, ws):
        self.calls.append("finish")
        self.seen = (ws[64:].view(torch.int64).clone(), acc_grav.clone())

    def sph_predict(self, *a):
        self.calls.append("predict")

    def sph_correct(self, *a):
        self.calls.append("correct")

    # ---- the SPH passes shared as well: the rank's targets (here: every world-th element) get a rank-tagged value, the
    # others ZERO, as the library writes them; the update call records what it was handed
    def sph_position_share_sph(self, posm, hsml, n_gas, n_halo, rank, world, i0, i1, params, grid, rho, acc_grav, ws):
        self.sph_position_share(posm, hsml, 0.0, n_gas, n_halo, rank, world, i0, i1, params, grid, rho, acc_grav, ws)
        self.calls[-1] = "share_sph"
        rho.zero_()
        rho[rank:n_gas:world] = 10.0 + rank

    def sph_forces_share(self, vele, hsml, n_gas, n_halo, rank, world, params, grid, rho, acc_sph, ws):
        self.calls.append("forces_share")
        self.rho_seen = rho.clone()
        acc_sph.zero_()
        acc_sph[rank:n_gas:world] = -1.5 - rank

    def sph_update(self, posm, vele, n_gas, n_halo, grid, dt, corrector, acc_sph, acc_grav, ws):
        self.calls.append("update1" if corrector else "update0")
        self.acc_sph_seen = acc_sph.clone()

    def sph_renew_hsml(self, *a):
        self.calls.append("renew_hsml")


def _sharded_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import numpy as np
    from types import SimpleNamespace
    from paper_1807_08116_b200.sharded import ShardedSimulation
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n = 2500
        w = SimpleNamespace(n_gas=1000, n_halo=1500, n_total=n, h=0.1, dt=1e-3, posm=np.zeros((n, 4), np.float32),
                            vele=np.zeros((n, 4), np.float32))
        res = {}
        for sym in (True, False):
            stub = _StubBinding(sym)
            sim = ShardedSimulation(w, rank, world, binding=stub, device="cpu", share_sph=False)
            sim.step()
            sums, acc = stub.seen
            res[sym] = (stub.calls, sums.numpy(), acc[:n].numpy(), (sim.i0, sim.i1))
        # the SPH passes shared as well (the default for world > 1), with per-particle smoothing lengths
        stub = _StubBinding(True)
        sim = ShardedSimulation(w, rank, world, binding=stub, device="cpu", sigma=1.3)
        assert sim.share_sph
        sim.step()
        res["sph"] = (stub.calls, stub.rho_seen.numpy(), stub.acc_sph_seen.numpy(), stub.seen[0].numpy())
        out[rank] = res
    finally:
        dist.destroy_process_group()


def test_sharded_step_exchange_gloo_world2():
    """The N > 1 step on CPU (gloo, world 2) with a stand-in for the library: per force evaluation every rank calls
    share -> path read-back -> the ONE collective that path needs -> finish, in that order, twice in the first step
    (seeding + the step); what finish sees is the SUM of the ranks' fixed-point parts (pair-symmetric path) or ALL
    ranks' acceleration rows (one-sided path), and the other buffer is NOT exchanged."""
    import numpy as np
    world, port = 2, _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_sharded_worker, args=(world, port, out), nprocs=world, join=True)
    k = np.arange(3 * 4096, dtype=np.int64) - 2 ** 40
    for rank in range(world):
        for sym in (True, False):
            calls, sums, acc, (i0, i1) = out[rank][sym]
            assert calls == ["share", "path", "finish", "predict", "share", "path", "finish", "correct"]
            if sym:
                assert np.array_equal(sums, 3 * k)                           # (1 + 2) * k: both ranks' parts, exact
                assert np.all(acc == 0)                                      # no all-gather on this path
            else:
                assert np.all(sums == 0)                                     # no all-reduce on this path
                b0 = out[0][sym][3]
                b1 = out[1][sym][3]
                assert b0[0] == 0 and b0[1] == b1[0] and b1[1] == 2500       # the slices tile [0, n)
                assert np.all(acc[b0[0]:b0[1]] == 1.0) and np.all(acc[b1[0]:b1[1]] == 2.0)
    assert np.array_equal(out[0][True][1], out[1][True][1]) and np.array_equal(out[0][False][2], out[1][False][2])
    # SPH passes shared: per evaluation share -> rho completed over the ranks (-> hsml renewed, after the seeding) ->
    # gravity exchange -> finish; per half step forces share -> acc_sph completed -> update.  What the forces and the
    # update calls see is EVERY rank's values, bit for bit (the all-reduce adds the bit patterns to zeros)
    for rank in range(world):
        calls, rho_seen, acc_seen, sums = out[rank]["sph"]
        assert calls == ["share_sph", "path", "finish", "forces_share", "update0",
                         "share_sph", "renew_hsml", "path", "finish", "forces_share", "update1"]
        assert np.array_equal(rho_seen[0:1000:2], np.full(500, 10.0, np.float32))
        assert np.array_equal(rho_seen[1:1000:2], np.full(500, 11.0, np.float32))
        assert np.array_equal(acc_seen[0:1000:2], np.full((500, 4), -1.5, np.float32))
        assert np.array_equal(acc_seen[1:1000:2], np.full((500, 4), -2.5, np.float32))
        assert np.array_equal(sums, 3 * k)


# ---------------------------------------------------------------- `python bench.py --gpus N` starts its own ranks
def test_bench_gpus_without_devices_fails_loudly():
    """On a box with fewer than N CUDA devices `python bench.py --gpus N` must refuse, not measure one GPU silently."""
    import subprocess
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        pytest.skip("box has 2 GPUs")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--config", "0"],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "needs 2 CUDA devices" in (r.stderr + r.stdout)
    # a launcher that started another number of ranks than --gpus says is refused as well
    env = dict(os.environ, RANK="0", WORLD_SIZE="4", LOCAL_RANK="0", MASTER_ADDR="127.0.0.1", MASTER_PORT="29999")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--config", "0"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode != 0 and "WORLD_SIZE=4" in (r.stderr + r.stdout)


def test_bench_launch_ranks_world2_gloo(tmp_path):
    """bench.launch_ranks — the code path `python bench.py --gpus 2` takes — started for 2 ranks on CPU: the probe
    script below is what bench.py's ranks do with the GPU parts replaced (gloo instead of NCCL, the recording stand-in
    instead of the library): rendezvous from the launcher's environment, ShardedSimulation steps with their collective,
    barrier, max over ranks, ONE JSON line from rank 0."""
    import json
    import subprocess
    sys.path.insert(0, ROOT)
    import bench
    out = tmp_path / "line.json"
    probe = os.path.join(ROOT, "tests", "spawn_probe.py")
    code = (f"import sys; sys.path.insert(0, {ROOT!r}); import bench; "
            f"sys.exit(bench.launch_ranks(2, {probe!r}, ['--out', {str(out)!r}], check_devices=False))")
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in open(out).read().splitlines() if ln.strip()]
    assert len(lines) == 1                                   # rank 0 alone reports
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["ranks_seen"] == [0, 1] and d["value"] == 15.0      # max over ranks of 10, 15
    assert d["calls"] == ["share_sph", "path", "finish", "forces_share", "update0",
                          "share_sph", "path", "finish", "forces_share", "update1"]
    assert d["parallelism"] == bench.parallelism_text(2, "pair_symmetric")
