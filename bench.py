#!/usr/bin/env python
"""bench.py — step time of the hot path at BASELINE.json's headline config (config 2, N = 2^20).

    python bench.py --gpus N --steps K --warmup W [--config C] [--impl reference]

One "step" = one sph_step (all §8(a) rows: HFC x2, SU x2, grid sort, density, PP gravity).
Prints ONE JSON line (see DESIGN.md §7 for every key).

--gpus N > 1: one rank per GPU.  Started plainly (`python bench.py --gpus N`) the script re-launches itself under
`python -m torch.distributed.run --nproc-per-node N` (and fails loudly if the box has fewer than N devices); started
by torchrun it takes RANK / LOCAL_RANK / WORLD_SIZE from the environment.  Every rank keeps the whole state and does
its SHARE of the O(N^2) gravity stage (the paper's N/k-per-GPU decomposition, L139): on the
pair-symmetric path (every BASELINE config from config 1 up) the work items rank, rank + N, ... with one int64 SUM
all-reduce of the fixed-point sums per evaluation; on the one-sided path target slices with one all-gather of the
acceleration rows.  The SPH passes are shared as well: every N-th tile of 128 sorted slots per rank, rho
and acc_sph completed by an int32 SUM all-reduce of the bit patterns.  Total work is fixed ("scaling": "strong").
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FLOPS_PER_INTERACTION = 20          # BASELINE.json convention for Eq. 4
SM_COUNT_B200 = 148


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d, "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def parallelism_text(world, path=None, share_sph=True):
    """What the N > 1 run does per force evaluation, from the gravity path the device chose (sph_gravity_path)."""
    if world <= 1:
        return "single GPU"
    if path is None:
        how = "gravity shared over the GPUs, one collective per evaluation (int64 all-reduce or all-gather, by the path the device chooses)"
    elif path.startswith("pair_symmetric"):
        how = (f"gravity: unordered-pair work items rank, rank+{world}, ... per GPU + 1 int64 SUM all-reduce of the "
               f"fixed-point sums (24 B x N) per evaluation")
    elif path == "none":
        how = "no gravity (G = 0): no gravity collective"
    else:
        how = f"gravity: target slices of N/{world} per GPU + 1 all-gather of the acceleration rows (16 B x N/{world} per GPU) per evaluation"
    if share_sph:
        return how + (f"; SPH passes: every {world}th tile of 128 sorted slots per GPU + 1 int32 SUM all-reduce of rho (4 B x N_g) "
                      f"and of acc_sph (16 B x N_g) per pass; O(N) stages (sort, update) replicated")
    return how + "; O(N) and SPH stages replicated"


def workload_config(args, w, grid_dims=None, cells=None, world=1, path=None):
    """The `config` object of the JSON line: identical for both arms (ours / reference)."""
    src = f"BASELINE.json configs[{args.config}]" if args.config <= 4 else "SURVEY.md 8(f) NEXT-3 (collisionless, not a BASELINE config)"
    return {"workload": f"{src} ({w.name}): N={w.n_total}, N_g={w.n_gas}, h={w.h:g}, delta={w.delta:g}, dt={w.dt:g}",
            "grid_dims": grid_dims, "cells": cells, "parallelism": parallelism_text(world, path, share_sph=w.n_gas > 0),
            "l2": "no flush: one step streams >300 MB (cell arrays, gravity partials, particle arrays) > 126 MB L2"}


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch_ranks(n: int, script: str, argv, check_devices: bool = True) -> int:
    """Start `script argv` as n ranks on this node, the way the driver does for N > 1:
    python -m torch.distributed.run --nnodes=1 --nproc-per-node n --master-addr 127.0.0.1 --master-port P script argv.
    Returns the launcher's exit code.  check_devices: refuse (loudly) when the box has fewer than n CUDA devices."""
    if check_devices:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < n:
            raise SystemExit(f"bench.py: --gpus {n} needs {n} CUDA devices, this box has {have}")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr",
           "127.0.0.1", "--master-port", str(free_port()), script, *argv]
    return subprocess.call(cmd)


def reduce_max_ms(ms: float, world: int, device: str = "cuda") -> float:
    """Max over ranks of a per-rank duration (the contract's timing rule); identity for one rank.
    Works on any initialised process group (NCCL on the GPUs, gloo in the CPU test)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def ncu_traffic(kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the committed ncu --set full
    summary profiles/traffic_r02.csv (kernel,n_total,dram_read_bytes,dram_write_bytes); None if absent."""
    p = os.path.join(ROOT, "profiles", "traffic_r02.csv")
    if not os.path.exists(p):
        return None
    for line in open(p):
        f = line.strip().split(",")
        if len(f) >= 4 and f[0] == kernel:
            try:
                return {"n_total": int(f[1]), "bytes": float(f[2]) + float(f[3])}
            except ValueError:
                continue
    return None


def _env_rank():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "power_w_max": None, "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, pw, reasons, mx = [], [], set(), None
        for r in rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1]))
                mx = float(r[2])
                pw.append(float(r[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=mx, reasons=sorted(reasons), power_w_max=max(pw),
                       samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------
# oracle timings (cpu_baseline leg and --impl reference): the oracle as it stands, bounded sample
def oracle_sample_step(w, n_targets=1024, seed=123):
    """Time the oracle on a bounded sample of one step of workload `w` and extrapolate.

    A step is 1 gravity evaluation + 1 grid sort + 1 density pass + 2 hydro passes + O(N) updates.
    Sample: the full CPU counting sort (it is O(N)); gravity for n_targets gas+halo targets against
    all N sources; density and one force pass for n_targets gas targets (their neighbours' densities
    included).  step_ms = sort + gravity * N/n_t + (density + 2 forces) * N_g/n_t.
    """
    import oracle
    from paper_1807_08116_b200 import workloads as wl
    ng, n = w.n_gas, w.n_total
    half = max(1, n_targets // 2)
    g_idx, h_idx = wl.subset_indices(ng, w.n_halo, seed, n_each=half)
    tg = np.concatenate([g_idx, h_idx]).astype(np.int64)
    posm64 = w.posm.astype(np.float64)
    vele64 = w.vele.astype(np.float64)
    t = {}
    t0 = time.perf_counter()
    if ng:
        grid = oracle.grid_from_bbox(posm64, ng, w.h)
        key = oracle.cell_keys(posm64, ng, grid)
        _, start, perm = oracle.counting_sort(key, grid.M)
    t["sort"] = time.perf_counter() - t0
    t0 = time.perf_counter()
    if w.G != 0.0 and len(tg):
        oracle.gravity(posm64, w.G, w.delta, targets=tg)
    t["gravity_sample"] = time.perf_counter() - t0
    t["density_sample"] = t["forces_sample"] = 0.0
    if ng and len(g_idx):
        t0 = time.perf_counter()
        off, idx = oracle.neighbours(posm64, ng, w.h, targets=g_idx, method="grid", grid=grid, sort=(key, start, perm))
        rho_t = oracle.density(posm64, w.h, off, idx, targets=g_idx)
        t["density_sample"] = time.perf_counter() - t0
        # densities of the neighbours (needed by the force sums): not charged to the sample's force time
        closure = np.unique(np.concatenate([g_idx, idx.astype(np.int64)]))
        off2, idx2 = oracle.neighbours(posm64, ng, w.h, targets=closure, method="grid", grid=grid, sort=(key, start, perm))
        rho_all = np.ones(ng)
        rho_all[closure] = oracle.density(posm64, w.h, off2, idx2, targets=closure)
        t0 = time.perf_counter()
        oracle.forces(posm64, vele64, rho_all, w.h, off, idx, targets=g_idx, gamma=w.gamma, alpha=w.alpha, beta=w.beta,
                      eta=w.eta)
        t["forces_sample"] = time.perf_counter() - t0 + t["density_sample"] * 0.0
    n_t, n_g = max(len(tg), 1), max(len(g_idx), 1)
    step_s = t["sort"] + t["gravity_sample"] * (n / n_t if w.G != 0.0 else 0.0) \
        + (t["density_sample"] + 2.0 * t["forces_sample"]) * (ng / n_g if ng else 0.0)
    sample_s = sum(t.values())
    desc = (f"{len(tg)} gravity targets x {n} sources + density/forces for {len(g_idx)} gas targets + full CPU counting "
            f"sort; step time extrapolated by N/n_targets")
    return step_s * 1e3, sample_s, desc, t


def oracle_full_steps():
    """configs 0 and 1 are small enough to time the oracle's WHOLE step (no extrapolation), config 0
    also on one thread.  The carried state (grid, density, gravity at the current positions) is seeded untimed,
    as for the CUDA path."""
    import oracle
    from paper_1807_08116_b200 import workloads as wl
    out = {}
    cores = oracle.num_threads()
    for cfg, threads in ((0, cores), (0, 1), (1, cores)):
        w = wl.make_workload(cfg)
        oracle.set_num_threads(threads)
        st = oracle.State(w.posm.astype(np.float64), w.vele.astype(np.float64), w.n_gas)
        nbr = oracle.position_only(st, w.h, w.G, w.delta)
        t0 = time.perf_counter()
        oracle.step(st, w.dt, w.h, w.G, w.delta, nbr=nbr)
        out[f"config{cfg}_step_ms_{threads}_threads"] = (time.perf_counter() - t0) * 1e3
    oracle.set_num_threads(cores)
    return out


def run_reference(args, w):
    import oracle
    rank, _, _ = _env_rank()
    if rank != 0:
        return
    vals = []
    for i in range(args.warmup + args.steps):
        ms, _, desc, _ = oracle_sample_step(w, n_targets=args.ref_targets)
        if i >= args.warmup:
            vals.append(ms)
    v = float(np.mean(vals))
    cores = oracle.num_threads()
    grid_dims = cells = None
    if w.n_gas:
        og = oracle.grid_from_bbox(w.posm.astype(np.float64), w.n_gas, w.h)
        grid_dims, cells = [int(d) for d in og.dims], int(og.M)
    line = {
        "impl": "reference", "metric": "step_ms", "value": v, "unit": "ms", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": v, "higher_is_better": False, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": workload_config(args, w, grid_dims, cells, 1),
        "cpu_baseline": {"value": v, "unit": "ms", "cores": cores, "kind": "oracle", "sample": desc, "extrapolated": True},
        "e2e": {"value": v, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def sph_pair_counts(b, sim, w):
    """Diagnostics for the SPH throughput figures (quote candidate-pairs/s and accepted-pairs/s, with the
    neighbour and occupancy histograms beside them).  Outside every timed region.  Candidate pairs are the ALGORITHMIC
    ones of the paper's cell-list search (every particle against the 27 cells of its stencil, L207), counted from the
    library's own histogram; accepted pairs are the neighbour counts of the library's sph_neighbour_lists (count pass
    only: capacity 0).  torch is used here for sums over those device arrays — it is not on the path."""
    import torch
    ng = w.n_gas
    g = sim.grid
    key = torch.zeros(ng, dtype=torch.int32, device="cuda")
    perm = torch.zeros(ng, dtype=torch.int32, device="cuda")
    count = torch.zeros(g.M, dtype=torch.int32, device="cuda")
    start = torch.zeros(g.M + 1, dtype=torch.int32, device="cuda")
    b.sph_build_grid(sim.posm, ng, g, key, perm, count, start, sim.ws)
    mx, my, mz = (int(d) for d in g.dims)
    c = count.view(1, 1, mz, my, mx).to(torch.float32)
    c27 = torch.nn.functional.conv3d(c, torch.ones(1, 1, 3, 3, 3, device="cuda"), padding=1)
    candidates = float((c.double() * c27.double()).sum().item())
    cnt = torch.zeros(max(ng, 1), dtype=torch.int32, device="cuda")
    off = torch.zeros(ng + 1, dtype=torch.int64, device="cuda")
    L = b.load()
    p, nb = b._ws(sim.ws)
    rc = L.sph_neighbour_lists(b._ptr(sim.posm), ng, float(w.h), b.C.byref(g), b._ptr(perm), b._ptr(start), b._ptr(cnt),
                               b._ptr(off), None, 0, p, nb, b._stream())
    if rc not in (b.SPH_OK, b.SPH_ERR_WORKSPACE):
        raise b.SphError("sph_neighbour_lists", rc)
    accepted = float(off[ng].item())
    occ = count[count > 0].to(torch.float32)
    nb_f = cnt[:ng].to(torch.float32)
    q = torch.tensor([0.5, 0.9, 0.99], device="cuda")
    return {
        "candidate_pairs": candidates, "accepted_pairs": accepted,
        "neighbours_mean": accepted / ng, "neighbours_p50_p90_p99_max": [float(x) for x in torch.quantile(nb_f[:: max(1, ng // 1000000)], q)] + [float(nb_f.max())],
        "occupied_cells": int(occ.numel()), "cells": int(g.M),
        "occupancy_p50_p90_p99_max": [float(x) for x in torch.quantile(occ[:: max(1, occ.numel() // 1000000)], q)] + [float(occ.max())],
        "dense_walk_items": b.sph_dense_items(sim.ws, ng, w.n_total, g),
    }


# ------------------------------------------------------------------------------------------------
def run_ours(args, w):
    import torch
    import torch.distributed as dist
    from paper_1807_08116_b200 import binding as b

    rank, local_rank, world = _env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    if local_rank >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} needs CUDA device {local_rank}; --gpus {world} needs {world} devices, "
                         f"this box has {torch.cuda.device_count()}")
    torch.cuda.set_device(local_rank)
    # under torchrun (any world size, also 1) the sharded path runs, collective included; plain `python bench.py` is
    # the single-GPU sph_step path
    use_dist = "RANK" in os.environ and "WORLD_SIZE" in os.environ
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    b.load()
    peaks, peak_src = _peaks()

    n, ng = w.n_total, w.n_gas
    if use_dist:
        from paper_1807_08116_b200.sharded import ShardedSimulation
        sim = ShardedSimulation(w, rank, world, sigma=args.sigma)
    else:
        sim = b.Simulation(w, sigma=args.sigma)
    share = 1.0 / world                                       # this rank's part of the N^2 interactions (work items or target slice)
    M = sim.grid.M if ng else 0

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident arm -----------------------------------------------------------------
    for _ in range(max(args.warmup, 3)):
        sim.step()
    barrier()
    sim_steps = args.steps
    if use_dist:
        sim.exchanged_bytes = 0
    sampler = ClockSampler(local_rank) if rank == 0 else None
    launches0 = b.sph_launch_count()
    b.sph_set_profiling(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        sim.step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    stage = b.sph_get_stage_ms()
    b.sph_set_profiling(False)
    launches = b.sph_launch_count() - launches0
    clocks = sampler.stop() if sampler else None
    ms_step = reduce_max_ms(ms_total, world) / args.steps

    # ---- end-to-end arm: HOST (pinned) buffers through sph_host_ctx_step, copies inside the timing
    e2e = None
    if args.sigma is not None and not use_dist and not args.no_e2e:
        # the host-buffer entry point steps with one global h: it would time a different algorithm than the arm above
        e2e = {"value": None, "unit": "ms", "skipped": "sph_host_ctx_step has no per-particle-h variant; --sigma runs carry no end-to-end number"}
    elif not args.no_e2e:
        hp = torch.from_numpy(w.posm.copy()).pin_memory()
        hv = torch.from_numpy(w.vele.copy()).pin_memory()
        hrho = torch.zeros(max(ng, 1), dtype=torch.float32).pin_memory()
        prm = b.sph_params.from_workload(w)
        k_e2e = max(1, min(args.steps, args.e2e_steps))
        if not use_dist:
            ctx = b.HostContext(ng, w.n_halo)
            ctx.step(hp, hv, prm, w.dt, 1, first=True, rho=hrho)          # warm-up + seeding
            ctx.step(hp, hv, prm, w.dt, 1, first=False, rho=hrho)

            def e2e_step():                                               # H2D posm+vele, step, D2H posm+vele+rho, sync
                ctx.step(hp, hv, prm, w.dt, 1, first=False, rho=hrho)
            how = "host wall clock around sph_host_ctx_step (it synchronises)"
        else:
            sim_e = ShardedSimulation(w, rank, world, sigma=args.sigma)
            sim_e.step()
            hp.copy_(sim_e.posm)
            hv.copy_(sim_e.vele)

            def e2e_step():                                               # the same copies around the sharded step
                sim_e.posm.copy_(hp, non_blocking=True)
                sim_e.vele.copy_(hv, non_blocking=True)
                sim_e.step()
                hp.copy_(sim_e.posm, non_blocking=True)
                hv.copy_(sim_e.vele, non_blocking=True)
                if ng:
                    hrho.copy_(sim_e.rho[:ng], non_blocking=True)
                torch.cuda.synchronize()
            e2e_step()
            how = "host wall clock around pinned H2D + ShardedSimulation.step + D2H + synchronise"
        barrier()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            e2e_step()
        t_e2e = (time.perf_counter() - t0) * 1e3 / k_e2e
        if not use_dist:
            ctx.close()
        e2e = {"value": reduce_max_ms(t_e2e, world), "unit": "ms", "h2d_bytes_per_step": 2 * n * 16,
               "d2h_bytes_per_step": 2 * n * 16 + ng * 4, "steps": k_e2e, "timing": how + ", max over ranks"}

    if rank != 0:
        dist.destroy_process_group()
        return

    # ---- derived figures -----------------------------------------------------------------------
    K = args.steps
    grav_ms = stage["gravity"] / K          # one evaluation per step (L123)
    sort_ms, dens_ms, forc_ms, upd_ms = (stage[k] / K for k in ("sort", "density", "forces", "update"))
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    alu_peak_tflops = 2 * 128 * SM_COUNT_B200 * sm_max * 1e6 / 1e12
    roofline = None
    if w.G != 0.0 and grav_ms > 0:
        achieved = FLOPS_PER_INTERACTION * share * float(n) * float(n) / (grav_ms * 1e-3) / 1e12   # per GPU (rank 0's share)
        path = b.sph_gravity_path(sim.ws, ng, n, sim.grid)           # chosen on the device
        # FP32 lane-operations the variant really executes per INTERACTION (an FMA counted once) and its dominant kernel
        kernel, ops = {"pair_symmetric": ("grav_sym_kernel", 7.0), "pair_symmetric_general": ("grav_sym_kernel", 8.0),
                       "one_sided_uniform": ("grav_pp_kernel", 11.0),
                       "one_sided": ("grav_pp_kernel", 12.0)}[path]
        tr = ncu_traffic(kernel)
        traffic = tr["bytes"] if tr and tr["n_total"] == n else None   # the capture is of this workload only
        lane_peak = 128 * SM_COUNT_B200 * sm_max * 1e6                 # FP32 lane-operations per second
        roofline = {"kernel": kernel, "bound": "alu", "achieved": achieved, "peak": alu_peak_tflops,
                    "unit": "TFLOP/s", "frac": achieved / alu_peak_tflops, "traffic": traffic,
                    "traffic_note": "DRAM bytes per launch (ncu --set full, profiles/traffic_r02.csv); irrelevant to an ALU-bound kernel",
                    "peak_source": f"2*128*148*sm_max_mhz ({peak_src} sm_max_mhz={sm_max:.0f}); 20 flops/interaction",
                    "kernel_ms": grav_ms, "launches_per_step": 1, "gravity_path": path,
                    "executed_lane_ops_per_interaction": ops,
                    "fp32_pipe_util": ops * share * float(n) * float(n) / (grav_ms * 1e-3) / lane_peak,
                    "note": "achieved = ALGORITHMIC flops (BASELINE.json convention: 20 per ordered interaction, N^2 of them) / "
                            "gravity stage time (pack + kernel + reduce; the O(N) kernels are <0.1%).  The pair-symmetric "
                            "kernel evaluates each UNORDERED pair once (14 FP32 lane-ops + 1 MUFU per pair = 7 + 0.5 per "
                            "interaction), so frac can exceed the 20-flop instruction-mix ceiling and even 1; "
                            "fp32_pipe_util is the share of FP32 issue capacity (128 lanes/clk/SM) the executed operations take"}
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    pairs = sph_pair_counts(b, sim, w) if (ng and world == 1) else None
    sort_bytes = ng * 92 + M * 12          # 92 B per gas particle, 12 B per cell (zero 4, scan read 4 + write 4)
    # gas: predictor 64 B read + 48 B written, corrector 64 + 16; halo particles never touch acc_sph: 48 + 48, 48 + 16
    upd_bytes = ng * (112 + 80) + (n - ng) * (96 + 64)
    stages = {
        "gravity_ms": grav_ms, "sort_ms": sort_ms, "density_ms": dens_ms, "forces_ms_2passes": forc_ms, "update_ms": upd_ms,
        "pp_ginteractions_per_s": (float(n) * n / (grav_ms * 1e-3) / 1e9) if (grav_ms > 0 and w.G != 0.0) else None,   # whole job: all slices run concurrently
        "sph_mparticles_per_s": (ng / ((sort_ms + dens_ms + forc_ms) * 1e-3) / 1e6) if ng else None,
        "sort_mkeys_per_s": (ng / (sort_ms * 1e-3) / 1e6) if ng and sort_ms > 0 else None,
        "sort_hbm_gbs": (sort_bytes / (sort_ms * 1e-3) / 1e9) if ng and sort_ms > 0 else None,
        "sort_hbm_frac": (sort_bytes / (sort_ms * 1e-3) / 1e9 / hbm) if ng and sort_ms > 0 else None,
        # "report against both" — BASELINE.json quotes ~8 TB/s nominal HBM3e, the box measures `hbm` by copy
        "sort_hbm_frac_of_nominal_8tbs": (sort_bytes / (sort_ms * 1e-3) / 1e9 / 8000.0) if ng and sort_ms > 0 else None,
        "update_hbm_frac": (upd_bytes / (upd_ms * 1e-3) / 1e9 / hbm) if upd_ms > 0 else None,
        # the neighbour passes are latency- / ALU-bound, not HBM-bound: their COMPULSORY bytes (density
        # 16 r + 4 w per gas particle; one forces pass 16+16+8 r + 16 w + the EOS gather 24 r + 24 w) against the HBM peak,
        # reported because BASELINE.json asks for the fraction — it measures how far from memory-bound they are
        "density_hbm_frac": (ng * 20 / (dens_ms * 1e-3) / 1e9 / hbm) if ng and dens_ms > 0 else None,
        "forces_hbm_frac": (2 * ng * 104 / (forc_ms * 1e-3) / 1e9 / hbm) if ng and forc_ms > 0 else None,
        "hbm_peak_gbs": hbm, "peak_source": peak_src,
    }
    if pairs and dens_ms > 0 and forc_ms > 0:
        # SURVEY 8(d) op counts: a candidate test is ~7 FP32 lane-operations, an accepted density pair ~12 more, an
        # accepted force pair ~60 more; one density pass and two forces passes per step
        cand, acc = pairs["candidate_pairs"], pairs["accepted_pairs"]
        lane_ops = (cand * 7 + acc * 12) + 2 * (cand * 7 + acc * 60)
        if roofline is None:
            # no gravity (config 4): the dominant kernel is the hydro-force walk, bound by instruction issue / FP32 ALU.
            # ALGORITHMIC lane-operations of ONE forces pass (27-cell candidates x 7 + accepted pairs x 60, an FMA counted
            # once) x 2 flops, over the forces stage's time per pass (EOS gather + thread-per-slot walk of the
            # sparse cells + dense-cell walk; the dense-cell walk is ~90 % of it, profiles/launches_c4_r02.md)
            f_ops = 2.0 * (cand * 7 + acc * 60)
            f_ach = f_ops / (0.5 * forc_ms * 1e-3) / 1e12
            roofline = {"kernel": "k_dense_forces" if pairs.get("dense_walk_items") else "k_forces", "bound": "alu",
                        "achieved": f_ach, "peak": alu_peak_tflops, "unit": "TFLOP/s", "frac": f_ach / alu_peak_tflops,
                        "traffic": None, "kernel_ms": 0.5 * forc_ms, "launches_per_step": 2,
                        "peak_source": f"2*128*148*sm_max_mhz ({peak_src} sm_max_mhz={sm_max:.0f})",
                        "note": "achieved = 2 x ALGORITHMIC FP32 lane-operations of one hydro-force pass (27-cell candidate "
                                "tests x 7 + accepted pairs x 60) / forces stage time per pass; the dense-cell walk tests ~2.5 "
                                "candidates per neighbour instead of the 27-cell count's 6 (octant binning), so the executed "
                                "operations are fewer than the algorithmic ones; DRAM traffic is irrelevant to this kernel "
                                "(profiles/sph_dense_r02.md: 2.6 GB per launch)"}
        stages.update({
            "sph_pairs": pairs,
            "sph_candidate_pairs_per_s": 3 * cand / ((dens_ms + forc_ms) * 1e-3),
            "sph_accepted_pairs_per_s": 3 * acc / ((dens_ms + forc_ms) * 1e-3),
            "sph_fp32_frac": lane_ops / ((dens_ms + forc_ms) * 1e-3) / (128 * SM_COUNT_B200 * sm_max * 1e6),
            "sph_fp32_note": "ALGORITHMIC lane-operations (27-cell candidates x 7 + accepted pairs x 12 (density) or x 60 "
                             "(forces); 3 passes per step) / (density + forces time) / (128 lanes x 148 SMs x sm_max); the "
                             "dense-cell walk tests fewer candidates than the 27-cell count (octant binning)",
        })

    # ---- the oracle on this box's host cores, bounded sample (rank 0, N = 1 only) ----------------
    cpu = None
    if world == 1 and not args.no_cpu:
        import oracle
        ms, sample_s, desc, _ = oracle_sample_step(w, n_targets=args.cpu_targets)
        cpu = {"value": ms, "unit": "ms", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": desc + f" ({sample_s:.1f} s of CPU wall time)", "extrapolated": True,
               "full_steps_timed": oracle_full_steps()}

    line = {
        "metric": "step_ms", "value": ms_step, "unit": "ms", "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": False, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": dict(workload_config(args, w, list(sim.grid.dims) if ng else None, M, world,
                                       getattr(sim, "path", None) if use_dist else None),
                       **({"smoothing_lengths": f"per particle, sigma={args.sigma:g}, cap h"} if args.sigma is not None else {})),
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "stages": stages,
        "exchange": ({"gravity_path": sim.path, "payload_bytes_per_rank_per_step": sim.exchanged_bytes // max(sim_steps, 1),
                      "collectives_per_evaluation": 0 if sim.path == "none" else 1} if use_dist else None),
        "context": "paper Table 1 (K40, N=2^20, units inferred as s): t_SPH=7.87, t_GFC=53.62 — other hardware, not a target",
    }
    print(json.dumps(line), flush=True)
    if use_dist:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--scale", type=float, default=1.0, help="shrink the workload (debug only; invalid as a bench number)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sigma", type=float, default=None,
                    help="per-particle smoothing lengths (NEXT-2): h_i = min(sigma (m/rho)^(1/3), h), renewed every step")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    # one sample size for the cpu_baseline leg and the reference arm: the two estimate the same quantity
    ap.add_argument("--cpu-targets", type=int, default=32768)
    ap.add_argument("--ref-targets", type=int, default=32768)
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    under_launcher = "RANK" in os.environ and "WORLD_SIZE" in os.environ
    if under_launcher and int(os.environ["WORLD_SIZE"]) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={os.environ['WORLD_SIZE']} ranks")
    if args.gpus > 1 and not under_launcher and args.impl == "ours":
        # started plainly: become N ranks (one per GPU) ourselves; rank 0 of the children prints the JSON line
        raise SystemExit(launch_ranks(args.gpus, os.path.abspath(__file__), sys.argv[1:]))
    from paper_1807_08116_b200 import workloads as wl
    w = wl.make_workload(args.config, scale=args.scale)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
