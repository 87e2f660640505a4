"""N/k-per-GPU decomposition of the step, one process per GPU.

The paper gives each of k GPUs N/k particles and, before the gravity kernel, copies the other GPUs' particles
over GPU-Direct (L139).  Here every rank keeps the whole state (64 B per particle: nothing at 180 GB per GPU) and
computes its SHARE of the O(N^2) gravity stage (`sph_position_share`).  Which gravity kernel runs is decided on the
device, identically on every rank (the replicas hold the same bits), so after the share each rank reads the choice back
(`sph_gravity_path`, one 8-byte read) and issues the ONE collective that path needs:
  * pair-symmetric path (positive masses, delta > 0, N >= 32768 — every BASELINE.json config from config 1 up): the
    rank's work items of the unordered-pair decomposition, accumulated as 64-bit fixed-point integers; one integer SUM
    all-reduce of that region (24 B x N: 25 MiB at N = 2^20).  Integer addition is exact, so every world size gives the
    same bits as one GPU.
  * one-sided path (delta = 0, a zero mass, small N, ...): the rank's TARGET slice against all N sources; one
    all-gather of the acceleration slices (16 B x N/k per rank).
  * G = 0 (config 4): Eq. 4 is identically zero — no collective at all.
`nbody_pp_gravity_finish` then writes the accelerations from the summed integers if that path was taken.  The exchange is
~25 MiB against ~0.26 s / k of gravity at N = 2^20, so there is nothing to gain from fusing it into the kernel.

The SPH passes ("SPH by i-slices over a replicated sorted gas array") are shared the same way when
`share_sph` is on (the default for world > 1): every rank sorts, then runs DC and HFC for every world-th tile of 128
sorted slots (`sph_position_share_sph`, `sph_forces_share`), writing zeros for the other ranks' targets, and the ranks
complete rho (4 B x N_g) and acc_sph (16 B x N_g) by a SUM all-reduce of the 32-bit patterns as integers: x + 0 + ... + 0,
exact, so every world size gives the bits of one GPU.  The O(N) stages (sort, EOS gather, update) run on every rank: they
are deterministic, so the replicas stay bitwise identical and no other exchange is needed.  With `share_sph` off the
SPH passes run redundantly too (0.2 % of the step at the galaxy configs).

This module holds no arithmetic of the method: slice bookkeeping, buffers and the collective.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist

SLICE_ALIGN = 1024          # one gravity target tile (128 threads x 8 targets): slices never split a tile


def slice_bounds(n: int, rank: int, world: int, align: int = SLICE_ALIGN):
    """Rank `rank`'s target slice [i0, i1) of n particles and the common padded slice length `chunk`
    (a multiple of `align`; world * chunk >= n; trailing ranks may get a short or empty slice)."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("bad rank / world / n")
    per = -(-n // world)
    chunk = max(align, -(-per // align) * align)
    i0 = min(rank * chunk, n)
    i1 = min(i0 + chunk, n)
    return i0, i1, chunk


def allreduce_sums(sums: torch.Tensor, world: int, group=None) -> None:
    """Integer SUM all-reduce of the fixed-point sums (int64; NCCL on the GPUs, gloo in the CPU tests)."""
    if world == 1 and not dist.is_initialized():
        return
    assert sums.dtype == torch.int64 and sums.is_contiguous()
    dist.all_reduce(sums, op=dist.ReduceOp.SUM, group=group)


def allreduce_bits(x: torch.Tensor, world: int, group=None) -> None:
    """Completes a float32 array of which every element was written by exactly one rank and is zero on the others:
    SUM all-reduce of the bit patterns as int32 (exact: one non-zero term per element)."""
    if world == 1 and not dist.is_initialized():
        return
    assert x.dtype == torch.float32 and x.is_contiguous()
    dist.all_reduce(x.view(torch.int32), op=dist.ReduceOp.SUM, group=group)


def allgather_rows(full: torch.Tensor, rank: int, world: int, chunk: int, group=None, send: torch.Tensor = None) -> None:
    """`full` has world * chunk rows; rank r has written rows [r * chunk, (r+1) * chunk).  After the call every
    rank holds all rows.  Works for any backend (NCCL on the GPUs, gloo in the CPU tests).  `send`: a persistent
    [chunk, ...] staging buffer (the input of an all-gather must not alias its output); allocated if not given."""
    if world == 1 and not dist.is_initialized():
        return                                   # no process group: plain single-GPU use of the staged calls
    assert full.shape[0] == world * chunk and full.is_contiguous()
    mine = full[rank * chunk:(rank + 1) * chunk]
    if send is None:
        send = torch.empty_like(mine)
    send.copy_(mine)
    dist.all_gather_into_tensor(full, send, group=group)


class ShardedSimulation:
    """The Simulation of binding.py with the gravity stage — and, with share_sph, the SPH passes — split over the ranks
    of `group`."""

    def __init__(self, workload, rank: int, world: int, group=None, sigma=None, binding=None, device="cuda",
                 share_sph=None):
        """binding / device: the C-ABI face and the device of the buffers; the CPU tests of the exchange pass a
        recording stand-in and "cpu" (the product path never does: without the CUDA library binding.load() raises)."""
        if binding is None:
            from . import binding
        b = binding
        self.b, self.w, self.rank, self.world, self.group = b, workload, rank, world, group
        w = workload
        self.n_gas, self.n_halo, self.n = w.n_gas, w.n_halo, w.n_total
        self.i0, self.i1, self.chunk = slice_bounds(self.n, rank, world)
        self.params = b.sph_params.from_workload(w)
        self.posm = torch.from_numpy(np.ascontiguousarray(w.posm)).to(device)
        self.vele = torch.from_numpy(np.ascontiguousarray(w.vele)).to(device)
        self.rho = torch.zeros(max(self.n_gas, 1), dtype=torch.float32, device=device)
        self.acc_sph = torch.zeros(max(self.n_gas, 1), 4, dtype=torch.float32, device=device)
        # world * chunk rows so that the all-gather slots are equal; the library only sees the first n
        self.acc_grav = torch.zeros(world * self.chunk, 4, dtype=torch.float32, device=device)
        self.grid = b.sph_grid_from_bbox(self.posm, self.n_gas, w.h) if self.n_gas > 0 else None
        self.ws = b.alloc_workspace(self.n_gas, self.n, self.grid)
        self.sums = b.gravity_sums_view(self.ws, self.n_gas, self.n, self.grid)   # int64 view, all-reduced each evaluation
        self.sigma = sigma
        self.hsml = None
        if sigma is not None and self.n_gas > 0:
            self.hsml = torch.full((self.n_gas,), float(np.float32(w.h)), dtype=torch.float32, device=device)
        self.share_sph = (world > 1) if share_sph is None else bool(share_sph)
        self.first = True
        self._send = None                        # staging buffer of the all-gather, made on first use
        self.path = None                         # gravity path of the last evaluation (sph_gravity_path)
        self.exchanged_bytes = 0                 # payload this rank handed to collectives so far (bench.py reports it)

    def _position(self, sigma):
        b = self.b
        if self.share_sph and self.n_gas > 0:
            # SP, the rank's targets of DC, the rank's share of GFC; then rho is completed over the ranks
            b.sph_position_share_sph(self.posm, self.hsml, self.n_gas, self.n_halo, self.rank, self.world, self.i0, self.i1,
                                     self.params, self.grid, self.rho, self.acc_grav, self.ws)
            allreduce_bits(self.rho[:self.n_gas], self.world, self.group)
            self.exchanged_bytes += self.n_gas * 4
            if sigma > 0.0 and self.hsml is not None:
                b.sph_renew_hsml(self.posm, self.hsml, sigma, self.n_gas, self.n_halo, self.params, self.grid, self.rho, self.ws)
        else:
            b.sph_position_share(self.posm, self.hsml, sigma, self.n_gas, self.n_halo, self.rank, self.world, self.i0,
                                 self.i1, self.params, self.grid, self.rho, self.acc_grav, self.ws)
        if self.params.G == 0.0 or self.n == 0:
            self.path = "none"                   # Eq. 4 is identically 0: the share zeroed its rows, nothing to exchange
            return
        # the device's choice — the same on every rank, because every rank holds the same bits
        self.path = b.sph_gravity_path(self.ws, self.n_gas, self.n, self.grid)
        if self.path.startswith("pair_symmetric"):
            allreduce_sums(self.sums, self.world, self.group)
            self.exchanged_bytes += self.sums.numel() * 8
        else:
            if self._send is None:
                self._send = torch.empty_like(self.acc_grav[:self.chunk])
            allgather_rows(self.acc_grav, self.rank, self.world, self.chunk, self.group, self._send)
            self.exchanged_bytes += self.chunk * 16
        b.nbody_pp_gravity_finish(self.posm, self.n_gas, self.n_halo, self.grid, self.params.G, self.acc_grav, self.ws)

    def _hydro_update(self, dt, corrector):
        """HFC + SU of one half of the step (Eqs. 10-14 or 10-11, 15-16)."""
        b = self.b
        if self.share_sph and self.n_gas > 0:
            b.sph_forces_share(self.vele, self.hsml, self.n_gas, self.n_halo, self.rank, self.world, self.params, self.grid,
                               self.rho, self.acc_sph, self.ws)
            allreduce_bits(self.acc_sph[:self.n_gas], self.world, self.group)
            self.exchanged_bytes += self.n_gas * 16
            b.sph_update(self.posm, self.vele, self.n_gas, self.n_halo, self.grid, dt, corrector, self.acc_sph, self.acc_grav,
                         self.ws)
        elif corrector:
            b.sph_correct(self.vele, self.hsml, self.n_gas, self.n_halo, self.params, self.grid, dt, self.rho, self.acc_sph,
                          self.acc_grav, self.ws)
        else:
            b.sph_predict(self.posm, self.vele, self.hsml, self.n_gas, self.n_halo, self.params, self.grid, dt, self.rho,
                          self.acc_sph, self.acc_grav, self.ws)

    def step(self, dt=None):
        dt = self.w.dt if dt is None else dt
        if self.first:
            self._position(0.0)                                  # seed: SP, DC, GFC at the current positions
            self.first = False
        self._hydro_update(dt, False)
        self._position(self.sigma or 0.0)                        # SP, DC, GFC slice at r(t+dt) + exchange
        self._hydro_update(dt, True)
