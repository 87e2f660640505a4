"""Thin ctypes face of libsph_b200.so — same names as include/sph_b200.h, argument
marshalling only.  Device arrays are torch CUDA tensors (PyTorch is used for device memory
and streams, nothing else); every step of the path runs inside the library's kernels.

There is no CPU fallback: if the library is missing it is built with nvcc (csrc/build.py),
and if that fails, or there is no CUDA device when a call is made, the call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

SPH_OK, SPH_ERR_ARG, SPH_ERR_GRID, SPH_ERR_WORKSPACE, SPH_ERR_CUDA, SPH_ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5
_ERR = {-1: "SPH_ERR_ARG", -2: "SPH_ERR_GRID", -3: "SPH_ERR_WORKSPACE", -4: "SPH_ERR_CUDA", -5: "SPH_ERR_UNSUPPORTED"}
STAGES = ("sort", "density", "forces", "gravity", "update")

EXPORTS = (
    "sph_last_cuda_error", "sph_grid_from_bbox", "sph_workspace_bytes", "sph_build_grid", "sph_neighbour_ranges",
    "sph_density", "sph_forces", "nbody_pp_gravity", "sph_step", "sph_evaluate", "sph_step_host",
    "sph_host_ctx_create", "sph_host_ctx_step", "sph_host_ctx_destroy", "sph_neighbour_lists",
    "sph_set_profiling", "sph_get_stage_ms", "sph_launch_count", "sph_cfl_dt",
    "nbody_pp_gravity_slice", "sph_position_slice", "sph_predict", "sph_correct",
    "sph_gravity_path", "sph_dense_items", "sph_workspace_status", "sph_position_share", "nbody_pp_gravity_share", "nbody_pp_gravity_finish",
    "sph_workspace_gravity_sums", "sph_smoothing_lengths", "sph_density_h", "sph_forces_h", "sph_evaluate_h", "sph_step_h", "sph_neighbour_lists_h", "sph_step_cfl",
    "sph_position_share_sph", "sph_renew_hsml", "sph_forces_share", "sph_update",
    "nbody_pp_gravity_static", "nbody_pp_gravity_static_max",
)


class SphError(RuntimeError):
    def __init__(self, fn, rc):
        self.rc = rc
        cu = _lib.sph_last_cuda_error() if (_lib is not None and rc == SPH_ERR_CUDA) else 0
        super().__init__(f"{fn} failed: {_ERR.get(rc, rc)}" + (f" (cudaError {cu})" if cu else ""))


class sph_grid(C.Structure):
    _fields_ = [("origin", C.c_float * 3), ("cell", C.c_float), ("inv_cell", C.c_float), ("dims", C.c_int32 * 3)]

    @property
    def M(self):
        return int(self.dims[0]) * int(self.dims[1]) * int(self.dims[2])

    @classmethod
    def make(cls, origin, cell, inv_cell, dims):
        g = cls()
        for a in range(3):
            g.origin[a] = origin[a]
            g.dims[a] = dims[a]
        g.cell, g.inv_cell = cell, inv_cell
        return g


class sph_params(C.Structure):
    _fields_ = [(k, C.c_float) for k in ("h", "gamma", "alpha", "beta", "eta", "G", "delta")]

    @classmethod
    def make(cls, h, G=1.0, delta=0.01, gamma=5.0 / 3.0, alpha=0.5, beta=1.0, eta=0.1):
        return cls(h, gamma, alpha, beta, eta, G, delta)

    @classmethod
    def from_workload(cls, w):
        return cls(w.h, w.gamma, w.alpha, w.beta, w.eta, w.G, w.delta)


def lib_path() -> str:
    return os.path.join(_HERE, "libsph_b200.so")


def load():
    """Load (building first if needed) the C-ABI library.  Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    from .csrc.build import build
    path = build()
    L = C.CDLL(path)
    vp, i64, f32, sz = C.c_void_p, C.c_int64, C.c_float, C.c_size_t
    gp, pp = C.POINTER(sph_grid), C.POINTER(sph_params)
    L.sph_last_cuda_error.restype = C.c_int
    L.sph_launch_count.restype = i64
    L.sph_set_profiling.argtypes = [C.c_int]
    L.sph_get_stage_ms.argtypes = [C.POINTER(C.c_float)]
    L.sph_grid_from_bbox.argtypes = [vp, i64, f32, gp, vp, sz, vp]
    L.sph_workspace_bytes.argtypes = [i64, i64, gp]
    L.sph_workspace_bytes.restype = sz
    L.sph_build_grid.argtypes = [vp, i64, gp, vp, vp, vp, vp, vp, sz, vp]
    L.sph_neighbour_ranges.argtypes = [gp, vp, vp, i64, vp, vp, vp]
    L.sph_density.argtypes = [vp, i64, pp, gp, vp, vp, vp, vp, sz, vp]
    L.sph_forces.argtypes = [vp, vp, vp, i64, pp, gp, vp, vp, vp, vp, sz, vp]
    L.nbody_pp_gravity.argtypes = [vp, i64, f32, f32, vp, vp, sz, vp]
    L.sph_position_share.argtypes = [vp, vp, f32, i64, i64, C.c_int, C.c_int, i64, i64, pp, gp, vp, vp, vp, sz, vp]
    L.nbody_pp_gravity_share.argtypes = [vp, i64, C.c_int, C.c_int, i64, i64, f32, f32, vp, vp, sz, vp]
    L.nbody_pp_gravity_finish.argtypes = [vp, i64, i64, gp, f32, vp, vp, sz, vp]
    L.sph_position_share_sph.argtypes = [vp, vp, i64, i64, C.c_int, C.c_int, i64, i64, pp, gp, vp, vp, vp, sz, vp]
    L.sph_renew_hsml.argtypes = [vp, vp, f32, i64, i64, pp, gp, vp, vp, sz, vp]
    L.sph_forces_share.argtypes = [vp, vp, i64, i64, C.c_int, C.c_int, pp, gp, vp, vp, vp, sz, vp]
    L.sph_update.argtypes = [vp, vp, i64, i64, gp, f32, C.c_int, vp, vp, vp, sz, vp]
    L.nbody_pp_gravity_static.argtypes = [vp, i64, f32, f32, vp, vp]
    L.nbody_pp_gravity_static_max.restype = i64
    L.sph_workspace_gravity_sums.argtypes = [i64, i64, gp, C.POINTER(sz), C.POINTER(sz)]
    L.sph_gravity_path.argtypes = [vp, sz, i64, i64, gp, C.POINTER(C.c_int), vp]
    L.sph_dense_items.argtypes = [vp, sz, i64, i64, gp, C.POINTER(C.c_uint32), vp]
    L.sph_workspace_status.argtypes = [vp, sz, i64, i64, gp, C.POINTER(C.c_uint32), vp]
    L.sph_cfl_dt.argtypes = [vp, vp, vp, vp, vp, i64, pp, gp, vp, vp, f32, vp, vp, vp, sz, vp]
    L.sph_step.argtypes = [vp, vp, i64, i64, pp, gp, f32, C.c_int, vp, vp, vp, vp, sz, vp]
    L.sph_evaluate.argtypes = [vp, vp, i64, i64, pp, gp, vp, vp, vp, vp, sz, vp]
    L.sph_step_host.argtypes = [vp, vp, i64, i64, pp, f32, C.c_int, vp, vp, vp]
    L.sph_host_ctx_create.argtypes = [i64, i64, C.POINTER(vp)]
    L.sph_host_ctx_step.argtypes = [vp, vp, vp, pp, f32, C.c_int, C.c_int, vp, vp, vp]
    L.sph_host_ctx_destroy.argtypes = [vp]
    L.sph_neighbour_lists.argtypes = [vp, i64, f32, gp, vp, vp, vp, vp, vp, C.c_uint64, vp, sz, vp]
    L.sph_neighbour_lists_h.argtypes = [vp, vp, i64, f32, gp, vp, vp, vp, vp, vp, C.c_uint64, vp, sz, vp]
    L.sph_smoothing_lengths.argtypes = [vp, vp, i64, f32, f32, vp, vp]
    L.nbody_pp_gravity_slice.argtypes = [vp, i64, i64, i64, f32, f32, vp, vp, sz, vp]
    L.sph_position_slice.argtypes = [vp, vp, f32, i64, i64, i64, i64, pp, gp, vp, vp, vp, sz, vp]
    L.sph_predict.argtypes = [vp, vp, vp, i64, i64, pp, gp, f32, vp, vp, vp, vp, sz, vp]
    L.sph_correct.argtypes = [vp, vp, i64, i64, pp, gp, f32, vp, vp, vp, vp, sz, vp]
    L.sph_density_h.argtypes = [vp, vp, i64, pp, gp, vp, vp, vp, vp, sz, vp]
    L.sph_forces_h.argtypes = [vp, vp, vp, vp, i64, pp, gp, vp, vp, vp, vp, sz, vp]
    L.sph_evaluate_h.argtypes = [vp, vp, vp, i64, i64, pp, gp, vp, vp, vp, vp, sz, vp]
    L.sph_step_h.argtypes = [vp, vp, vp, i64, i64, pp, gp, f32, f32, C.c_int, vp, vp, vp, vp, sz, vp]
    L.sph_step_cfl.argtypes = [vp, vp, vp, i64, i64, pp, gp, f32, f32, f32, C.c_int, vp, vp, vp, vp, vp, sz, vp]
    _lib = L
    return L


def _chk(fn, rc):
    if rc != SPH_OK:
        raise SphError(fn, rc)


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        assert t.is_cuda and t.is_contiguous(), "device arguments must be contiguous CUDA tensors"
        return t.data_ptr()
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    raise TypeError(type(t))


def _stream():
    return torch.cuda.current_stream().cuda_stream


def _ws(ws):
    return _ptr(ws), ws.numel() * ws.element_size()


def alloc_workspace(n_gas, n_total, grid=None) -> torch.Tensor:
    nbytes = sph_workspace_bytes(n_gas, n_total, grid)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ws[:256].zero_()          # the status word (sph_workspace_status) starts clear
    return ws


# ------------------------------------------------------------------ the boundary, one function per entry point
def sph_workspace_bytes(n_gas, n_total, grid=None) -> int:
    n = load().sph_workspace_bytes(int(n_gas), int(n_total), C.byref(grid) if grid is not None else None)
    if n == 0:
        raise SphError("sph_workspace_bytes", SPH_ERR_ARG)
    return int(n)


def sph_grid_from_bbox(posm, n_gas, h, ws=None) -> sph_grid:
    if ws is None:
        ws = torch.empty(4096, dtype=torch.uint8, device="cuda")
    g = sph_grid()
    p, nb = _ws(ws)
    _chk("sph_grid_from_bbox", load().sph_grid_from_bbox(_ptr(posm), int(n_gas), float(h), C.byref(g), p, nb, _stream()))
    return g


def sph_build_grid(posm, n_gas, grid, key, perm, cell_count, cell_start, ws):
    p, nb = _ws(ws)
    _chk("sph_build_grid", load().sph_build_grid(_ptr(posm), int(n_gas), C.byref(grid), _ptr(key), _ptr(perm),
                                                 _ptr(cell_count), _ptr(cell_start), p, nb, _stream()))


def sph_neighbour_ranges(grid, key, cell_start, n_gas, cell_range=None, particle_runs=None):
    _chk("sph_neighbour_ranges", load().sph_neighbour_ranges(C.byref(grid), _ptr(key), _ptr(cell_start), int(n_gas),
                                                             _ptr(cell_range), _ptr(particle_runs), _stream()))


def sph_density(posm, n_gas, params, grid, perm, cell_start, rho, ws):
    p, nb = _ws(ws)
    _chk("sph_density", load().sph_density(_ptr(posm), int(n_gas), C.byref(params), C.byref(grid), _ptr(perm),
                                           _ptr(cell_start), _ptr(rho), p, nb, _stream()))


def sph_forces(posm, vele, rho, n_gas, params, grid, perm, cell_start, acc_sph, ws):
    p, nb = _ws(ws)
    _chk("sph_forces", load().sph_forces(_ptr(posm), _ptr(vele), _ptr(rho), int(n_gas), C.byref(params), C.byref(grid),
                                         _ptr(perm), _ptr(cell_start), _ptr(acc_sph), p, nb, _stream()))


def nbody_pp_gravity(posm, n_total, G, delta, acc_grav, ws):
    p, nb = _ws(ws)
    _chk("nbody_pp_gravity", load().nbody_pp_gravity(_ptr(posm), int(n_total), float(G), float(delta), _ptr(acc_grav),
                                                     p, nb, _stream()))


def sph_cfl_dt(posm, vele, rho, acc_sph, acc_grav, n_gas, params, grid, perm, cell_start, c_cfl, dt_out, dt_particle, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_cfl_dt", load().sph_cfl_dt(_ptr(posm), _ptr(vele), _ptr(rho), _ptr(acc_sph), _ptr(acc_grav), int(n_gas),
                                         C.byref(params), g, _ptr(perm), _ptr(cell_start), float(c_cfl), _ptr(dt_out),
                                         _ptr(dt_particle), p, nb, _stream()))


def sph_step(posm, vele, n_gas, n_halo, params, grid, dt, first, rho, acc_sph, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_step", load().sph_step(_ptr(posm), _ptr(vele), int(n_gas), int(n_halo), C.byref(params), g, float(dt),
                                     int(bool(first)), _ptr(rho), _ptr(acc_sph), _ptr(acc_grav), p, nb, _stream()))


def sph_evaluate(posm, vele, n_gas, n_halo, params, grid, rho, acc_sph, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_evaluate", load().sph_evaluate(_ptr(posm), _ptr(vele), int(n_gas), int(n_halo), C.byref(params), g,
                                             _ptr(rho), _ptr(acc_sph), _ptr(acc_grav), p, nb, _stream()))


def nbody_pp_gravity_static(posm, n_total, G, delta, acc_grav):
    """Eq. 4 with the library's own fixed scratch: no workspace, no allocation; n_total <= nbody_pp_gravity_static_max().
    Calls on one device share that scratch and must not overlap on the GPU (include/sph_b200.h)."""
    _chk("nbody_pp_gravity_static", load().nbody_pp_gravity_static(_ptr(posm), int(n_total), float(G), float(delta),
                                                                   _ptr(acc_grav), _stream()))


def nbody_pp_gravity_static_max() -> int:
    return int(load().nbody_pp_gravity_static_max())


# ------------------------------------------------------------------ NEXT-4: stages of a step, target slices
def nbody_pp_gravity_slice(posm, n_total, i0, i1, G, delta, acc_grav, ws):
    p, nb = _ws(ws)
    _chk("nbody_pp_gravity_slice", load().nbody_pp_gravity_slice(_ptr(posm), int(n_total), int(i0), int(i1), float(G),
                                                                 float(delta), _ptr(acc_grav), p, nb, _stream()))


def sph_position_share(posm, hsml, sigma, n_gas, n_halo, rank, world, i0, i1, params, grid, rho, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_position_share", load().sph_position_share(_ptr(posm), _ptr(hsml), float(sigma), int(n_gas), int(n_halo),
                                                         int(rank), int(world), int(i0), int(i1), C.byref(params), g,
                                                         _ptr(rho), _ptr(acc_grav), p, nb, _stream()))


def nbody_pp_gravity_share(posm, n_total, rank, world, i0, i1, G, delta, acc_grav, ws):
    p, nb = _ws(ws)
    _chk("nbody_pp_gravity_share", load().nbody_pp_gravity_share(_ptr(posm), int(n_total), int(rank), int(world), int(i0),
                                                                 int(i1), float(G), float(delta), _ptr(acc_grav), p, nb,
                                                                 _stream()))


def nbody_pp_gravity_finish(posm, n_gas, n_halo, grid, G, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("nbody_pp_gravity_finish", load().nbody_pp_gravity_finish(_ptr(posm), int(n_gas), int(n_halo), g, float(G),
                                                                   _ptr(acc_grav), p, nb, _stream()))


def gravity_sums_view(ws, n_gas, n_total, grid=None) -> torch.Tensor:
    """int64 view of the workspace region that holds the pair-symmetric path's fixed-point sums (for the all-reduce)."""
    off, nbytes = C.c_size_t(0), C.c_size_t(0)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_workspace_gravity_sums", load().sph_workspace_gravity_sums(int(n_gas), int(n_total), g, C.byref(off),
                                                                         C.byref(nbytes)))
    return ws[off.value:off.value + nbytes.value].view(torch.int64)


# ---- the SPH passes shared as well: include/sph_b200.h
def sph_position_share_sph(posm, hsml, n_gas, n_halo, rank, world, i0, i1, params, grid, rho, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_position_share_sph", load().sph_position_share_sph(_ptr(posm), _ptr(hsml), int(n_gas), int(n_halo), int(rank),
                                                                 int(world), int(i0), int(i1), C.byref(params), g, _ptr(rho),
                                                                 _ptr(acc_grav), p, nb, _stream()))


def sph_renew_hsml(posm, hsml, sigma, n_gas, n_halo, params, grid, rho, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_renew_hsml", load().sph_renew_hsml(_ptr(posm), _ptr(hsml), float(sigma), int(n_gas), int(n_halo),
                                                 C.byref(params), g, _ptr(rho), p, nb, _stream()))


def sph_forces_share(vele, hsml, n_gas, n_halo, rank, world, params, grid, rho, acc_sph, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_forces_share", load().sph_forces_share(_ptr(vele), _ptr(hsml), int(n_gas), int(n_halo), int(rank), int(world),
                                                     C.byref(params), g, _ptr(rho), _ptr(acc_sph), p, nb, _stream()))


def sph_update(posm, vele, n_gas, n_halo, grid, dt, corrector, acc_sph, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_update", load().sph_update(_ptr(posm), _ptr(vele), int(n_gas), int(n_halo), g, float(dt), int(bool(corrector)),
                                         _ptr(acc_sph), _ptr(acc_grav), p, nb, _stream()))


def sph_position_slice(posm, hsml, sigma, n_gas, n_halo, i0, i1, params, grid, rho, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_position_slice", load().sph_position_slice(_ptr(posm), _ptr(hsml), float(sigma), int(n_gas), int(n_halo),
                                                         int(i0), int(i1), C.byref(params), g, _ptr(rho), _ptr(acc_grav),
                                                         p, nb, _stream()))


def sph_predict(posm, vele, hsml, n_gas, n_halo, params, grid, dt, rho, acc_sph, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_predict", load().sph_predict(_ptr(posm), _ptr(vele), _ptr(hsml), int(n_gas), int(n_halo), C.byref(params), g,
                                           float(dt), _ptr(rho), _ptr(acc_sph), _ptr(acc_grav), p, nb, _stream()))


def sph_correct(vele, hsml, n_gas, n_halo, params, grid, dt, rho, acc_sph, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_correct", load().sph_correct(_ptr(vele), _ptr(hsml), int(n_gas), int(n_halo), C.byref(params), g, float(dt),
                                           _ptr(rho), _ptr(acc_sph), _ptr(acc_grav), p, nb, _stream()))


# ------------------------------------------------------------------ NEXT-2: per-particle smoothing lengths
def sph_smoothing_lengths(posm, rho, n_gas, sigma, h_max, hsml):
    _chk("sph_smoothing_lengths", load().sph_smoothing_lengths(_ptr(posm), _ptr(rho), int(n_gas), float(sigma),
                                                               float(h_max), _ptr(hsml), _stream()))


def sph_density_h(posm, hsml, n_gas, params, grid, perm, cell_start, rho, ws):
    p, nb = _ws(ws)
    _chk("sph_density_h", load().sph_density_h(_ptr(posm), _ptr(hsml), int(n_gas), C.byref(params), C.byref(grid),
                                               _ptr(perm), _ptr(cell_start), _ptr(rho), p, nb, _stream()))


def sph_forces_h(posm, vele, rho, hsml, n_gas, params, grid, perm, cell_start, acc_sph, ws):
    p, nb = _ws(ws)
    _chk("sph_forces_h", load().sph_forces_h(_ptr(posm), _ptr(vele), _ptr(rho), _ptr(hsml), int(n_gas), C.byref(params),
                                             C.byref(grid), _ptr(perm), _ptr(cell_start), _ptr(acc_sph), p, nb, _stream()))


def sph_evaluate_h(posm, vele, hsml, n_gas, n_halo, params, grid, rho, acc_sph, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_evaluate_h", load().sph_evaluate_h(_ptr(posm), _ptr(vele), _ptr(hsml), int(n_gas), int(n_halo),
                                                 C.byref(params), g, _ptr(rho), _ptr(acc_sph), _ptr(acc_grav), p, nb,
                                                 _stream()))


def sph_step_h(posm, vele, hsml, n_gas, n_halo, params, grid, sigma, dt, first, rho, acc_sph, acc_grav, ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_step_h", load().sph_step_h(_ptr(posm), _ptr(vele), _ptr(hsml), int(n_gas), int(n_halo), C.byref(params), g,
                                         float(sigma), float(dt), int(bool(first)), _ptr(rho), _ptr(acc_sph),
                                         _ptr(acc_grav), p, nb, _stream()))


def sph_step_cfl(posm, vele, hsml, n_gas, n_halo, params, grid, sigma, c_cfl, dt_max, first, rho, acc_sph, acc_grav, dt_used,
                 ws):
    p, nb = _ws(ws)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_step_cfl", load().sph_step_cfl(_ptr(posm), _ptr(vele), _ptr(hsml), int(n_gas), int(n_halo), C.byref(params), g,
                                             float(sigma), float(c_cfl), float(dt_max), int(bool(first)), _ptr(rho),
                                             _ptr(acc_sph), _ptr(acc_grav), _ptr(dt_used), p, nb, _stream()))


def _hp(a):
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        assert not a.is_cuda and a.is_contiguous()
        return a.data_ptr()
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data


def sph_step_host(posm, vele, n_gas, n_halo, params, dt, n_steps, rho=None, acc_sph=None, acc_grav=None):
    """HOST arrays (numpy float32 or CPU torch tensors), updated in place."""
    _chk("sph_step_host", load().sph_step_host(_hp(posm), _hp(vele), int(n_gas), int(n_halo), C.byref(params),
                                               float(dt), int(n_steps), _hp(rho), _hp(acc_sph), _hp(acc_grav)))


class HostContext:
    """sph_host_ctx_*: persistent device buffers for repeated end-to-end calls on HOST arrays."""

    def __init__(self, n_gas, n_halo):
        self._h = C.c_void_p()
        _chk("sph_host_ctx_create", load().sph_host_ctx_create(int(n_gas), int(n_halo), C.byref(self._h)))

    def step(self, posm, vele, params, dt, n_steps, first=True, rho=None, acc_sph=None, acc_grav=None):
        _chk("sph_host_ctx_step", load().sph_host_ctx_step(self._h, _hp(posm), _hp(vele), C.byref(params), float(dt),
                                                           int(n_steps), int(bool(first)), _hp(rho), _hp(acc_sph),
                                                           _hp(acc_grav)))

    def close(self):
        if self._h:
            load().sph_host_ctx_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def sph_neighbour_lists(posm, n_gas, h, grid, perm, cell_start, ws, hsml=None):
    """Returns (count[n] uint32, offset[n+1] uint64 as int64 tensor, index[total] uint32) on the device.
    hsml: per-particle smoothing lengths (sph_neighbour_lists_h; h is then their cap)."""
    L = load()
    n = int(n_gas)
    cnt = torch.zeros(max(n, 1), dtype=torch.int32, device="cuda")
    off = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
    p, nb = _ws(ws)
    rc = L.sph_neighbour_lists_h(_ptr(posm), _ptr(hsml), n, float(h), C.byref(grid), _ptr(perm), _ptr(cell_start),
                                 _ptr(cnt), _ptr(off), None, 0, p, nb, _stream())
    total = int(off[n].item())
    if rc == SPH_OK and total == 0:
        return cnt[:n], off, torch.zeros(0, dtype=torch.int32, device="cuda")
    if rc != SPH_ERR_WORKSPACE:
        _chk("sph_neighbour_lists", rc)
    idx = torch.zeros(total, dtype=torch.int32, device="cuda")
    _chk("sph_neighbour_lists", L.sph_neighbour_lists_h(_ptr(posm), _ptr(hsml), n, float(h), C.byref(grid), _ptr(perm),
                                                        _ptr(cell_start), _ptr(cnt), _ptr(off), _ptr(idx), total, p, nb,
                                                        _stream()))
    return cnt[:n], off, idx


def sph_set_profiling(on: bool):
    _chk("sph_set_profiling", load().sph_set_profiling(int(bool(on))))


def sph_get_stage_ms() -> dict:
    out = (C.c_float * 5)()
    _chk("sph_get_stage_ms", load().sph_get_stage_ms(out))
    return dict(zip(STAGES, [float(x) for x in out]))


GRAV_PATHS = ("one_sided", "one_sided_uniform", "pair_symmetric", "pair_symmetric_general")


def sph_gravity_path(ws, n_gas, n_total, grid=None) -> str:
    """Which gravity kernel variant the last evaluation with workspace `ws` took (chosen on the device)."""
    p, nb = _ws(ws)
    out = C.c_int(-1)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_gravity_path", load().sph_gravity_path(p, nb, int(n_gas), int(n_total), g, C.byref(out), _stream()))
    return GRAV_PATHS[out.value]


SPH_STATUS_HSML_ABOVE_CAP = 1


def sph_workspace_status(ws, n_gas, n_total, grid=None) -> int:
    """Status bits the device raised in `ws` since the last read (read back and cleared; synchronises)."""
    p, nb = _ws(ws)
    out = C.c_uint32(0)
    g = C.byref(grid) if grid is not None else None
    _chk("sph_workspace_status", load().sph_workspace_status(p, nb, int(n_gas), int(n_total), g, C.byref(out), _stream()))
    return int(out.value)


def sph_dense_items(ws, n_gas, n_total, grid) -> int:
    """Work items the last density / forces / grid-building call with `ws` gave to the dense-cell walk (0: none)."""
    p, nb = _ws(ws)
    out = C.c_uint32(0)
    _chk("sph_dense_items", load().sph_dense_items(p, nb, int(n_gas), int(n_total), C.byref(grid), C.byref(out), _stream()))
    return int(out.value)


def sph_launch_count() -> int:
    return int(load().sph_launch_count())


class Simulation:
    """Convenience holder of the device buffers one run needs (no arithmetic: allocation and calls only)."""

    def __init__(self, workload, grid=None, sigma=None):
        """sigma: None = one global h (sph_step); a float = per-particle smoothing lengths (sph_step_h), started at
        the cap h_max = workload.h and renewed every step with that sigma (0 keeps them fixed)."""
        w = workload
        self.w = w
        self.n_gas, self.n_halo, self.n = w.n_gas, w.n_halo, w.n_total
        self.params = sph_params.from_workload(w)
        self.posm = torch.from_numpy(np.ascontiguousarray(w.posm)).cuda()
        self.vele = torch.from_numpy(np.ascontiguousarray(w.vele)).cuda()
        self.rho = torch.zeros(max(self.n_gas, 1), dtype=torch.float32, device="cuda")
        self.acc_sph = torch.zeros(max(self.n_gas, 1), 4, dtype=torch.float32, device="cuda")
        self.acc_grav = torch.zeros(max(self.n, 1), 4, dtype=torch.float32, device="cuda")
        self.grid = grid
        if self.grid is None and self.n_gas > 0:
            self.grid = sph_grid_from_bbox(self.posm, self.n_gas, w.h)
        self.ws = alloc_workspace(self.n_gas, self.n, self.grid)
        self.first = True
        self.sigma = sigma
        self.hsml = None
        if sigma is not None and self.n_gas > 0:
            self.hsml = torch.full((self.n_gas,), float(np.float32(w.h)), dtype=torch.float32, device="cuda")

    def evaluate(self):
        sph_evaluate_h(self.posm, self.vele, self.hsml, self.n_gas, self.n_halo, self.params, self.grid, self.rho,
                       self.acc_sph, self.acc_grav, self.ws)
        self.first = False

    def step(self, dt=None, c_cfl=None):
        """c_cfl: the step is min(dt, C_CFL min_i [...]) of Eq. 17, chosen on the device; self.dt_used (a device float)
        holds it afterwards."""
        dt = self.w.dt if dt is None else dt
        if c_cfl is None:
            sph_step_h(self.posm, self.vele, self.hsml, self.n_gas, self.n_halo, self.params, self.grid,
                       self.sigma or 0.0, dt, self.first, self.rho, self.acc_sph, self.acc_grav, self.ws)
        else:
            if getattr(self, "dt_used", None) is None:
                self.dt_used = torch.zeros(1, dtype=torch.float32, device="cuda")
            sph_step_cfl(self.posm, self.vele, self.hsml, self.n_gas, self.n_halo, self.params, self.grid,
                         self.sigma or 0.0, c_cfl, dt, self.first, self.rho, self.acc_sph, self.acc_grav, self.dt_used,
                         self.ws)
        self.first = False
