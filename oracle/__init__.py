"""Python face of the FP64 CPU oracle (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It never imports the CUDA package; the CUDA package never
imports it.  The arithmetic of the SPH sums, gravity, keys and sort lives in
sph_oracle.c; this file marshals arrays and writes out the O(N) formulas of the
integration scheme (Eqs. 12-16) and the step sequence (DESIGN.md
reading A11) in plain numpy FP64.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from .build import build as _build

_lib = None


class _Grid(C.Structure):
    _fields_ = [("origin", C.c_float * 3), ("cell", C.c_float), ("inv_cell", C.c_float), ("dims", C.c_int32 * 3)]


class _Params(C.Structure):
    _fields_ = [("h", C.c_double), ("gamma", C.c_double), ("alpha", C.c_double), ("beta", C.c_double),
                ("eta", C.c_double)]


@dataclass
class Grid:
    origin: tuple
    cell: float
    inv_cell: float
    dims: tuple

    @property
    def M(self) -> int:
        return int(self.dims[0]) * int(self.dims[1]) * int(self.dims[2])

    def _c(self) -> _Grid:
        g = _Grid()
        for a in range(3):
            g.origin[a] = self.origin[a]
            g.dims[a] = self.dims[a]
        g.cell = self.cell
        g.inv_cell = self.inv_cell
        return g


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        dp, fp, ip, up = (C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int64), C.POINTER(C.c_uint32))
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        for f in (L.orc_W, L.orc_Wp, L.orc_dWp_dxi):
            f.restype = C.c_double
            f.argtypes = [C.c_double, C.c_double]
        L.orc_gravity.argtypes = [dp, C.c_int64, C.c_double, C.c_double, ip, C.c_int64, dp]
        L.orc_gravity.restype = None
        L.orc_potential_energy.argtypes = [dp, C.c_int64, C.c_double, C.c_double]
        L.orc_potential_energy.restype = C.c_double
        L.orc_grid_from_bbox.argtypes = [dp, C.c_int64, C.c_float, C.POINTER(_Grid)]
        L.orc_grid_from_bbox.restype = C.c_int
        L.orc_cell_keys.argtypes = [dp, C.c_int64, C.POINTER(_Grid), up]
        L.orc_cell_keys.restype = None
        L.orc_counting_sort.argtypes = [up, C.c_int64, C.c_int64, up, up, up]
        L.orc_counting_sort.restype = C.c_int
        L.orc_rc2.argtypes = [C.c_float]
        L.orc_rc2.restype = C.c_float
        L.orc_neighbours_brute.argtypes = [dp, C.c_int64, C.c_float, fp, ip, C.c_int64, up, ip, up]
        L.orc_neighbours_brute.restype = None
        L.orc_neighbours_grid.argtypes = [dp, C.c_int64, C.c_float, fp, C.POINTER(_Grid), up, up, up, ip, C.c_int64,
                                          up, ip, up]
        L.orc_neighbours_grid.restype = None
        L.orc_density.argtypes = [dp, C.c_double, dp, ip, C.c_int64, ip, up, dp]
        L.orc_density.restype = None
        L.orc_cfl_terms.argtypes = [dp, dp, dp, C.POINTER(_Params), dp, ip, C.c_int64, ip, up, dp]
        L.orc_cfl_terms.restype = None
        L.orc_forces.argtypes = [dp, dp, dp, C.POINTER(_Params), dp, ip, C.c_int64, ip, up, dp, dp]
        L.orc_forces.restype = None
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _tg(targets):
    if targets is None:
        return None
    return np.ascontiguousarray(targets, dtype=np.int64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


# ------------------------------------------------------------------ kernels (Eqs. 8, 9)
def W(xi, h):
    return float(lib().orc_W(float(xi), float(h)))


def Wp(xi, h):
    return float(lib().orc_Wp(float(xi), float(h)))


def dWp_dxi(xi, h):
    return float(lib().orc_dWp_dxi(float(xi), float(h)))


# ------------------------------------------------------------------ gravity (Eq. 4)
def gravity(posm, G, delta, targets=None):
    """a^g for `targets` (default all) against all N sources; returns float64 [nt,3]."""
    posm = _f64(posm)
    n = posm.shape[0]
    tg = _tg(targets)
    nt = n if tg is None else len(tg)
    out = np.zeros((nt, 3), dtype=np.float64)
    if nt and n:
        lib().orc_gravity(_p(posm, C.c_double), n, float(G), float(delta), _p(tg, C.c_int64), nt, _p(out, C.c_double))
    return out


def potential_energy(posm, G, delta) -> float:
    posm = _f64(posm)
    return float(lib().orc_potential_energy(_p(posm, C.c_double), posm.shape[0], float(G), float(delta)))


# ------------------------------------------------------------------ grid sort (a1-a5)
def grid_from_bbox(posm, n_gas, h) -> Grid:
    posm = _f64(posm)
    g = _Grid()
    rc = lib().orc_grid_from_bbox(_p(posm, C.c_double), int(n_gas), np.float32(h), C.byref(g))
    if rc != 0:
        raise ValueError("grid_from_bbox: invalid grid (dimension > 4096, M >= 2^31 or no gas)")
    return Grid(tuple(g.origin), float(g.cell), float(g.inv_cell), tuple(g.dims))


def cell_keys(posm, n_gas, grid: Grid):
    posm = _f64(posm)
    key = np.zeros(int(n_gas), dtype=np.uint32)
    if n_gas:
        lib().orc_cell_keys(_p(posm, C.c_double), int(n_gas), C.byref(grid._c()), _p(key, C.c_uint32))
    return key


def counting_sort(key, M):
    """Returns (count[M], start[M+1], perm[n]) — perm maps sorted slot -> original index, stable."""
    key = np.ascontiguousarray(key, dtype=np.uint32)
    count = np.zeros(M, dtype=np.uint32)
    start = np.zeros(M + 1, dtype=np.uint32)
    perm = np.zeros(len(key), dtype=np.uint32)
    rc = lib().orc_counting_sort(_p(key, C.c_uint32), len(key), int(M), _p(count, C.c_uint32), _p(start, C.c_uint32),
                                 _p(perm, C.c_uint32))
    if rc != 0:
        raise ValueError("counting_sort: key out of range")
    return count, start, perm


def rc2(h) -> np.float32:
    return np.float32(lib().orc_rc2(np.float32(h)))


# ------------------------------------------------------------------ neighbour sets (O2)
def _hs32(hs):
    return None if hs is None else np.ascontiguousarray(hs, dtype=np.float32)


def _hs64(hs):
    return None if hs is None else np.ascontiguousarray(np.asarray(hs, dtype=np.float32), dtype=np.float64)


def smoothing_lengths(posm, rho, sigma, h_max):
    """L82: h_i = sigma (m_i / rho_i)^(1/3), capped at h_max (reading A25: the grid's cells are 2 h_max wide,
    so no pair farther apart than that can be found).  Returned as FP32, the type both sides carry h in."""
    m = _f64(posm)[: len(rho), 3]
    return np.minimum(float(sigma) * np.cbrt(m / np.asarray(rho, dtype=np.float64)), float(h_max)).astype(np.float32)


def neighbours(posm, n_gas, h, targets=None, method="brute", grid=None, sort=None, hs=None):
    """CSR neighbour lists (offsets int64[nt+1], index uint32[...]), each list ascending in j, j != i.
    method "brute": definition, O(nt * n_gas).  method "grid": the oracle's own 3x3x3 search.
    hs: per-particle smoothing lengths (FP32, all <= h): pair cutoff fl(fl(h_i + h_j)^2) (reading A24)."""
    posm = _f64(posm)
    hs = _hs32(hs)
    tg = _tg(targets)
    nt = int(n_gas) if tg is None else len(tg)
    cnt = np.zeros(nt, dtype=np.uint32)
    L = lib()
    if method == "grid":
        if grid is None:
            grid = grid_from_bbox(posm, n_gas, h)
        if sort is None:
            key = cell_keys(posm, n_gas, grid)
            _, start, perm = counting_sort(key, grid.M)
        else:
            key, start, perm = sort
        gc = grid._c()

        def call(c, off, idx):
            L.orc_neighbours_grid(_p(posm, C.c_double), int(n_gas), np.float32(h), _p(hs, C.c_float), C.byref(gc), _p(key, C.c_uint32),
                                  _p(start, C.c_uint32), _p(perm, C.c_uint32), _p(tg, C.c_int64), nt, _p(c, C.c_uint32),
                                  _p(off, C.c_int64), _p(idx, C.c_uint32))
    else:
        def call(c, off, idx):
            L.orc_neighbours_brute(_p(posm, C.c_double), int(n_gas), np.float32(h), _p(hs, C.c_float), _p(tg, C.c_int64), nt,
                                   _p(c, C.c_uint32), _p(off, C.c_int64), _p(idx, C.c_uint32))
    if nt:
        call(cnt, None, None)
    off = np.zeros(nt + 1, dtype=np.int64)
    np.cumsum(cnt, out=off[1:])
    idx = np.zeros(max(int(off[-1]), 1), dtype=np.uint32)
    if nt and off[-1] > 0:
        call(cnt, off, idx)
    return off, idx[: int(off[-1])]


# ------------------------------------------------------------------ SPH sums (Eqs. 7, 10, 11)
def density(posm, h, offsets, index, targets=None, hs=None):
    posm = _f64(posm)
    hs = _hs64(hs)
    tg = _tg(targets)
    nt = len(offsets) - 1
    rho = np.zeros(nt, dtype=np.float64)
    idx = np.ascontiguousarray(index, dtype=np.uint32)
    if len(idx) == 0:
        idx = np.zeros(1, dtype=np.uint32)
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    if nt:
        lib().orc_density(_p(posm, C.c_double), float(h), _p(hs, C.c_double), _p(tg, C.c_int64), nt, _p(off, C.c_int64), _p(idx, C.c_uint32),
                          _p(rho, C.c_double))
    return rho


def forces(posm, vele, rho_all, h, offsets, index, targets=None, gamma=5.0 / 3.0, alpha=0.5, beta=1.0, eta=0.1,
           with_gross=False, hs=None):
    """(ax, ay, az, de/dt) of Eqs. 10-11 (hydro part) for `targets`; rho_all indexed by gas index.
    with_gross: also return [nt,2] sums of the term magnitudes (conditioning diagnostic, reading A17)."""
    posm, vele, rho_all = _f64(posm), _f64(vele), _f64(rho_all)
    tg = _tg(targets)
    nt = len(offsets) - 1
    out = np.zeros((nt, 4), dtype=np.float64)
    idx = np.ascontiguousarray(index, dtype=np.uint32)
    if len(idx) == 0:
        idx = np.zeros(1, dtype=np.uint32)
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    prm = _Params(float(h), float(gamma), float(alpha), float(beta), float(eta))
    gross = np.zeros((nt, 2), dtype=np.float64) if with_gross else None
    hs = _hs64(hs)
    if nt:
        lib().orc_forces(_p(posm, C.c_double), _p(vele, C.c_double), _p(rho_all, C.c_double), C.byref(prm),
                         _p(hs, C.c_double), _p(tg, C.c_int64), nt, _p(off, C.c_int64), _p(idx, C.c_uint32), _p(out, C.c_double),
                         _p(gross, C.c_double))
    return (out, gross) if with_gross else out


def cfl_dt(posm, vele, rho_all, acc_sph, acc_grav, h, offsets, index, c_cfl, targets=None, gamma=5.0 / 3.0, alpha=0.5,
           beta=1.0, eta=0.1, hs=None):
    """Eq. 17 (L125-129): returns (dt, bracket[nt]) with dt = C_CFL min_i bracket_i,
    bracket_i = s_i / (c_i^max (1 + 1.2 alpha) + 1.2 beta mu_i^max + sqrt(s_i (|Q_i| + |E_i|))).
    acc_sph[nt,4] = (a_sph, de/dt) and acc_grav[nt,>=3] are given FOR THE TARGETS (Q_i = a_sph + a_grav is the
    right-hand side of Eq. 10, E_i of Eq. 11); rho_all is indexed by gas index.
    hs: per-particle smoothing lengths (L82): mu_ij then uses h_ij = (h_i + h_j)/2 and a particle without a neighbour
    takes s = 2 h_i (reading A22)."""
    posm, vele, rho_all = _f64(posm), _f64(vele), _f64(rho_all)
    tg = _tg(targets)
    nt = len(offsets) - 1
    terms = np.zeros((nt, 3), dtype=np.float64)
    idx = np.ascontiguousarray(index, dtype=np.uint32)
    if len(idx) == 0:
        idx = np.zeros(1, dtype=np.uint32)
    off = np.ascontiguousarray(offsets, dtype=np.int64)
    prm = _Params(float(h), float(gamma), float(alpha), float(beta), float(eta))
    if nt == 0:
        return np.inf, np.zeros(0)
    hs = _hs64(hs)
    lib().orc_cfl_terms(_p(posm, C.c_double), _p(vele, C.c_double), _p(rho_all, C.c_double), C.byref(prm),
                        _p(hs, C.c_double), _p(tg, C.c_int64), nt, _p(off, C.c_int64), _p(idx, C.c_uint32), _p(terms, C.c_double))
    a_s = np.asarray(acc_sph, dtype=np.float64)
    a_g = np.asarray(acc_grav, dtype=np.float64)
    Q = np.linalg.norm(a_s[:, :3] + a_g[:, :3], axis=1)
    E = np.abs(a_s[:, 3])
    s, cmax, mumax = terms[:, 0], terms[:, 1], terms[:, 2]
    with np.errstate(divide="ignore"):
        bracket = s / (cmax * (1.0 + 1.2 * alpha) + 1.2 * beta * mumax + np.sqrt(s * (Q + E)))
    return float(c_cfl * bracket.min()), bracket


# ------------------------------------------------------------------ whole evaluation / step (O6)
@dataclass
class State:
    """Carried state of the scheme (reading A11): r, v, e and the position-only
    quantities at the current r (rho, a_grav)."""
    posm: np.ndarray      # float64 [N,4]
    vele: np.ndarray      # float64 [N,4]
    n_gas: int
    rho: np.ndarray = None       # float64 [n_gas]
    acc_grav: np.ndarray = None  # float64 [N,3]


def _nbr(posm, n_gas, h, method, hs=None):
    if n_gas == 0:
        return np.zeros(1, dtype=np.int64), np.zeros(0, dtype=np.uint32)
    return neighbours(posm, n_gas, h, method=method, hs=hs)


def position_only(state: State, h, G, delta, method="grid", hs=None):
    """SP + DC + GFC at the current positions (the quantities that depend on r only, L123).
    hs: per-particle smoothing lengths (then h is their cap h_max, which sizes the grid)."""
    off, idx = _nbr(state.posm, state.n_gas, h, method, hs)
    state.rho = density(state.posm, h, off, idx, hs=hs)
    state.acc_grav = gravity(state.posm, G, delta) if G != 0.0 else np.zeros((len(state.posm), 3))
    return off, idx


def hydro(state: State, h, nbr, hs=None, **visc):
    if state.n_gas == 0:
        return np.zeros((0, 4))
    off, idx = nbr
    return forces(state.posm, state.vele, state.rho, h, off, idx, hs=hs, **visc)


def step(state: State, dt, h, G, delta, nbr=None, method="grid", hs=None, sigma=0.0, c_cfl=None, **visc):
    """One predictor-corrector step, Eqs. 12-16 (L103-121), sequence of DESIGN.md A11:
    HFC(pred) -> SU(pred) -> SP, DC, GFC at r(t+dt) -> HFC(corr) -> SU(corr).
    `state` must carry rho and acc_grav at the current r (call position_only first);
    `nbr` are the neighbour lists at the current r (recomputed if None).
    Returns (new_state, nbr_new, diagnostics).
    Per-particle smoothing lengths (L82, reading A26): with `hs` the pair length is h_ij = (h_i + h_j)/2 and h is the
    cap h_max; with sigma > 0 the lengths are renewed from the refined density, h_i = min(sigma (m_i/rho_i)^(1/3), h_max),
    right after DC at r(t+dt) — the density itself was summed with the old lengths — and used by the corrector and by
    the next step (diag["hs"]).
    Step size (Eq. 17): with c_cfl the step taken is min(dt, C_CFL min_i [...]) (diag["dt"]), the bracket
    evaluated over the gas particles at the time layer t the step starts from — s^min, c^max, mu^max come out of the
    same neighbour walk as HFC(predictor), Q_i and E_i are that walk's results — so `dt` is then the largest step
    allowed (and the step of a run without gas, which Eq. 17 does not bound)."""
    ng = state.n_gas
    if nbr is None:
        nbr = _nbr(state.posm, ng, h, method, hs)
    Q = state.acc_grav.copy()                                  # halo: Q_i = a^g_i
    hy = hydro(state, h, nbr, hs=hs, **visc)                   # HFC(predictor) at (r, v, e, rho)(t)
    Q[:ng] += hy[:, :3]
    E = hy[:, 3] if ng else np.zeros(0)
    bracket = None
    if c_cfl is not None and ng:
        dt_cfl, bracket = cfl_dt(state.posm, state.vele, state.rho, hy, state.acc_grav[:ng], h, nbr[0], nbr[1], c_cfl, hs=hs,
                                 **visc)
        dt = min(float(dt), dt_cfl)
    v0 = state.vele[:, :3].copy()
    e0 = state.vele[:ng, 3].copy()
    v_t = v0 + dt * Q                                          # Eq. 12
    e_t = e0 + dt * E                                          # Eq. 13
    new = State(state.posm.copy(), state.vele.copy(), ng)
    new.posm[:, :3] = state.posm[:, :3] + 0.5 * dt * (v_t + v0)   # Eq. 14
    new.vele[:, :3] = v_t
    new.vele[:ng, 3] = e_t
    nbr1 = position_only(new, h, G, delta, method, hs=hs)      # density "refined" (L115), gravity once (L123)
    hs1 = hs
    if hs is not None and sigma > 0.0 and ng:
        hs1 = smoothing_lengths(new.posm, new.rho, sigma, h)
        nbr1 = _nbr(new.posm, ng, h, method, hs1)              # the pair cutoff follows the lengths
    Q1 = new.acc_grav.copy()
    hy1 = hydro(new, h, nbr1, hs=hs1, **visc)                  # HFC(corrector) at (r(t+dt), v~, e~, rho(t+dt))
    Q1[:ng] += hy1[:, :3]
    E1 = hy1[:, 3] if ng else np.zeros(0)
    new.vele[:, :3] = 0.5 * (v0 + v_t) + 0.5 * dt * Q1         # Eq. 15
    new.vele[:ng, 3] = 0.5 * (e0 + e_t) + 0.5 * dt * E1        # Eq. 16
    diag = dict(hydro_pred=hy, hydro_corr=hy1, v_pred=v_t, e_pred=e_t, hs=hs1, dt=float(dt), cfl_bracket=bracket)
    return new, nbr1, diag


def total_energy(state: State, G, delta) -> float:
    """E = sum 1/2 m v^2 + sum_gas m e + U (pin P7)."""
    m = state.posm[:, 3]
    ke = 0.5 * np.sum(m * np.sum(state.vele[:, :3] ** 2, axis=1))
    ie = np.sum(m[: state.n_gas] * state.vele[: state.n_gas, 3])
    return float(ke + ie + (potential_energy(state.posm, G, delta) if G != 0.0 else 0.0))
