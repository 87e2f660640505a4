"""Pins for the oracle: what the paper and the mathematics fix,
checked without reference to the oracle's own formulas.  CPU only."""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_1807_08116_b200 import workloads as wl

PI = math.pi


# ---------------------------------------------------------------- P2: kernels (Eqs. 8, 9; L69)
def _simpson(f, a, b, n=20000):
    x = np.linspace(a, b, n + 1)
    y = np.array([f(t) for t in x])
    return (b - a) / (3 * n) * (y[0] + y[-1] + 4 * y[1:-1:2].sum() + 2 * y[2:-1:2].sum())


@pytest.mark.parametrize("h", [1.0, 0.2, 0.05])
def test_P2_W_normalised(h):
    # L69: integral of W over space = 1.  4 pi int_0^{2h} W(r/h, h) r^2 dr, split at the knot r = h.
    f = lambda r: 4 * PI * oracle.W(r / h, h) * r * r
    total = _simpson(f, 0, h) + _simpson(f, h, 2 * h)
    assert abs(total - 1.0) < 1e-12
    # the two pieces separately, exact rationals 19/120 and 11/120 (tests/golden/closed_forms.txt)
    assert abs(_simpson(f, 0, h) - 4 * Fraction(19, 120)) < 1e-12
    assert abs(_simpson(f, h, 2 * h) - 4 * Fraction(11, 120)) < 1e-12
    assert oracle.W(2.0, h) == 0.0 and oracle.W(2.5, h) == 0.0
    # continuity at the knot xi = 1 and value at 0
    assert abs(oracle.W(1.0 - 1e-12, h) - oracle.W(1.0 + 1e-12, h)) < 1e-9 / h ** 3
    assert abs(oracle.W(0.0, h) * PI * h ** 3 - 1.0) < 1e-15


@pytest.mark.parametrize("h", [1.0, 0.1])
def test_P2_Wp_normalised(h):
    f = lambda r: 4 * PI * oracle.Wp(r / h, h) * r * r
    assert abs(_simpson(f, 0, 2 * h) - 1.0) < 1e-12
    assert abs(oracle.Wp(0.0, h) * h ** 3 - 15 * 8 / (64 * PI)) < 1e-15
    assert oracle.Wp(2.0, h) == 0.0


def test_P2_dWp_is_derivative_of_Wp():
    # reading A3: dWp/dxi is Eq. 9 differentiated.  Central differences of the oracle's own Wp
    # pin the *relation*; the closed value -45/(16 pi h^3) at 0 pins the scale.
    h = 0.7
    for xi in [0.0, 0.3, 1.0, 1.7, 1.999]:
        d = 1e-6
        lo = max(xi - d, 0.0)
        num = (oracle.Wp(xi + d, h) - oracle.Wp(lo, h)) / (xi + d - lo)
        assert abs(num - oracle.dWp_dxi(xi, h)) < 2e-5 / h ** 3
    assert abs(oracle.dWp_dxi(0.0, h) * PI * h ** 3 - (-45 / 16)) < 1e-14
    assert oracle.dWp_dxi(2.0, h) == 0.0


def test_L84_cubic_spline_clustering_region():
    # L84: lim dW/dxi = 0 at xi -> 0 and the force weakens for 0 < xi < 2/3: |dW/dxi| is maximal at 2/3.
    h = 1.0
    d = 1e-6
    dW = lambda x: (oracle.W(x + d, h) - oracle.W(max(x - d, 0), h)) / (x + d - max(x - d, 0))
    assert abs(dW(0.0)) < 1e-5
    xs = np.linspace(0.01, 1.99, 397)
    assert abs(xs[np.argmin([dW(x) for x in xs])] - 2 / 3) < 0.01
    assert abs(dW(2 / 3) * PI - (-1.0)) < 1e-5


# ---------------------------------------------------------------- P4: two-body Eq. 4
def test_P4_two_body_closed_form():
    G, delta = 2.5, 0.3
    posm = np.array([[0.1, -0.2, 0.3, 2.0], [1.1, 0.8, -0.7, 0.5]], dtype=np.float32)
    a = oracle.gravity(posm, G, delta)
    p = posm.astype(np.float64)
    dr = p[0, :3] - p[1, :3]
    d2 = dr @ dr
    a0 = -G * p[1, 3] * dr / (d2 + delta ** 2) ** 1.5
    assert np.allclose(a[0], a0, rtol=1e-14, atol=0)
    assert np.allclose(a[1], -(p[0, 3] / p[1, 3]) * a0, rtol=1e-14, atol=0)
    # direction: attraction (a_0 points from 0 to 1)
    assert a[0] @ (p[1, :3] - p[0, :3]) > 0
    # coincident bodies: exactly zero; also with delta = 0 (0/0 skipped)
    same = np.array([[1, 2, 3, 1.0], [1, 2, 3, 2.0]], dtype=np.float32)
    assert np.all(oracle.gravity(same, G, delta) == 0.0)
    assert np.all(oracle.gravity(same, G, 0.0) == 0.0)
    # delta = 0, unit separation: plain Newton
    unit = np.array([[0, 0, 0, 1.0], [1, 0, 0, 3.0]], dtype=np.float32)
    assert np.allclose(oracle.gravity(unit, 1.0, 0.0), [[3.0, 0, 0], [-1.0, 0, 0]], rtol=1e-15)
    # far field: softening irrelevant, inverse-square law
    far = np.array([[0, 0, 0, 1.0], [1000, 0, 0, 1.0]], dtype=np.float32)
    assert abs(oracle.gravity(far, 1.0, 0.01)[0, 0] - 1e-6) < 1e-15


def test_P4_gravity_targets_subset_and_sign_matches_numpy():
    w = wl.make_workload(0, scale=0.05)
    p = w.posm.astype(np.float64)
    tg = np.array([0, 5, 17, w.n_total - 1])
    a = oracle.gravity(w.posm, w.G, w.delta, targets=tg)
    for t, i in enumerate(tg):
        dr = p[i, :3] - p[:, :3]
        r2 = (dr ** 2).sum(1) + w.delta ** 2
        ref = -(w.G * p[:, 3] / r2 ** 1.5) @ dr
        assert np.allclose(a[t], ref, rtol=1e-12)


# ---------------------------------------------------------------- P5: momentum
def test_P5_gravity_momentum_zero():
    w = wl.make_workload(0, scale=0.125)
    a = oracle.gravity(w.posm, w.G, w.delta)
    m = w.posm[:, 3].astype(np.float64)
    assert np.linalg.norm((m[:, None] * a).sum(0)) <= 1e-13 * (m * np.linalg.norm(a, axis=1)).sum()


def _dense_gas(n=1500, seed=7, h=0.11, e_lo=0.5):
    rng = np.random.Generator(np.random.Philox(key=[seed, 0]))
    posm = np.zeros((n, 4), np.float32)
    vele = np.zeros((n, 4), np.float32)
    posm[:, :3] = rng.random((n, 3))
    posm[:, 3] = (0.5 + rng.random(n)) / n          # unequal masses on purpose
    vele[:, :3] = rng.standard_normal((n, 3)) * 0.5
    vele[:, 3] = e_lo + 0.5 * rng.random(n)
    return posm, vele, h


def test_P5_P6_sph_momentum_and_energy_identity():
    posm, vele, h = _dense_gas()
    n = len(posm)
    off, idx = oracle.neighbours(posm, n, h)
    assert (off[1:] - off[:-1]).mean() > 15          # a real SPH neighbourhood
    rho = oracle.density(posm, h, off, idx)
    f = oracle.forces(posm, vele, rho, h, off, idx)
    m = posm[:, 3].astype(np.float64)
    v = vele[:, :3].astype(np.float64)
    scale = (m * np.linalg.norm(f[:, :3], axis=1)).sum()
    # P5: "ensuring Newton's third law" (L95) -> sum m_i a_i = 0.  Holds only with p_j/rho_j^2 (reading A2).
    assert np.linalg.norm((m[:, None] * f[:, :3]).sum(0)) <= 1e-13 * scale
    # P6: Pi_ij symmetric, grad W_p antisymmetric -> sum m (de/dt + v.a) = 0: pins the sign and 1/2 of Eq. 11.
    resid = (m * f[:, 3]).sum() + (m * (v * f[:, :3]).sum(1)).sum()
    assert abs(resid) <= 1e-13 * ((m * np.abs(f[:, 3])).sum() + (m * np.abs((v * f[:, :3]).sum(1))).sum())
    assert np.abs(f[:, 3]).max() > 0


def test_P6_compression_heats_expansion_cools():
    posm, vele, h = _dense_gas(n=800, h=0.14)
    n = len(posm)
    off, idx = oracle.neighbours(posm, n, h)
    rho = oracle.density(posm, h, off, idx)
    m = posm[:, 3].astype(np.float64)
    c = posm[:, :3] - 0.5
    vin, vout = vele.copy(), vele.copy()
    vin[:, :3] = -c
    vout[:, :3] = c
    assert (m * oracle.forces(posm, vin, rho, h, off, idx)[:, 3]).sum() > 0     # Eq. 3: de/dt = -(p/rho) div v
    assert (m * oracle.forces(posm, vout, rho, h, off, idx)[:, 3]).sum() < 0
    # pressure gradient pushes outward from an over-dense blob: mean radial acceleration of the outer shell > 0
    still = vele.copy()
    still[:, :3] = 0
    a = oracle.forces(posm, still, rho, h, off, idx)[:, :3]
    r = np.linalg.norm(c, axis=1)
    shell = r > 0.6
    assert ((a[shell] * c[shell]).sum(1) / r[shell]).mean() > 0


# ---------------------------------------------------------------- P10: one SPH pair by hand
def test_P10_single_pair_by_hand():
    h, gamma, alpha, beta, eta = 0.5, 1.4, 0.5, 1.0, 0.1
    m1, m2, e1, e2 = 0.3, 0.7, 1.2, 0.8
    d = 0.6                                                     # xi = 1.2: outer branch of Eq. 8
    posm = np.array([[0, 0, 0, m1], [d, 0, 0, m2]], dtype=np.float64)
    vele = np.array([[0.4, 0.1, 0, e1], [-0.2, 0.0, 0, e2]], dtype=np.float64)   # approaching
    off, idx = oracle.neighbours(posm, 2, h)
    assert off.tolist() == [0, 1, 2] and idx.tolist() == [1, 0]
    rho = oracle.density(posm, h, off, idx)
    s = 1 / (PI * h ** 3)
    xi = d / h
    w12 = s * 0.25 * (2 - xi) ** 3
    assert np.allclose(rho, [m1 * s + m2 * w12, m2 * s + m1 * w12], rtol=1e-15)
    f = oracle.forces(posm, vele, rho, h, off, idx, gamma=gamma, alpha=alpha, beta=beta, eta=eta)
    p1, p2 = (gamma - 1) * rho[0] * e1, (gamma - 1) * rho[1] * e2          # Eq. 5
    c1, c2 = math.sqrt(gamma * p1 / rho[0]), math.sqrt(gamma * p2 / rho[1])
    dr = np.array([-d, 0, 0])                                              # r_1 - r_2
    dv = np.array([0.6, 0.1, 0])                                           # v_1 - v_2
    rv = dr @ dv
    assert rv < 0
    mu = h * rv / (d * d + eta * h * h)
    nu = mu * (beta * mu - alpha * 0.5 * (c1 + c2)) / (0.5 * (rho[0] + rho[1]))
    Pi = p1 / rho[0] ** 2 + p2 / rho[1] ** 2 + nu
    gradWp = (-45 / (64 * PI * h ** 3) * (2 - xi) ** 2) * (dr / d) / h      # L95 with Eq. 9
    assert np.allclose(f[0, :3], -m2 * Pi * gradWp, rtol=1e-14)
    assert np.allclose(f[1, :3], +m1 * Pi * gradWp, rtol=1e-14)
    assert np.isclose(f[0, 3], 0.5 * m2 * Pi * (dv @ gradWp), rtol=1e-14)
    assert np.isclose(f[1, 3], 0.5 * m1 * Pi * (dv @ gradWp), rtol=1e-14)
    # repulsive: particle 1 (at the origin) is pushed towards -x
    assert f[0, 0] < 0 < f[1, 0]
    # receding pair: viscosity off (mu = 0), Pi is the pure pressure term
    vele2 = vele.copy()
    vele2[:, :3] *= -1
    f2 = oracle.forces(posm, vele2, rho, h, off, idx, gamma=gamma, alpha=alpha, beta=beta, eta=eta)
    Pi0 = p1 / rho[0] ** 2 + p2 / rho[1] ** 2
    assert np.allclose(f2[0, :3], -m2 * Pi0 * gradWp, rtol=1e-14)


def _golden_frac(name):
    import os
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")):
        f = line.split()
        if f and f[0] == name:
            return float(Fraction(f[1]))
    raise KeyError(name)


def test_A17_gross_sums_by_hand():
    """The second output of oracle.forces, S_i = (sum_j |m_j Pi_ij grad W_p|, sum_j |1/2 m_j Pi_ij dv.grad W_p|), sets the
    floor of the parity tolerance (reading A17, tests/parity_util.py), so it is pinned like a value:
    (1) one pair (the P10 configuration): a single term, so S equals the magnitude of the value itself;
    (2) three collinear particles worked by hand (tests/golden/closed_forms.txt: gross_collinear_*): the two terms of
        the middle particle cancel exactly — value 0, S = twice one term — which is the situation S exists for;
    (3) the same with unequal neighbour masses: value = difference, S = sum of the two magnitudes."""
    # (1) P10's pair, viscosity on (approaching)
    h, gamma = 0.5, 1.4
    posm = np.array([[0, 0, 0, 0.3], [0.6, 0, 0, 0.7]], dtype=np.float64)
    vele = np.array([[0.4, 0.1, 0, 1.2], [-0.2, 0.0, 0, 0.8]], dtype=np.float64)
    off, idx = oracle.neighbours(posm, 2, h)
    rho = oracle.density(posm, h, off, idx)
    f, g = oracle.forces(posm, vele, rho, h, off, idx, gamma=gamma, with_gross=True)
    assert g.shape == (2, 2)
    assert np.allclose(g[:, 0], np.linalg.norm(f[:, :3], axis=1), rtol=1e-14)
    assert np.allclose(g[:, 1], np.abs(f[:, 3]), rtol=1e-14)
    assert np.all(g > 0)
    # (2) three collinear particles; rho is an INPUT of the force sums, so round values are given
    h = 1.0
    posm = np.array([[0, 0, 0, 1.0], [1, 0, 0, 2.0], [-1, 0, 0, 2.0]], dtype=np.float64)
    vele = np.array([[0, 0, 0, 1.5], [0.5, 0, 0, 1.5], [0.5, 0, 0, 1.5]], dtype=np.float64)
    rho = np.array([1.0, 2.0, 2.0])
    off, idx = oracle.neighbours(posm, 3, h)
    assert np.diff(off).tolist() == [2, 1, 1]                   # the outer two are exactly 2h apart: not a pair (A8)
    kw = dict(gamma=5.0 / 3.0, alpha=0.0, beta=0.0, eta=0.1)
    f, g = oracle.forces(posm, vele, rho, h, off, idx, with_gross=True, **kw)
    assert np.all(np.abs(f[0]) < 1e-16)                         # exact cancellation
    assert np.isclose(g[0, 0] * PI, _golden_frac("gross_collinear_a_times_pi"), rtol=1e-14)
    assert np.isclose(g[0, 1] * PI, _golden_frac("gross_collinear_e_times_pi"), rtol=1e-14)
    # the outer particles have one term each: S = |value| again, half of the middle particle's S per unit mass
    assert np.allclose(g[1:, 0], np.linalg.norm(f[1:, :3], axis=1), rtol=1e-14)
    assert np.allclose(g[1:, 1], np.abs(f[1:, 3]), rtol=1e-14)
    assert np.isclose(g[1, 0] * 2 * posm[1, 3] / posm[0, 3], g[0, 0], rtol=1e-14)   # term m_0 Pi |grad| vs 2 terms m_1 Pi |grad|
    # (3) unequal neighbour masses: net and gross differ
    posm[2, 3] = 1.0
    f, g = oracle.forces(posm, vele, rho, h, off, idx, with_gross=True, **kw)
    assert np.isclose(f[0, 0] * PI, _golden_frac("gross_unequal_net_times_pi"), rtol=1e-14)
    assert np.isclose(g[0, 0] * PI, _golden_frac("gross_unequal_a_times_pi"), rtol=1e-14)
    assert f[0, 1] == 0 and f[0, 2] == 0
    # S never falls below the value it bounds, on a dense random gas (triangle inequality), and is invariant under
    # relabelling of the neighbours (a sum of magnitudes has no order)
    posm, vele, h = _dense_gas()
    n = len(posm)
    off, idx = oracle.neighbours(posm, n, h)
    rho = oracle.density(posm, h, off, idx)
    f, g = oracle.forces(posm, vele, rho, h, off, idx, with_gross=True)
    assert np.all(g[:, 0] >= np.linalg.norm(f[:, :3], axis=1) * (1 - 1e-12))
    assert np.all(g[:, 1] >= np.abs(f[:, 3]) * (1 - 1e-12))


def test_A9_coincident_pair_contributes_density_only():
    h = 0.5
    posm = np.array([[1, 1, 1, 0.2], [1, 1, 1, 0.3], [1.3, 1, 1, 0.1]], dtype=np.float32)
    vele = np.array([[0, 0, 0, 1.0], [1, 0, 0, 1.0], [0, 0, 0, 1.0]], dtype=np.float32)
    off, idx = oracle.neighbours(posm, 3, h)
    assert idx[off[0]:off[1]].tolist() == [1, 2]
    rho = oracle.density(posm, h, off, idx)
    s = 1 / (PI * h ** 3)
    xi = float(np.float64(posm[2, 0]) - 1.0) / h
    w = s * (1 - 1.5 * xi ** 2 + 0.75 * xi ** 3)
    assert np.isclose(rho[0], (0.2 + 0.3) * s + np.float64(posm[2, 3]) * w, rtol=1e-7)
    f = oracle.forces(posm, vele, rho, h, off, idx)
    assert np.all(np.isfinite(f))
    # particle 0's force comes from particle 2 alone
    f_wo = oracle.forces(posm, vele, rho, h, np.array([0, 1, 1, 1]), np.array([2], dtype=np.uint32))
    assert np.allclose(f[0], f_wo[0])


# ---------------------------------------------------------------- P3: uniform lattice
@pytest.mark.parametrize("ratio,expect", [(1.0, None), (1.2, 1.000809548), (1.3, 0.997261828), (2.0, 1.000079182)])
def test_P3_lattice_density(ratio, expect):
    a, rho0 = 0.1, 3.0
    w = wl.lattice(11, a, rho0=rho0)
    h = ratio * a
    n = w.n_gas
    off, idx = oracle.neighbours(w.posm, n, h)
    rho = oracle.density(w.posm, h, off, idx)
    pos = w.posm[:, :3].astype(np.float64)
    interior = np.all(np.abs(pos) <= 5 * a - 2 * h - 1e-6, axis=1)
    assert interior.sum() >= 1
    r_int = rho[interior] / np.float64(w.posm[0, 3]) * a ** 3      # in units of rho0 (FP32 mass as stored)
    # independent value: direct lattice sum of Eq. 8 in exact lattice geometry
    rng = range(-5, 6)
    tot = 0.0
    for i in rng:
        for j in rng:
            for k in rng:
                xi = math.sqrt(i * i + j * j + k * k) / ratio
                if xi <= 1:
                    tot += 1 - 1.5 * xi ** 2 + 0.75 * xi ** 3
                elif xi < 2:
                    tot += 0.25 * (2 - xi) ** 3
    lat = tot / (PI * ratio ** 3)
    assert np.allclose(r_int, lat, rtol=2e-6)      # FP32 lattice coordinates
    if ratio == 1.0:
        closed = (1 + 6 / 4 + 12 / 4 * (2 - math.sqrt(2)) ** 3 + 8 / 4 * (2 - math.sqrt(3)) ** 3) / PI
        assert abs(closed - 0.999972466) < 1e-9     # tests/golden/closed_forms.txt
        assert abs(lat - closed) < 1e-12
    else:
        assert abs(lat - expect) < 1e-8
    assert np.all(np.abs(r_int - 1) < 5e-3)        # "equal to rho0 in the interior" (north star check 3)
    # symmetry: no hydro force and no heating in the interior for uniform e and v
    f = oracle.forces(w.posm, w.vele, rho, h, off, idx)
    deep = np.all(np.abs(pos) <= 5 * a - 4 * h - 1e-6, axis=1)
    if deep.any():
        typical = np.abs(f[~interior, :3]).max()
        assert np.abs(f[deep]).max() < 1e-5 * typical


# ---------------------------------------------------------------- P1 / P9: grid sort and neighbour sets
def _check_sort(key, M, count, start, perm):
    n = len(key)
    # L171 recurrence, sequentially (independent of the oracle's loop): incl[k] = incl[k-1] + count[k]
    assert start[0] == 0 and start[M] == n
    assert np.array_equal(np.diff(start.astype(np.int64)), count.astype(np.int64))
    assert np.array_equal(count, np.bincount(key, minlength=M).astype(np.uint32))
    assert np.array_equal(np.sort(perm), np.arange(n, dtype=np.uint32))           # bijection
    ks = key[perm]
    assert np.all(np.diff(ks.astype(np.int64)) >= 0)                              # key o perm non-decreasing
    same = ks[1:] == ks[:-1]
    assert np.all(perm[1:][same] > perm[:-1][same])                               # stable inside a cell
    assert np.array_equal(perm, np.argsort(key, kind="stable").astype(np.uint32))  # library routine


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_P9_counting_sort_invariants(seed):
    rng = np.random.Generator(np.random.Philox(key=[seed, 9]))
    M = 777
    key = rng.integers(0, M, size=5000).astype(np.uint32)
    key[rng.integers(0, 5000, 800)] = 13          # one crowded cell
    count, start, perm = oracle.counting_sort(key, M)
    _check_sort(key, M, count, start, perm)
    with pytest.raises(ValueError):
        oracle.counting_sort(np.array([M], dtype=np.uint32), M)


def test_A7_grid_geometry_and_keys():
    w = wl.make_workload(0, scale=0.25)
    g = oracle.grid_from_bbox(w.posm, w.n_gas, w.h)
    f32 = np.float32
    cell = f32(f32(2) * f32(w.h)) * f32(1 + 2.0 ** -9)
    assert f32(g.cell) == cell and f32(g.inv_cell) == f32(1) / cell
    gas = w.posm[: w.n_gas, :3]
    assert np.array_equal(np.array(g.origin, dtype=f32), gas.min(0))
    dims = ((gas.max(0) - gas.min(0)) * f32(g.inv_cell)).astype(np.int32) + 1
    assert tuple(dims) == tuple(g.dims)
    key = oracle.cell_keys(w.posm, w.n_gas, g)
    c = np.floor((gas - gas.min(0)) * f32(g.inv_cell))
    c = np.minimum(np.maximum(c, 0), np.array(g.dims, dtype=f32) - 1).astype(np.int64)
    assert np.array_equal(key, (c[:, 0] + g.dims[0] * (c[:, 1] + g.dims[1] * c[:, 2])).astype(np.uint32))
    assert key.max() < g.M
    # particles outside the descriptor's box are clamped into the boundary cells
    small = oracle.Grid(g.origin, g.cell, g.inv_cell, (3, 2, 1))
    k2 = oracle.cell_keys(w.posm, w.n_gas, small)
    assert k2.max() < 6
    far = np.array([[1e30, -1e30, 0, 1]], dtype=np.float32)
    assert oracle.cell_keys(far, 1, small)[0] == 2 + 3 * 0


@pytest.mark.parametrize("case", ["galaxy", "dense", "clamped", "one_cell", "duplicates"])
def test_P1_grid_sets_equal_brute_force(case):
    if case == "galaxy":
        w = wl.make_workload(0, scale=0.5)
        posm, n, h, grid = w.posm, w.n_gas, w.h, None
    elif case == "dense":
        posm, _, h = _dense_gas(n=3000, h=0.06)
        n, grid = 3000, None
    elif case == "clamped":
        # descriptor covers only the core: the outskirts are clamped into boundary cells
        w = wl.make_workload(0, scale=0.5)
        posm, n, h = w.posm, w.n_gas, w.h
        g = oracle.grid_from_bbox(posm, n, h)
        grid = oracle.Grid((-1.0, -1.0, -1.0), g.cell, g.inv_cell, (5, 4, 6))
    elif case == "one_cell":
        posm, _, _ = _dense_gas(n=600)
        n, h, grid = 600, 5.0, None                   # 2h >> box: M = 1, everybody neighbours everybody
    else:
        posm, _, h = _dense_gas(n=500, h=0.1)
        posm[250:] = posm[:250]                       # exact duplicates
        n, grid = 500, None
    ob, ib = oracle.neighbours(posm, n, h, method="brute")
    og, ig = oracle.neighbours(posm, n, h, method="grid", grid=grid)
    assert np.array_equal(ob, og) and np.array_equal(ib, ig)
    if case == "one_cell":
        assert np.all(np.diff(ob) == n - 1)
    if case == "duplicates":
        assert all(250 + i in ib[ob[i]:ob[i + 1]] for i in range(250))
    # symmetry of the predicate: j in N(i) <=> i in N(j)
    pairs = set()
    for i in range(n):
        for j in ib[ob[i]:ob[i + 1]]:
            pairs.add((i, int(j)))
    assert all((j, i) in pairs for (i, j) in pairs)
    # the FP32 predicate itself, re-evaluated in numpy float32 for a few particles
    p = posm[:n, :3].astype(np.float32)
    rc2 = np.float32(np.float32(2) * np.float32(h)) ** 2
    assert np.float32(rc2) == oracle.rc2(h)
    for i in [0, n // 3, n - 1]:
        d = p[i] - p
        xx = (d[:, 0] * d[:, 0]).astype(np.float32)
        s = (d[:, 1].astype(np.float64) * d[:, 1].astype(np.float64) + xx.astype(np.float64)).astype(np.float32)  # fma
        d2 = (d[:, 2].astype(np.float64) * d[:, 2].astype(np.float64) + s.astype(np.float64)).astype(np.float32)  # fma
        want = np.flatnonzero((d2 < rc2) & (np.arange(n) != i))
        assert np.array_equal(want, ib[ob[i]:ob[i + 1]])


# ---------------------------------------------------------------- P8: collisionless reduction = velocity Verlet
def _verlet(pos, vel, m, G, delta, dt, steps):
    def acc(p):
        d = p[:, None, :] - p[None, :, :]
        r2 = (d ** 2).sum(-1) + delta ** 2
        np.fill_diagonal(r2, np.inf)
        return -G * (m[None, :, None] * d / r2[..., None] ** 1.5).sum(1)
    a = acc(pos)
    for _ in range(steps):
        pos = pos + dt * vel + 0.5 * dt * dt * a
        a1 = acc(pos)
        vel = vel + 0.5 * dt * (a + a1)
        a = a1
    return pos, vel


def test_P8_collisionless_is_velocity_verlet():
    rng = np.random.Generator(np.random.Philox(key=[11, 0]))
    n, G, delta, dt = 40, 1.0, 0.05, 1e-2
    posm = np.zeros((n, 4))
    vele = np.zeros((n, 4))
    posm[:, :3] = rng.standard_normal((n, 3))
    posm[:, 3] = (0.5 + rng.random(n)) / n
    vele[:, :3] = 0.3 * rng.standard_normal((n, 3))
    st = oracle.State(posm.copy(), vele.copy(), 0)
    oracle.position_only(st, 0.1, G, delta)
    for _ in range(7):
        st, _, _ = oracle.step(st, dt, 0.1, G, delta)
    p, v = _verlet(posm[:, :3], vele[:, :3], posm[:, 3], G, delta, dt, 7)
    assert np.allclose(st.posm[:, :3], p, rtol=0, atol=1e-13)
    assert np.allclose(st.vele[:, :3], v, rtol=0, atol=1e-13)


def test_P8_circular_orbit_second_order():
    # two equal masses on a circular orbit; phase error after one period shrinks ~4x when dt halves
    G, m, d = 1.0, 0.5, 1.0
    v = math.sqrt(G * m / (2 * d))          # each body: v^2/(d/2) = G m / d^2
    period = 2 * PI * (d / 2) / v

    def run(nsteps):
        posm = np.array([[-d / 2, 0, 0, m], [d / 2, 0, 0, m]])
        vele = np.array([[0, -v, 0, 0], [0, v, 0, 0.0]])
        st = oracle.State(posm, vele, 0)
        oracle.position_only(st, 0.1, G, 0.0)
        for _ in range(nsteps):
            st, _, _ = oracle.step(st, period / nsteps, 0.1, G, 0.0)
        return np.linalg.norm(st.posm[1, :3] - np.array([d / 2, 0, 0]))
    e1, e2 = run(200), run(400)
    assert e1 < 2e-2 and 3.5 < e1 / e2 < 4.5


# ---------------------------------------------------------------- P7: energy and momentum over steps
def test_P7_energy_drift_config0():
    w = wl.make_workload(0)
    m = w.posm[:, 3].astype(np.float64)

    def run(dt, steps):
        st = oracle.State(w.posm.astype(np.float64), w.vele.astype(np.float64), w.n_gas)
        nbr = oracle.position_only(st, w.h, w.G, w.delta)
        e0 = oracle.total_energy(st, w.G, w.delta)
        p0 = (m[:, None] * st.vele[:, :3]).sum(0)
        for _ in range(steps):
            st, nbr, _ = oracle.step(st, dt, w.h, w.G, w.delta, nbr=nbr)
        e1 = oracle.total_energy(st, w.G, w.delta)
        p1 = (m[:, None] * st.vele[:, :3]).sum(0)
        return abs((e1 - e0) / e0), np.linalg.norm(p1 - p0)
    drift, dp = run(1e-3, 10)
    assert drift <= 1e-7                    # stated bound: oracle, 10 steps, config 0
    assert dp <= 1e-15
    # halving dt at fixed end time shrinks the drift by >= 4x (third-order local energy error)
    d_big, _ = run(2e-3, 5)
    assert d_big >= 4 * drift * 0.9


# ---------------------------------------------------------------- NEXT-1: modified CFL step, Eq. 17 (L125-129)
def _golden(name):
    import os
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")):
        f = line.split()
        if f and f[0] == name:
            return f[1]
    raise KeyError(name)


def test_CFL_two_particles_by_hand():
    """Worked example (tests/golden/closed_forms.txt: cfl_two_particles), every factor a round number."""
    h = 1.0
    posm = np.array([[0, 0, 0, 1.0], [1, 0, 0, 1.0]], dtype=np.float64)
    vele = np.array([[0.5, 0, 0, 0.9], [-0.5, 0, 0, 0.9]], dtype=np.float64)    # closing speed 1, c = 1
    off, idx = oracle.neighbours(posm, 2, h)
    rho = oracle.density(posm, h, off, idx)
    acc_sph = np.array([[3.0, 0, 0, 1.0], [0, 2.0, 0, -1.0]])                    # |Q| = 3 (with a_grav below), |E| = 1
    acc_grav = np.array([[0.0, 0, 0, 0], [0, 1.0, 0, 0]])
    dt, br = oracle.cfl_dt(posm, vele, rho, acc_sph, acc_grav, h, off, idx, 0.5)
    num, den = _golden("cfl_two_particles").split("/")
    expect = float(Fraction(num) / Fraction(den))
    assert abs(expect - 0.5 / (3.6 + 12.0 / 11.0)) < 1e-15
    assert np.isclose(dt, expect, rtol=1e-14)
    assert np.allclose(br, 2 * expect, rtol=1e-14)                               # symmetric pair: same bracket
    # receding pair: mu = 0 (L97), the viscous term drops out
    vele[:, 0] *= -1
    dt2, _ = oracle.cfl_dt(posm, vele, rho, acc_sph, acc_grav, h, off, idx, 0.5)
    assert np.isclose(dt2, 0.5 / (1.6 + 2.0), rtol=1e-14)


def test_CFL_static_lattice_reduces_to_courant():
    """Uniform lattice at rest, no forces: Eq. 17 collapses to the textbook Courant condition
    dt = C a / (c (1 + 1.2 alpha)) with a the lattice spacing and c = sqrt(gamma (gamma-1) e)."""
    a, h, e, gamma, alpha = 0.25, 0.3, 0.7, 1.4, 0.5
    g = np.arange(5) * a
    x, y, z = np.meshgrid(g, g, g, indexing="ij")
    n = x.size
    posm = np.stack([x.ravel(), y.ravel(), z.ravel(), np.full(n, a ** 3)], 1)
    vele = np.zeros((n, 4))
    vele[:, :3] = (0.3, -0.2, 0.1)                  # uniform motion: Galilean invariance, all dv = 0
    vele[:, 3] = e
    off, idx = oracle.neighbours(posm, n, h)
    rho = oracle.density(posm, h, off, idx)
    zero = np.zeros((n, 4))
    dt, br = oracle.cfl_dt(posm, vele, rho, zero, zero, h, off, idx, 0.8, gamma=gamma, alpha=alpha)
    c = math.sqrt(gamma * (gamma - 1) * e)
    assert np.allclose(br, a / (c * (1 + 1.2 * alpha)), rtol=1e-12)
    assert np.isclose(dt, 0.8 * a / (c * (1 + 1.2 * alpha)), rtol=1e-12)


def test_CFL_isolated_particle_and_monotonicity():
    """A22: a particle with no neighbour takes s = 2h; a larger |Q| can only shrink the step; dt is
    the minimum of the per-particle brackets."""
    h, gamma = 0.1, 5.0 / 3.0
    posm = np.array([[0, 0, 0, 1.0], [5, 5, 5, 1.0], [5.05, 5, 5, 1.0]], dtype=np.float64)
    vele = np.array([[0, 0, 0, 0.9], [0, 0, 0, 0.9], [0, 0, 0, 0.9]], dtype=np.float64)
    off, idx = oracle.neighbours(posm, 3, h)
    assert np.diff(off).tolist() == [0, 1, 1]
    rho = oracle.density(posm, h, off, idx)
    zero = np.zeros((3, 4))
    dt, br = oracle.cfl_dt(posm, vele, rho, zero, zero, h, off, idx, 1.0, gamma=gamma, alpha=0.5)
    assert np.isclose(br[0], 2 * h / 1.6, rtol=1e-14)           # c = 1
    assert np.isclose(br[1], 0.05 / 1.6, rtol=1e-12) and np.isclose(dt, br.min())
    acc = zero.copy()
    acc[:, 0] = 10.0
    dt2, br2 = oracle.cfl_dt(posm, vele, rho, acc, zero, h, off, idx, 1.0, gamma=gamma, alpha=0.5)
    assert np.all(br2 < br) and dt2 < dt
    assert np.isclose(br2[0], 2 * h / (1.6 + math.sqrt(2 * h * 10.0)), rtol=1e-14)


def test_CFL_pair_lengths_by_hand():
    """Eq. 17 with per-particle smoothing lengths (L82): mu_ij takes h_ij = (h_1 + h_2)/2.  The hand-worked pair of
    cfl_two_particles with h_1 = 0.75, h_2 = 1.25 (h_ij = 1) gives the same bracket as the global h = 1; with h_1 = h_2 = 2
    |mu| = 2/(1 + 0.4) = 10/7: bracket 1/(1.6 + 1.2*10/7 + 2).  A particle without a neighbour takes s = 2 h_i (A22)."""
    posm = np.array([[0, 0, 0, 1.0], [1, 0, 0, 1.0], [50, 0, 0, 1.0]], dtype=np.float64)
    vele = np.array([[0.5, 0, 0, 0.9], [-0.5, 0, 0, 0.9], [0, 0, 0, 0.9]], dtype=np.float64)
    acc_sph = np.array([[3.0, 0, 0, 1.0], [0, 2.0, 0, -1.0], [0, 0, 0, 0.0]])
    acc_grav = np.array([[0.0, 0, 0, 0], [0, 1.0, 0, 0], [0, 0, 0, 0]])
    num, den = _golden("cfl_two_particles").split("/")
    expect = float(Fraction(num) / Fraction(den)) / 0.5                          # the bracket itself
    for hs, want in (([0.75, 1.25, 0.25], expect), ([2.0, 2.0, 0.25], 1.0 / (1.6 + 12.0 / 7.0 + 2.0))):   # exact in FP32
        hs = np.array(hs)
        off, idx = oracle.neighbours(posm, 3, 2.0, hs=hs)
        assert np.diff(off).tolist() == [1, 1, 0]
        rho = oracle.density(posm, 2.0, off, idx, hs=hs)
        dt, br = oracle.cfl_dt(posm, vele, rho, acc_sph, acc_grav, 2.0, off, idx, 1.0, hs=hs)
        assert np.allclose(br[:2], want, rtol=1e-14, atol=0)
        assert np.isclose(br[2], 2 * 0.25 / 1.6, rtol=1e-14, atol=0)             # isolated: s = 2 h_i, c = 1, alpha = 0.5
        assert np.isclose(dt, br.min())
    # equal lengths reduce to the global-h result
    off, idx = oracle.neighbours(posm, 3, 1.0)
    rho = oracle.density(posm, 1.0, off, idx)
    _, br_g = oracle.cfl_dt(posm, vele, rho, acc_sph, acc_grav, 1.0, off, idx, 1.0)
    _, br_h = oracle.cfl_dt(posm, vele, rho, acc_sph, acc_grav, 1.0, off, idx, 1.0, hs=np.ones(3))
    assert np.array_equal(br_g, br_h)


def test_CFL_adaptive_step():
    """oracle.step(c_cfl=): the step taken is min(dt, C_CFL min_i bracket_i) with the bracket of Eq. 17 at the time layer
    the step starts from.  (1) a large ceiling: the step equals C_CFL times the minimum of cfl_dt called by hand on the
    same state; (2) a ceiling below the CFL value: bit for bit the fixed-step result; (3) energy (pin P7): 10 adaptive
    steps at config 0, C_CFL = 0.5, stay inside the drift bound of the fixed-step run over the same time."""
    w = wl.make_workload(0, scale=0.25)
    st0 = oracle.State(w.posm.astype(np.float64), w.vele.astype(np.float64), w.n_gas)
    nbr = oracle.position_only(st0, w.h, w.G, w.delta)
    hy = oracle.hydro(st0, w.h, nbr)
    dt_hand, br = oracle.cfl_dt(st0.posm, st0.vele, st0.rho, hy, st0.acc_grav[: w.n_gas], w.h, nbr[0], nbr[1], 0.5)
    s1, _, d1 = oracle.step(st0, 1.0, w.h, w.G, w.delta, nbr=nbr, c_cfl=0.5)
    assert d1["dt"] == dt_hand and dt_hand == 0.5 * br.min() and 0 < dt_hand < 1.0
    tiny = 0.1 * dt_hand
    s2, _, d2 = oracle.step(st0, tiny, w.h, w.G, w.delta, nbr=nbr, c_cfl=0.5)
    s3, _, _ = oracle.step(st0, tiny, w.h, w.G, w.delta, nbr=nbr)
    assert d2["dt"] == tiny and np.array_equal(s2.posm, s3.posm) and np.array_equal(s2.vele, s3.vele)
    # energy over 10 adaptive steps
    e0 = oracle.total_energy(st0, w.G, w.delta)
    st, nb, t = st0, nbr, 0.0
    for _ in range(10):
        st, nb, d = oracle.step(st, 1.0, w.h, w.G, w.delta, nbr=nb, c_cfl=0.5)
        t += d["dt"]
    drift = abs(oracle.total_energy(st, w.G, w.delta) - e0) / abs(e0)
    assert t > 0 and drift < 1e-7 * max(1.0, t / 0.01), (drift, t)


# ---------------------------------------------------------------- NEXT-2: per-particle smoothing lengths (L82)
def _varh_case(n=1500, seed=11, h_max=0.08):
    rng = np.random.Generator(np.random.Philox(key=[seed, 0]))
    posm = np.zeros((n, 4), np.float32)
    vele = np.zeros((n, 4), np.float32)
    posm[:, :3] = rng.random((n, 3)) * 0.6
    posm[:, 3] = (0.5 + rng.random(n)) / n
    vele[:, :3] = 0.5 * rng.standard_normal((n, 3))
    vele[:, 3] = 0.5 + 0.5 * rng.random(n)
    hs = (h_max * (0.45 + 0.55 * rng.random(n))).astype(np.float32)
    return posm, vele, hs


def test_VARH_equal_lengths_reduce_to_global_h():
    """h_i = h for all i: h_ij = h, so sets, density and forces must equal the (pinned) global-h results."""
    posm, vele, _ = _varh_case()
    n, h = len(posm), np.float32(0.06)
    hs = np.full(n, h, np.float32)
    o0, i0 = oracle.neighbours(posm, n, h)
    o1, i1 = oracle.neighbours(posm, n, h, hs=hs)
    assert np.array_equal(o0, o1) and np.array_equal(i0, i1)
    r0 = oracle.density(posm, h, o0, i0)
    r1 = oracle.density(posm, h, o1, i1, hs=hs)
    assert np.allclose(r0, r1, rtol=1e-14)
    f0 = oracle.forces(posm, vele, r0, h, o0, i0)
    f1 = oracle.forces(posm, vele, r0, h, o1, i1, hs=hs)
    assert np.allclose(f0, f1, rtol=1e-12, atol=1e-14 * np.abs(f0).max())


def test_VARH_grid_sets_equal_brute_force_and_are_symmetric():
    posm, _, hs = _varh_case()
    n, h_max = len(posm), 0.08
    ob, ib = oracle.neighbours(posm, n, h_max, hs=hs, method="brute")
    og, ig = oracle.neighbours(posm, n, h_max, hs=hs, method="grid")
    assert np.array_equal(ob, og) and np.array_equal(ib, ig)
    pairs = set()
    for i in range(n):
        for j in ib[ob[i]:ob[i + 1]]:
            pairs.add((i, int(j)))
    assert all((j, i) in pairs for (i, j) in pairs)               # h_ij is symmetric, so is the relation
    # the cutoff really is h_i + h_j: every listed pair is inside it, and some pair is outside 2 min(h_i, h_j)
    d = np.array([np.linalg.norm(posm[i, :3].astype(np.float64) - posm[j, :3]) for (i, j) in pairs])
    lim = np.array([float(hs[i]) + float(hs[j]) for (i, j) in pairs])
    small = np.array([2.0 * min(float(hs[i]), float(hs[j])) for (i, j) in pairs])
    assert np.all(d < lim * (1 + 1e-6)) and np.any(d > small)


def test_VARH_momentum_and_energy_identity():
    """h_ij symmetric => Pi_ij symmetric and grad W_p antisymmetric as before: P5 and P6 must still hold."""
    posm, vele, hs = _varh_case()
    n, h_max = len(posm), 0.08
    off, idx = oracle.neighbours(posm, n, h_max, hs=hs)
    rho = oracle.density(posm, h_max, off, idx, hs=hs)
    f = oracle.forces(posm, vele, rho, h_max, off, idx, hs=hs)
    m = posm[:, 3].astype(np.float64)
    v = vele[:, :3].astype(np.float64)
    scale = (m * np.linalg.norm(f[:, :3], axis=1)).sum()
    assert np.linalg.norm((m[:, None] * f[:, :3]).sum(0)) < 1e-13 * scale
    resid = (m * f[:, 3]).sum() + (m * (v * f[:, :3]).sum(1)).sum()
    assert abs(resid) < 1e-13 * ((m * np.abs(f[:, 3])).sum() + (m * np.abs((v * f[:, :3]).sum(1))).sum())


def test_VARH_single_pair_by_hand():
    gamma, alpha, beta, eta = 1.4, 0.5, 1.0, 0.1
    h1, h2, d = 0.5, 0.3, 0.6                    # h_12 = 0.4, xi = 1.5 (outer branch); 2 h_12 = 0.8 > d
    m1, m2, e1, e2 = 0.3, 0.7, 1.2, 0.8
    posm = np.array([[0, 0, 0, m1], [d, 0, 0, m2]], dtype=np.float64)
    vele = np.array([[0.4, 0.1, 0, e1], [-0.2, 0.0, 0, e2]], dtype=np.float64)
    hs = np.array([h1, h2], dtype=np.float32)
    h1, h2 = float(hs[0]), float(hs[1])          # the FP32 values both sides carry
    h12 = 0.5 * (h1 + h2)
    off, idx = oracle.neighbours(posm, 2, 0.5, hs=hs)
    assert off.tolist() == [0, 1, 2]
    rho = oracle.density(posm, 0.5, off, idx, hs=hs)
    xi = d / h12
    w12 = 0.25 * (2 - xi) ** 3 / (PI * h12 ** 3)
    assert np.allclose(rho, [m1 / (PI * h1 ** 3) + m2 * w12, m2 / (PI * h2 ** 3) + m1 * w12], rtol=1e-14)
    f = oracle.forces(posm, vele, rho, 0.5, off, idx, gamma=gamma, alpha=alpha, beta=beta, eta=eta, hs=hs)
    p1, p2 = (gamma - 1) * rho[0] * e1, (gamma - 1) * rho[1] * e2
    c1, c2 = math.sqrt(gamma * p1 / rho[0]), math.sqrt(gamma * p2 / rho[1])
    dr, dv = np.array([-d, 0, 0]), np.array([0.6, 0.1, 0])
    mu = h12 * (dr @ dv) / (d * d + eta * h12 * h12)
    nu = mu * (beta * mu - alpha * 0.5 * (c1 + c2)) / (0.5 * (rho[0] + rho[1]))
    Pi = p1 / rho[0] ** 2 + p2 / rho[1] ** 2 + nu
    gradWp = (-45 / (64 * PI * h12 ** 3) * (2 - xi) ** 2) * (dr / d) / h12
    assert np.allclose(f[0, :3], -m2 * Pi * gradWp, rtol=1e-13)
    assert np.isclose(f[1, 3], 0.5 * m1 * Pi * (dv @ gradWp), rtol=1e-13)
    # farther apart than h_1 + h_2 = 0.8 but closer than 2 h_1 = 1.0: not neighbours (the pair length decides)
    posm[1, 0] = 0.9
    off, _ = oracle.neighbours(posm, 2, 0.5, hs=hs)
    assert off.tolist() == [0, 0, 0]


def test_VARH_smoothing_lengths_on_lattice():
    """L82 on a uniform lattice with m = rho0 a^3: (m/rho)^(1/3) = a (rho0/rho)^(1/3); capped at h_max (A25)."""
    w = wl.lattice(7, 0.1, rho0=2.0)
    n = w.n_gas
    off, idx = oracle.neighbours(w.posm, n, 0.1)
    rho = oracle.density(w.posm, 0.1, off, idx)
    hs = oracle.smoothing_lengths(w.posm, rho, 1.3, 1.0)
    assert hs.dtype == np.float32
    assert np.allclose(hs, 1.3 * 0.1 * np.cbrt(2.0 / rho), rtol=2e-7)
    centre = n // 2
    assert abs(hs[centre] / (1.3 * 0.1) - 1) < 1e-4              # interior rho = 0.99997 rho0 (pin P3)
    assert np.all(oracle.smoothing_lengths(w.posm, rho, 1.3, 0.12) <= np.float32(0.12))
