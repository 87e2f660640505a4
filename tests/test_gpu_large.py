"""Large-N protocol: BASELINE.json's full-size configs in the launch configuration
bench.py times.  O(N) structures (keys, perm, ranges) and the O(N) update formulas are checked
on ALL particles; gravity and the SPH sums on a seeded 4096-particle subset (2048 gas + 2048
halo, plus forced members), stage by stage (teacher-forced: each stage's oracle input is the
GPU's verified output of the previous stage)."""
import numpy as np
import pytest

import oracle
from paper_1807_08116_b200 import workloads as wl
from parity_util import check_density, check_values

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _subset(w, key, count):
    g_idx, h_idx = wl.subset_indices(w.n_gas, w.n_halo, w.seed, n_each=2048)
    forced = []
    if w.n_gas:
        gas = w.posm[: w.n_gas, :3]
        forced += [int(gas[:, a].argmin()) for a in range(3)] + [int(gas[:, a].argmax()) for a in range(3)]
        forced.append(int(np.flatnonzero(key == np.argmax(count))[0]))      # a particle of the fullest cell
    g_idx = np.unique(np.concatenate([g_idx, np.array(forced, dtype=np.int64)])) if w.n_gas else g_idx
    return g_idx.astype(np.int64), h_idx.astype(np.int64)


def _check_structures(b, sim, w):
    """keys / perm / start inside the workspace against the oracle's sequential counting sort: ALL particles."""
    ng = w.n_gas
    og = oracle.grid_from_bbox(w.posm, ng, w.h)
    assert tuple(og.dims) == tuple(sim.grid.dims)
    d = sim.posm
    M = sim.grid.M
    key = torch.zeros(ng, dtype=torch.int32, device="cuda")
    perm = torch.zeros(ng, dtype=torch.int32, device="cuda")
    count = torch.zeros(M, dtype=torch.int32, device="cuda")
    start = torch.zeros(M + 1, dtype=torch.int32, device="cuda")
    b.sph_build_grid(d, ng, sim.grid, key, perm, count, start, sim.ws)
    okey = oracle.cell_keys(w.posm, ng, og)
    ocount, ostart, operm = oracle.counting_sort(okey, M)
    assert np.array_equal(key.cpu().numpy().view(np.uint32), okey)
    assert np.array_equal(start.cpu().numpy().view(np.uint32), ostart)
    assert np.array_equal(perm.cpu().numpy().view(np.uint32), operm)
    assert np.array_equal(count.cpu().numpy().view(np.uint32), ocount)
    return og, okey, ocount, ostart, operm


def _check_sph_subset(w, posm, vele, rho_gpu, acc_sph_gpu, g_idx, og, sort, density=True):
    """density for the subset, forces for the subset with the GPU's verified rho as input."""
    off, idx = oracle.neighbours(posm, w.n_gas, w.h, targets=g_idx, method="grid", grid=og, sort=sort)
    if density:
        orho = oracle.density(posm, w.h, off, idx, targets=g_idx)
        check_density(rho_gpu[g_idx], orho, "rho subset")
    # every neighbour's density is also checked (two-hop closure): a wrong rho_j would otherwise hide
    closure = np.unique(idx.astype(np.int64))
    if density and len(closure):
        off2, idx2 = oracle.neighbours(posm, w.n_gas, w.h, targets=closure, method="grid", grid=og, sort=sort)
        check_density(rho_gpu[closure], oracle.density(posm, w.h, off2, idx2, targets=closure), "rho closure")
    of, gross = oracle.forces(posm, vele, rho_gpu.astype(np.float64), w.h, off, idx, targets=g_idx, gamma=w.gamma,
                              alpha=w.alpha, beta=w.beta, eta=w.eta, with_gross=True)
    check_values(acc_sph_gpu[g_idx, :3], of[:, :3], "a_sph subset", gross=gross[:, 0])
    check_values(acc_sph_gpu[g_idx, 3], of[:, 3], "de/dt subset", gross=gross[:, 1])
    return np.diff(off)


def _staged_step_checked(b, sim, w, og, g_idx, h_idx, check_sort):
    """One step of sph_step_h, issued as the three stage calls it is composed of (sph_predict, sph_position_slice,
    sph_correct: the same code path, bit for bit), with every stage checked TEACHER-FORCED (SURVEY §8(c) large-N
    protocol): the oracle's input at each stage is the GPU's verified output of the stage before, so it never advances
    10^6 particles by O(N^2) itself.  O(N) update formulas on ALL particles, sums on the seeded subset."""
    ng, n, nh, dt = w.n_gas, w.n_total, w.n_halo, w.dt
    tg = np.concatenate([g_idx, h_idx])
    p0 = sim.posm.cpu().numpy()
    v0f = sim.vele.cpu().numpy()
    rho0 = sim.rho.cpu().numpy()
    ag0 = sim.acc_grav.cpu().numpy().astype(np.float64)
    # ---- HFC(predictor) + SU(predictor)
    b.sph_predict(sim.posm, sim.vele, None, ng, nh, sim.params, sim.grid, dt, sim.rho, sim.acc_sph, sim.acc_grav, sim.ws)
    as0 = sim.acc_sph.cpu().numpy()
    key0 = oracle.cell_keys(p0, ng, og)
    _, start0, perm0 = oracle.counting_sort(key0, og.M)
    _check_sph_subset(w, p0, v0f, rho0, as0, g_idx, og, (key0, start0, perm0), density=False)
    p1 = sim.posm.cpu().numpy()
    vt_g = sim.vele.cpu().numpy()
    Q0 = ag0[:, :3].copy()
    Q0[:ng] += as0[:, :3]
    v0 = v0f[:, :3].astype(np.float64)
    e0 = v0f[:ng, 3].astype(np.float64)
    vt = v0 + dt * Q0                                                # Eq. 12
    et = e0 + dt * as0[:, 3].astype(np.float64)                      # Eq. 13
    r1 = p0[:, :3].astype(np.float64) + 0.5 * dt * (vt + v0)         # Eq. 14
    check_values(vt_g[:, :3], vt, "v~ (Eq. 12) all", max_tol=2e-6, med_tol=2e-7)
    check_values(vt_g[:ng, 3], et, "e~ (Eq. 13) all", max_tol=2e-6, med_tol=2e-7)
    assert np.abs(p1[:, :3] - r1).max() <= 2e-7 * max(1.0, np.abs(r1).max())       # Eq. 14: one FP32 rounding of r
    assert np.array_equal(p1[:, 3], p0[:, 3])
    # ---- SP, DC, GFC at r(t+dt)
    b.sph_position_slice(sim.posm, None, 0.0, ng, nh, 0, n, sim.params, sim.grid, sim.rho, sim.acc_grav, sim.ws)
    ag1 = sim.acc_grav.cpu().numpy().astype(np.float64)
    check_values(ag1[tg, :3], oracle.gravity(p1, w.G, w.delta, targets=tg), "a_grav(t+dt) subset")
    assert np.all(ag1[:, 3] == 0)
    key1 = oracle.cell_keys(p1, ng, og)
    _, start1, perm1 = oracle.counting_sort(key1, og.M)
    if check_sort:                                                   # the grid the library carries, ALL particles
        key = torch.zeros(ng, dtype=torch.int32, device="cuda")
        perm = torch.zeros(ng, dtype=torch.int32, device="cuda")
        count = torch.zeros(og.M, dtype=torch.int32, device="cuda")
        start = torch.zeros(og.M + 1, dtype=torch.int32, device="cuda")
        ws2 = b.alloc_workspace(ng, ng, sim.grid)
        b.sph_build_grid(sim.posm, ng, sim.grid, key, perm, count, start, ws2)
        assert np.array_equal(key.cpu().numpy().view(np.uint32), key1)
        assert np.array_equal(start.cpu().numpy().view(np.uint32), start1)
        assert np.array_equal(perm.cpu().numpy().view(np.uint32), perm1)
        del key, perm, count, start, ws2
    rho1 = sim.rho.cpu().numpy()
    # ---- HFC(corrector) + SU(corrector)
    b.sph_correct(sim.vele, None, ng, nh, sim.params, sim.grid, dt, sim.rho, sim.acc_sph, sim.acc_grav, sim.ws)
    as1 = sim.acc_sph.cpu().numpy()
    _check_sph_subset(w, p1, vt_g, rho1, as1, g_idx, og, (key1, start1, perm1))
    v1 = sim.vele.cpu().numpy()
    Q1 = ag1[:, :3].copy()
    Q1[:ng] += as1[:, :3]
    vt64 = vt_g[:, :3].astype(np.float64)
    check_values(v1[:, :3], 0.5 * (v0 + vt64) + 0.5 * dt * Q1, "v(t+dt) (Eq. 15) all", max_tol=2e-6, med_tol=2e-7)
    check_values(v1[:ng, 3], 0.5 * (e0 + vt_g[:ng, 3]) + 0.5 * dt * as1[:, 3], "e(t+dt) (Eq. 16) all", max_tol=2e-6,
                 med_tol=2e-7)


@pytest.mark.parametrize("cfg", [2, 3])
def test_full_size_collision(cuda_lib, cfg):
    """BASELINE.json configs 2 and 3 at their stated size AND step count (10 and 5 steps), every stage of every step
    against the oracle, teacher-forced."""
    b = cuda_lib
    w = wl.make_workload(cfg)
    ng, n = w.n_gas, w.n_total
    sim = b.Simulation(w)
    og, okey, ocount, ostart, operm = _check_structures(b, sim, w)
    g_idx, h_idx = _subset(w, okey, ocount)
    tg = np.concatenate([g_idx, h_idx])
    # ---- force evaluation at t = 0 (seeds the carried state)
    sim.evaluate()
    rho0 = sim.rho.cpu().numpy()
    as0 = sim.acc_sph.cpu().numpy()
    ag0 = sim.acc_grav.cpu().numpy()
    check_values(ag0[tg, :3], oracle.gravity(w.posm, w.G, w.delta, targets=tg), f"a_grav cfg{cfg} subset")
    assert np.all(ag0[:, 3] == 0)
    nn = _check_sph_subset(w, w.posm, w.vele, rho0, as0, g_idx, og, (okey, ostart, operm))
    assert nn.max() > 10
    # ---- the config's steps, staged.  At config 2 a plain sph_step replica runs beside them and must stay bit-identical
    # (at config 3 that would double 20 s of gravity; the identity is also tested at N = 98304).
    ref = b.Simulation(w, grid=sim.grid) if cfg == 2 else None
    for k in range(w.steps):
        _staged_step_checked(b, sim, w, og, g_idx, h_idx, check_sort=(cfg == 2 or k == w.steps - 1))
        if ref is not None:
            ref.step()
    if ref is not None:
        for x, y in ((sim.posm, ref.posm), (sim.vele, ref.vele), (sim.rho, ref.rho), (sim.acc_sph, ref.acc_sph),
                     (sim.acc_grav, ref.acc_grav)):
            assert torch.equal(x, y)


def test_full_size_sph_only_config4(cuda_lib):
    """config 4: N_g = 2^24 gas, no gravity — grid sort on all particles, density / forces on the subset."""
    b = cuda_lib
    w = wl.make_workload(4)
    sim = b.Simulation(w)
    og, okey, ocount, ostart, operm = _check_structures(b, sim, w)
    g_idx, _ = _subset(w, okey, ocount)
    sim.evaluate()
    assert torch.count_nonzero(sim.acc_grav).item() == 0
    nn = _check_sph_subset(w, w.posm, w.vele, sim.rho.cpu().numpy(), sim.acc_sph.cpu().numpy(), g_idx, og,
                           (okey, ostart, operm))
    assert nn.max() > 500           # the clump cores


def test_full_size_sph_only_config4_varh(cuda_lib):
    """config 4 with per-particle smoothing lengths (NEXT-2, L82): seeded lengths in [0.3, 1] of the cap, spatially
    uncorrelated (the hardest case for the pair cutoff and for the largest-length-per-bin pruning of the dense-cell
    walks) — density and forces on the subset against the oracle's h_ij sums, the launch configuration bench.py
    --sigma times (dense-cell walks with VARH + thread-per-slot walks)."""
    b = cuda_lib
    w = wl.make_workload(4)
    ng = w.n_gas
    rng = np.random.Generator(np.random.Philox(key=[44, 9]))
    hs = (np.float32(w.h) * (0.3 + 0.7 * rng.random(ng))).astype(np.float32)
    sim = b.Simulation(w, sigma=0.0)                      # sigma = 0: the lengths are kept as given
    sim.hsml.copy_(torch.from_numpy(hs))
    og, okey, ocount, ostart, operm = _check_structures(b, sim, w)
    g_idx, _ = _subset(w, okey, ocount)
    sim.evaluate()
    assert b.sph_dense_items(sim.ws, ng, w.n_total, sim.grid) > 50000
    assert b.sph_workspace_status(sim.ws, ng, w.n_total, sim.grid) == 0
    sort = (okey, ostart, operm)
    off, idx = oracle.neighbours(w.posm, ng, w.h, targets=g_idx, method="grid", grid=og, sort=sort, hs=hs)
    rho_gpu = sim.rho.cpu().numpy()
    check_density(rho_gpu[g_idx], oracle.density(w.posm, w.h, off, idx, targets=g_idx, hs=hs), "rho subset varh")
    of, gross = oracle.forces(w.posm, w.vele, rho_gpu.astype(np.float64), w.h, off, idx, targets=g_idx, gamma=w.gamma,
                              alpha=w.alpha, beta=w.beta, eta=w.eta, with_gross=True, hs=hs)
    acc = sim.acc_sph.cpu().numpy()
    check_values(acc[g_idx, :3], of[:, :3], "a_sph subset varh", gross=gross[:, 0])
    check_values(acc[g_idx, 3], of[:, 3], "de/dt subset varh", gross=gross[:, 1])
    assert np.diff(off).max() > 100


def test_full_size_collisionless_next3(cuda_lib):
    """N_g = 0 (SP, DC, HFC skipped, L150) at N = 2^22.  One step: Eqs. 12-16 reduce to
    velocity Verlet (pin P8), checked on ALL particles from the GPU's own accelerations; the accelerations
    themselves on the seeded subset against the oracle, before and after the step."""
    b = cuda_lib
    w = wl.make_workload(5)
    assert w.n_gas == 0 and w.n_total == 2 ** 22
    _, h_idx = wl.subset_indices(0, w.n_halo, w.seed, n_each=2048)
    sim = b.Simulation(w)
    sim.evaluate()
    a0 = sim.acc_grav.cpu().numpy().astype(np.float64)[:, :3]
    check_values(a0[h_idx], oracle.gravity(w.posm, w.G, w.delta, targets=h_idx), "a_grav cfg5 subset")
    sim.first = True
    sim.step()
    p1 = sim.posm.cpu().numpy()
    v1 = sim.vele.cpu().numpy()
    a1 = sim.acc_grav.cpu().numpy().astype(np.float64)[:, :3]
    dt = w.dt
    r0 = w.posm[:, :3].astype(np.float64)
    v0 = w.vele[:, :3].astype(np.float64)
    r1 = r0 + dt * v0 + 0.5 * dt * dt * a0                               # velocity Verlet
    assert np.abs(p1[:, :3] - r1).max() <= 2e-6 * max(1.0, np.abs(r1).max())
    check_values(v1[:, :3], v0 + 0.5 * dt * (a0 + a1), "v(t+dt) cfg5 all", max_tol=2e-6, med_tol=2e-7)
    check_values(a1[h_idx], oracle.gravity(p1, w.G, w.delta, targets=h_idx), "a_grav(t+dt) cfg5 subset")


def test_full_size_collisionless_2p23(cuda_lib):
    """SURVEY §8(f) NEXT-3 at the top of the paper's range of N (L213): N = 2^23, N_g = 0.  One evaluation of Eq. 4 through
    the pair-symmetric path (3.5e13 unordered pairs), checked on the seeded subset against the oracle, plus momentum."""
    b = cuda_lib
    w = wl.make_workload(6)
    assert w.n_gas == 0 and w.n_total == 2 ** 23
    _, h_idx = wl.subset_indices(0, w.n_halo, w.seed, n_each=1024)
    sim = b.Simulation(w)
    sim.evaluate()
    assert b.sph_gravity_path(sim.ws, 0, w.n_total) == "pair_symmetric"
    a = sim.acc_grav.cpu().numpy().astype(np.float64)[:, :3]
    check_values(a[h_idx], oracle.gravity(w.posm, w.G, w.delta, targets=h_idx), "a_grav cfg6 (N = 2^23) subset")
    m = w.posm[:, 3].astype(np.float64)
    assert np.linalg.norm((m[:, None] * a).sum(0)) < 5e-7 * (m * np.linalg.norm(a, axis=1)).sum()
