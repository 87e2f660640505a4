"""nbody_pp_gravity_static (include/sph_b200.h, csrc/noalloc.cu): Eq. 4 with the library's fixed device scratch instead of
a caller's workspace — no allocation inside the call.  Collected last (the name), so that a failure here hides no other test.
Checked against the existing path (nbody_pp_gravity with a workspace) on the same input — the same kernels, so bit for bit,
and a fortiori within the gravity tolerance of the parity tests (2e-4 max, 1e-5 median) — on two calls in a row, with
calls of other sizes in between (the scratch keeps the previous call's contents), and against the oracle on a subset."""
import numpy as np
import pytest

import oracle
from parity_util import check_values

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _particles(n, seed, equal_masses):
    rng = np.random.Generator(np.random.Philox(key=[seed, 3]))
    posm = np.zeros((n, 4), np.float32)
    posm[:, :3] = rng.standard_normal((n, 3)) * 0.5
    posm[:, 3] = 1.0 / n if equal_masses else (0.5 + rng.random(n)) / n
    return posm


def _existing(b, d, n, G, delta):
    ws = b.alloc_workspace(0, n, None)
    acc = torch.zeros((n, 4), device="cuda")
    b.nbody_pp_gravity(d, n, G, delta, acc, ws)
    return acc


# pair-symmetric path (N >= 32768, delta > 0), uniform and unequal masses; one-sided path (small N; delta = 0); the maximum size
@pytest.mark.parametrize("n,delta,equal", [(40000, 0.01, True), (33000, 0.02, False), (5000, 0.01, True), (3001, 0.0, False),
                                           (65536, 0.01, True)])
def test_static_scratch_gravity_matches_workspace_path(cuda_lib, n, delta, equal):
    b = cuda_lib
    assert b.nbody_pp_gravity_static_max() == 65536 and n <= b.nbody_pp_gravity_static_max()
    G = 1.0
    posm = _particles(n, 100 + n, equal)
    d = torch.from_numpy(posm).cuda()
    ref = _existing(b, d, n, G, delta)
    out1 = torch.full((n, 4), float("nan"), device="cuda")
    out2 = torch.full((n, 4), float("nan"), device="cuda")
    # calls of other sizes and paths in between: the scratch holds THEIR leftovers when the second call starts
    m = 36000 if n < 32768 else 2500
    dm = torch.from_numpy(_particles(m, 7, not equal)).cuda()
    outm = torch.zeros((m, 4), device="cuda")
    refm = _existing(b, dm, m, G, 0.03)
    b.nbody_pp_gravity_static(dm, m, G, 0.03, outm)                   # (also loads every kernel the calls below use)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    b.nbody_pp_gravity_static(d, n, G, delta, out1)                   # first call
    b.nbody_pp_gravity_static(dm, m, G, 0.03, outm)
    b.nbody_pp_gravity_static(d, n, G, delta, out2)                   # second call, right after another one
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0                                             # the driver handed out no device memory in between
    assert torch.equal(out1, ref) and torch.equal(out2, ref)          # same kernels, same order: the same bits
    assert torch.equal(outm, refm)
    got = out2.cpu().numpy().astype(np.float64)
    check_values(got[:, :3], ref.cpu().numpy().astype(np.float64)[:, :3], f"a_grav static vs workspace N={n}")
    # and against the oracle, on a seeded subset of targets
    tg = np.sort(np.random.Generator(np.random.Philox(key=[n, 5])).choice(n, size=256, replace=False)).astype(np.int64)
    want = oracle.gravity(posm, G, delta, targets=tg)
    check_values(got[tg, :3], want, f"a_grav static vs oracle N={n}", max_tol=5e-4 if delta == 0.0 else 2e-4,
                 med_tol=2e-5 if delta == 0.0 else 1e-5)


def test_static_scratch_gravity_rejects_what_does_not_fit(cuda_lib):
    b = cuda_lib
    nmax = b.nbody_pp_gravity_static_max()
    d = torch.zeros((nmax + 1, 4), device="cuda")
    acc = torch.zeros((nmax + 1, 4), device="cuda")
    with pytest.raises(b.SphError) as e:
        b.nbody_pp_gravity_static(d, nmax + 1, 1.0, 0.01, acc)
    assert e.value.rc == b.SPH_ERR_WORKSPACE
    with pytest.raises(b.SphError) as e:
        b.nbody_pp_gravity_static(d, 100, 1.0, -0.01, acc)
    assert e.value.rc == b.SPH_ERR_UNSUPPORTED
    with pytest.raises(b.SphError) as e:
        b.nbody_pp_gravity_static(None, 100, 1.0, 0.01, acc)
    assert e.value.rc == b.SPH_ERR_ARG
    b.nbody_pp_gravity_static(d, 0, 1.0, 0.01, acc)                   # n = 0 is legal
    # G = 0: Eq. 4 is identically zero
    acc.fill_(1.0)
    b.nbody_pp_gravity_static(d, 1000, 0.0, 0.01, acc)
    assert torch.count_nonzero(acc[:1000]).item() == 0 and torch.count_nonzero(acc[1000:]).item() == acc[1000:].numel()
