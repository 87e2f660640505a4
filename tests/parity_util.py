"""Error measures used by the GPU parity tests (reading A17).

north_star: density to a relative 1e-5; accelerations and de/dt to 2e-4 of the per-particle
value (1e-5 median).  The per-particle value can be exactly 0 (a gas particle without
neighbours) or tiny by cancellation, so
    err_i = |a_i - ref_i| / max(|ref_i|, floor),   floor = 1e-3 * median of the non-zero |ref|,
with |.| the 2-norm for vectors, and exact zeros of the reference must be matched exactly.
"""
import numpy as np

RHO_TOL = 1e-5
VAL_TOL = 2e-4
MED_TOL = 1e-5


def rel_err(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    if got.ndim == 1:
        num, mag = np.abs(got - ref), np.abs(ref)
    else:
        num, mag = np.linalg.norm(got - ref, axis=1), np.linalg.norm(ref, axis=1)
    nz = mag[mag > 0]
    floor = 1e-3 * np.median(nz) if len(nz) else 1.0
    err = num / np.maximum(mag, floor)
    touched = int(np.count_nonzero((mag < floor) & (mag > 0)))
    return err, touched, mag == 0


def check_values(got, ref, what, max_tol=VAL_TOL, med_tol=MED_TOL):
    err, touched, zero = rel_err(got, ref)
    got = np.asarray(got, dtype=np.float64)
    gz = got[zero]
    assert np.all(gz == 0), f"{what}: reference zeros not matched exactly"
    nz = err[~zero]
    if len(nz) == 0:
        return 0.0, 0.0
    mx, med = float(nz.max()), float(np.median(nz))
    assert mx <= max_tol, f"{what}: max rel err {mx:.3e} > {max_tol} (floor touched {touched})"
    assert med <= med_tol, f"{what}: median rel err {med:.3e} > {med_tol}"
    return mx, med


def check_density(got, ref, what="rho"):
    got = np.asarray(got, dtype=np.float64)
    err = np.abs(got - ref) / ref
    assert err.max() <= RHO_TOL, f"{what}: max rel err {err.max():.3e} > {RHO_TOL}"
    return float(err.max())
