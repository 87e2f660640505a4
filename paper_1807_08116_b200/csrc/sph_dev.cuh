// sph_dev.cuh — device functions of the SPH walks (sph.cu: thread per sorted slot, the sparse galaxy grids;
// sph_dense.cu / sph_dense_rho.cu: CTA per populated cell, shared-memory staged).  The cutoff predicate (dist2_f32, A8)
// and the cell assignment (cell_of, A7) are the same operation sequence everywhere, so every walk sees the same
// neighbour set; the pair TERM has two forms — hydro_pair (sparse walk: few terms, all near the kernel edge, so FP64
// numerator and IEEE divisions) and hydro_pair_fast (dense walk: many terms, MUFU reciprocals) — and which one a
// particle's sum uses is decided by its cell's population alone (kDenseMin), so results stay reproducible.
// Internal to libsph_b200; nothing here is shared with the oracle.
#pragma once
#include "common.cuh"

namespace sphb {

// Cutoff predicate (A8), identical op sequence to the oracle:
//   dx = x_i (-) x_j ...  d2 = fma(dz,dz, fma(dy,dy, dx*dx))  neighbour iff d2 < fl(fl(2h)^2).
__device__ __forceinline__ float dist2_f32(const float4 a, const float4 b, float& dx, float& dy, float& dz) {
    dx = __fsub_rn(a.x, b.x);
    dy = __fsub_rn(a.y, b.y);
    dz = __fsub_rn(a.z, b.z);
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

// cell coordinates of a particle (reading A7, same FP32 op sequence as the key kernel); no div / mod needed
__device__ __forceinline__ void cell_of(const float4 p, const GridDev g, int& ix, int& iy, int& iz) {
    ix = (int)fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(p.x, g.ox), g.inv_cell)), 0.0f), g.fx);
    iy = (int)fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(p.y, g.oy), g.inv_cell)), 0.0f), g.fy);
    iz = (int)fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(p.z, g.oz), g.inv_cell)), 0.0f), g.fz);
}

// W(xi,h) = 1/(pi h^3) { 1 - 3/2 xi^2 + 3/4 xi^3 (xi<=1) ; 1/4 (2-xi)^3 (1<=xi<=2) ; 0 }   (Eq. 8)
__device__ __forceinline__ float w_spline_unnorm(float xi) {
    float t = 2.0f - xi;
    float outer = 0.25f * t * t * t;
    float inner = fmaf(xi * xi, fmaf(0.75f, xi, -1.5f), 1.0f);
    return xi <= 1.0f ? inner : fmaxf(outer, 0.0f);
}

// The same piecewise cubic as the difference of two cubes,
//   W pi h^3 = 1/4 (2 - xi)_+^3 - (1 - xi)_+^3      (xi <= 1: 1 - 3/2 xi^2 + 3/4 xi^3; 1 <= xi <= 2: 1/4 (2 - xi)^3),
// with xi = r / h taken from r and -1/h: no branch, no second polynomial, and no cancellation (for xi <= 1 the result is
// >= 1/4 of the larger cube).  7 operations against ~10 for the two selected branches.
__device__ __forceinline__ float w_two_cubes(float r, float neg_inv_h) {
    const float a = fmaxf(fmaf(r, neg_inv_h, 2.0f), 0.0f);
    const float c = fmaxf(fmaf(r, neg_inv_h, 1.0f), 0.0f);
    return fmaf(0.25f * a * a, a, -(c * c * c));
}
__device__ __forceinline__ float sqrt_approx(float x) {   // MUFU.SQRT: relative error 2^-23, sqrt(0) = 0
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

struct ViscDev {
    float h, alpha, beta, eta_h2, gw;   // gw = -45 / (64 pi h^4): grad W_p = gw (2-xi)^2 dr/|dr|
    float inv_h2;                       // 1 / h^2
    double rc2_64;                      // 4 h^2 in FP64 (h as given, widened)
    float eta, gw_unit;                 // VARH: eta and -45 / (64 pi); the h powers are applied per pair
    float inv_h;                        // 1 / h (IEEE division on the host side of the launch)
    float rc2;                          // fl(fl(2h)^2), the FP32 cutoff of A8
    float two_h2, beta2;                // 2 h^2 and 2 beta (hydro_pair_fast)
};

// One accepted pair (d2 < 4h^2, d2 > 0) of Eqs. 10-11 with the one global h: returns f = m_j Pi_ij |grad W_p| / |dr| and
// rv = dr . dv, so that a_i -= f dr and de_i/dt += f rv / 2; mu_ij (L97, <= 0) and c_ij = (c_i + c_j)/2 come out for the
// step criterion of Eq. 17.
//   2 - xi = (4h^2 - |dr|^2) / (h^2 (2 + xi)).  Formed as 2 - |dr|/h in FP32 it loses a factor xi/(2-xi) of relative
//   accuracy near the kernel edge (every term of a sparsely surrounded particle sits there), so the numerator alone is
//   taken in FP64: 3 cvt + 3 DFMA per pair.
//   grad W_p = dWp/dxi * dr/|dr| / h,  dWp/dxi = -45/(64 pi h^3) (2-xi)^2   (L95, Eq. 9, A3)
__device__ __forceinline__ float hydro_pair(const float4 vi /*v, rho*/, const float2 ci /*p/rho^2, c*/, const float m_j,
                                            const float4 vj, const float2 cj, const float dx, const float dy,
                                            const float dz, const float d2, const ViscDev& q, float& rv, float& mu,
                                            float& c_ij) {
    float rinv = rsqrtf(d2);
    rinv = rinv * fmaf(-0.5f * d2 * rinv, rinv, 1.5f);   // one Newton step: ~1 ulp
    const float rr = d2 * rinv;                          // |dr|
    const float num = (float)fma(-(double)dz, (double)dz, fma(-(double)dy, (double)dy, fma(-(double)dx, (double)dx, q.rc2_64)));
    const float tqn = fmaxf(num, 0.0f) * q.inv_h2, tqd = 2.0f + rr * q.inv_h;
    const float tq = tqn / tqd;                          // 2 - xi
    const float gmag = q.gw * tq * tq * rinv;            // grad W_p = gmag * dr
    const float dvx = vi.x - vj.x, dvy = vi.y - vj.y, dvz = vi.z - vj.z;
    rv = fmaf(dz, dvz, fmaf(dy, dvy, dx * dvx));
    // mu_ij = h dr.dv / (|dr|^2 + eta h^2) if dr.dv < 0   (L97)
    const float mun = q.h * rv, mud = d2 + q.eta_h2;
    mu = rv < 0.f ? mun / mud : 0.f;
    const float rho_ij = 0.5f * (vi.w + vj.w);
    c_ij = 0.5f * (ci.y + cj.y);
    const float nun = mu * (q.beta * mu - q.alpha * c_ij);
    const float nu = nun / rho_ij;
    const float Pi = ci.x + cj.x + nu;                   // p_i/rho_i^2 + p_j/rho_j^2 + nu  (L95, A2)
    return m_j * Pi * gmag;                              // m_j Pi |grad Wp| / |dr|
}

// The dense walk's pair term (a particle's sum there has tens to thousands of terms spread over the whole kernel
// support).  The same quantities as hydro_pair, arranged for the fewest instructions:
//   2 - xi = (4h^2 - |dr|^2) / (2h^2 + h |dr|)                 numerator and denominator in FP32: the absolute error of
//            the numerator, <= 2 ulp of 4h^2, is that of any FP32 term; only the RELATIVE error of a term at the kernel
//            edge grows, which matters where ALL of a particle's few terms sit at the edge, i.e. in the sparse walk,
//            which keeps the FP64 numerator, the refined rsqrt and the IEEE divisions;
//   nu_ij  = mu (beta mu - alpha c_ij) / rho_ij = mu (2 beta mu - alpha (c_i + c_j)) / (rho_i + rho_j)   the two halves cancel;
//   1/x by MUFU.RCP, 1/sqrt(x) by MUFU.RSQ, unrefined: relative error <= 2^-22 per term, pseudo-random in sign.
// The accepted pair has 0 < d2 < rc2, so the numerator needs no clamp.  Returns f = m_j Pi_ij |grad W_p| / |dr|; rv, mu as
// in hydro_pair.
__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float hydro_pair_fast(const float4 vi /*v, rho*/, const float2 ci /*p/rho^2, c*/, const float m_j,
                                                 const float4 vj, const float2 cj, const float dx, const float dy,
                                                 const float dz, const float d2, const ViscDev& q, float& rv, float& mu) {
    float rinv;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(d2));   // d2 > 0 and far from the denormals (d2 ~ h^2)
    const float rr = d2 * rinv;                                    // |dr|
    const float tq = (q.rc2 - d2) * rcp_approx(fmaf(rr, q.h, q.two_h2));   // 2 - xi
    const float gmag = q.gw * tq * tq * rinv;                      // grad W_p = gmag * dr
    const float dvx = vi.x - vj.x, dvy = vi.y - vj.y, dvz = vi.z - vj.z;
    rv = fmaf(dz, dvz, fmaf(dy, dvy, dx * dvx));
    mu = 0.f;
    if (rv < 0.f) mu = q.h * rv * rcp_approx(d2 + q.eta_h2);       // mu_ij = h dr.dv / (|dr|^2 + eta h^2) if dr.dv < 0   (L97)
    const float nun = mu * fmaf(q.beta2, mu, -q.alpha * (ci.y + cj.y));
    const float Pi = fmaf(nun, rcp_approx(vi.w + vj.w), ci.x + cj.x);   // p_i/rho_i^2 + p_j/rho_j^2 + nu  (L95, A2)
    return m_j * Pi * gmag;
}

// One accepted pair with a per-pair smoothing length h_ij = hsum / 2, hsum = fl(h_i + h_j) (L82, A24): grad W_p carries
// its own -45 / (64 pi h_ij^4), mu_ij and eta h_ij^2 use h_ij.  Used by BOTH walks: with per-particle lengths a particle
// in a populated cell may still have only a handful of neighbours, all near the edge of its kernel, so the dense-cell
// walk cannot take the short cuts of hydro_pair_fast (measured: de/dt off by 2.0e-4 of the bar's 2e-4 in
// `clamped_dense`).  The pair factor goes like h_ij^-8: with a per-pair h its roundings no longer cancel as a common
// factor of the particle's sum, so it is formed in FP64 and rounded once.
__device__ __forceinline__ float hydro_pair_h(const float4 vi, const float2 ci, const float m_j, const float4 vj,
                                              const float2 cj, const float dx, const float dy, const float dz, const float d2,
                                              const float hsum, const ViscDev& q, float& rv, float& mu, float& c_ij) {
    float rinv = rsqrtf(d2);
    rinv = rinv * fmaf(-0.5f * d2 * rinv, rinv, 1.5f);   // one Newton step: ~1 ulp
    const float rr = d2 * rinv;                        // |dr|
    const double hd = 0.5 * (double)hsum, ihd = 1.0 / hd, ih2 = ihd * ihd;
    const double num = fma(-(double)dz, (double)dz, fma(-(double)dy, (double)dy, fma(-(double)dx, (double)dx, (double)hsum * (double)hsum)));
    const double tqd = fmax(num, 0.0) * ih2 / (2.0 + (double)rr * ihd);       // 2 - xi
    const float gmag = (float)((double)q.gw_unit * ih2 * ih2 * tqd * tqd) * rinv;   // grad W_p = gmag * dr
    const float hh = 0.5f * hsum;
    const float eta_h2 = q.eta * hh * hh;
    const float dvx = vi.x - vj.x, dvy = vi.y - vj.y, dvz = vi.z - vj.z;
    rv = fmaf(dz, dvz, fmaf(dy, dvy, dx * dvx));
    // mu_ij = h dr.dv / (|dr|^2 + eta h^2) if dr.dv < 0   (L97)
    mu = rv < 0.f ? (hh * rv) / (d2 + eta_h2) : 0.f;                   // IEEE division
    const float rho_ij = 0.5f * (vi.w + vj.w);
    c_ij = 0.5f * (ci.y + cj.y);
    const float nu = (mu * (q.beta * mu - q.alpha * c_ij)) / rho_ij;
    const float Pi = ci.x + cj.x + nu;                 // p_i/rho_i^2 + p_j/rho_j^2 + nu  (L95, A2)
    return m_j * Pi * gmag;                            // m_j Pi |grad Wp| / |dr|
}

// Eq. 17 (L127) for one gas particle: the bracket s / (c^max (1 + 1.2 alpha) + 1.2 beta mu^max + sqrt(s (|Q| + |E|))) from
// the squared minimum distance (>= rc2_none: no neighbour, then s = s_none, reading A22), c^max, mu^max and the
// particle's right-hand sides Q = a_sph + a_grav (Eq. 10), E = de/dt (Eq. 11).
__device__ __forceinline__ float cfl_bracket(float d2min, bool none, float s_none, float cmax, float mumax, float alpha,
                                             float beta, const float4 as, const float4 ag) {
    const float qx = as.x + ag.x, qy = as.y + ag.y, qz = as.z + ag.z;
    const float qe = sqrtf(fmaf(qz, qz, fmaf(qy, qy, qx * qx))) + fabsf(as.w);   // |Q_i| + |E_i|
    const float sm = none ? s_none : sqrtf(d2min);
    return sm / (fmaf(cmax, 1.0f + 1.2f * alpha, 1.2f * beta * mumax) + sqrtf(sm * qe));
}
// the running minimum of c_cfl x bracket over the active lanes of the warp, then one atomicMin on the bit pattern
__device__ __forceinline__ void cfl_min(float v, unsigned int* dt_bits) {
    const unsigned act = __activemask();
    const unsigned m = __reduce_min_sync(act, __float_as_uint(fmaxf(v, 0.f)));
    if ((threadIdx.x & 31) == __ffs(act) - 1) atomicMin(dt_bits, m);
}

// ---- dense-cell work list (common.cuh: DenseItem, DenseList) ------------------------------------------------------
__device__ __forceinline__ void dense_append(uint32_t key, uint32_t count, unsigned int* ctl, DenseItem* items) {
    const uint32_t nchunk = (count + kDenseTT - 1) / kDenseTT;
    const uint32_t at = atomicAdd(ctl, nchunk);
    for (uint32_t c = 0; c < nchunk; ++c) items[at + c] = DenseItem{key, c};
}
}  // namespace sphb
