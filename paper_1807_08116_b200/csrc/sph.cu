// sph.cu — (a7) density, (a8) EOS, (a9) hydro force / energy rate over the grid-sort ranges.
//
// Work is laid out in CELL ORDER (the sorted copy posm_s written by the grid build): thread s
// owns sorted slot s, so the threads of a warp sit in the same or adjacent cells, walk nearly the
// same candidate ranges, and their loads of posm_s[t] are warp-broadcasts / L1 hits.  The 27-cell
// stencil is walked as 9 x-runs: the cells (cx-1, cx, cx+1) of one (y, z) row are contiguous in
// sorted order, so each run is one [start, end) slot range (L160, L203, L207).
// Candidates come out in ascending sorted slot, so every sum has a fixed order: results are
// bitwise reproducible.
//
// Cutoff predicate (A8), identical op sequence to the oracle:
//   dx = x_i (-) x_j ...  d2 = fma(dz,dz, fma(dy,dy, dx*dx))  neighbour iff d2 < fl(fl(2h)^2).
#include "sph_dev.cuh"

namespace sphb {

// 9 x-runs of the stencil of the cell (ix,iy,iz): run r -> [lo, hi) sorted slots, (0,0) outside the grid
__device__ __forceinline__ void stencil_run(const uint32_t* __restrict__ start, const GridDev g, int ix, int iy, int iz,
                                            int r, uint32_t& lo, uint32_t& hi) {
    const int cy = iy + (r % 3) - 1, cz = iz + (r / 3) - 1;
    lo = hi = 0u;
    if (cy >= 0 && cy < g.my && cz >= 0 && cz < g.mz) {
        const uint32_t row = (uint32_t)g.mx * ((uint32_t)cy + (uint32_t)g.my * (uint32_t)cz);   // M < 2^31 (check_grid)
        lo = start[row + (uint32_t)max(ix - 1, 0)];
        hi = start[row + (uint32_t)min(ix + 1, g.mx - 1) + 1u];
    }
}

// dense_min > 0: the cells holding at least that many particles belong to the dense walk (sph_dense.cu)
__device__ __forceinline__ bool own_cell_is_dense(const uint32_t* __restrict__ start, const GridDev g, int ix, int iy,
                                                  int iz, uint32_t dense_min) {
    if (dense_min == 0u) return false;
    const uint32_t k = (uint32_t)ix + (uint32_t)g.mx * ((uint32_t)iy + (uint32_t)g.my * (uint32_t)iz);
    return start[k + 1u] - start[k] >= dense_min;
}

// ---------------------------------------------------------------- (a7) density, Eq. 7-8
// VARH: per-particle smoothing lengths h_s[] in cell order; the pair length is
// h_ij = (h_i + h_j)/2, the pair is a neighbour pair iff d2 < fl(fl(h_i + h_j)^2) (reading A24, FP32 like A8),
// and W(|dr|/h_ij, h_ij) carries its own 1/(pi h_ij^3).  VARH = false is the global-h kernel, unchanged.
template <bool VARH>
__global__ void __launch_bounds__(128) k_density(const float4* __restrict__ posm_s, const float* __restrict__ h_s,
                                                 const uint32_t* __restrict__ perm, const uint32_t* __restrict__ start,
                                                 int n, GridDev g, float rc2, float inv_h, float norm,
                                                 uint32_t dense_min, Shard sh, float* __restrict__ rho) {
    const int s = (int)((blockIdx.x * sh.world + sh.rank) * 128u + threadIdx.x);   // the rank's tiles of 128 slots
    if (s >= n) return;
    const float4 pi = posm_s[s];
    const float h_i = VARH ? h_s[s] : 0.f;
    int ix, iy, iz;
    cell_of(pi, g, ix, iy, iz);
    if (own_cell_is_dense(start, g, ix, iy, iz, dense_min)) return;   // sph_dense_rho.cu walks that cell
    float sum = 0.f;   // includes the self term m_i W(0): j = i passes the predicate with d2 = 0 (A5)
#pragma unroll 1
    for (int r = 0; r < 9; ++r) {
        uint32_t lo, hi;
        stencil_run(start, g, ix, iy, iz, r, lo, hi);
        for (uint32_t t = lo; t < hi; ++t) {
            const float4 pj = posm_s[t];
            float dx, dy, dz;
            const float d2 = dist2_f32(pi, pj, dx, dy, dz);
            if (VARH) {
                const float hsum = __fadd_rn(h_i, h_s[t]);         // 2 h_ij
                if (d2 < __fmul_rn(hsum, hsum)) {
                    const float inv = 1.0f / (0.5f * hsum);        // IEEE division
                    const float xi = sqrtf(d2) * inv;
                    sum = fmaf(pj.w, w_spline_unnorm(xi) * (inv * inv * inv), sum);
                }
            } else if (d2 < rc2) {
                // the density is a sum of positive terms held to 1e-5: MUFU.SQRT (2^-23) and the branch-free form of W
                sum = fmaf(pj.w, w_two_cubes(sqrt_approx(d2), -inv_h), sum);
            }
        }
    }
    rho[perm[s]] = sum * norm;
}

// smoothing lengths into cell order; a length above the cap h_max (which sized the cells: the 3x3x3 stencil would miss
// neighbours) raises SPH_STATUS_HSML_ABOVE_CAP in the workspace's status word (sph_workspace_status)
__global__ void __launch_bounds__(256) k_gather_h(const float* __restrict__ a, const uint32_t* __restrict__ perm, int n,
                                                  float h_max, unsigned int* __restrict__ status, float* __restrict__ a_s) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const float v = a[perm[s]];
    a_s[s] = v;
    if (!(v <= h_max)) atomicOr(status, (unsigned int)SPH_STATUS_HSML_ABOVE_CAP);   // also catches NaN
}

// L82: h_i = sigma (m_i / rho_i)^(1/3), capped at h_max (reading A25).  cbrtf is within 1 ulp.
__global__ void __launch_bounds__(256) k_smoothing_lengths(const float4* __restrict__ posm, const float* __restrict__ rho,
                                                           int n, float sigma, float h_max, float* __restrict__ hsml) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) hsml[i] = fminf(sigma * cbrtf(posm[i].w / rho[i]), h_max);
}

int smoothing_lengths(const float4* posm, const float* rho, int64_t n_gas, float sigma, float h_max, float* hsml,
                      cudaStream_t st) {
    if (n_gas <= 0) return SPH_OK;
    k_smoothing_lengths<<<(unsigned)cdiv(n_gas, 256), 256, 0, st>>>(posm, rho, (int)n_gas, sigma, h_max, hsml);
    SPHB_LAUNCHED();
    return SPH_OK;
}

int gather_sorted_h(const float* hsml, const uint32_t* perm, int64_t n_gas, float h_max, unsigned int* status, float* h_s,
                    cudaStream_t st) {
    if (n_gas <= 0) return SPH_OK;
    k_gather_h<<<(unsigned)cdiv(n_gas, 256), 256, 0, st>>>(hsml, perm, (int)n_gas, h_max, status, h_s);
    SPHB_LAUNCHED();
    return SPH_OK;
}

int forces_dense(const float4* posm_s, const float4* velr_s, const float2* pc_s, const float* h_s, const uint32_t* perm,
                 const uint32_t* cell_start, const sph_grid* g, float rc2, const ViscDev& q, const DenseList& dl,
                 const CflArgs* cfl, float4* acc_sph, cudaStream_t st, Shard sh);   // sph_dense.cu

int density_dense(const float4* posm_s, const float* h_s, const uint32_t* perm, const uint32_t* cell_start, const sph_params* p,
                  const sph_grid* g, const DenseList& dl, float* rho, cudaStream_t st, Shard sh);   // sph_dense_rho.cu

// CTAs of a thread-per-slot pass: the rank's tiles rank, rank + world, ... of the cdiv(n, 128)
static unsigned shard_blocks(int64_t n, Shard sh) {
    const int64_t tiles = cdiv(n, 128);
    return tiles > (int64_t)sh.rank ? (unsigned)((tiles - sh.rank + sh.world - 1) / sh.world) : 0u;
}

int density_sorted(const float4* posm_s, const float* h_s /*cell order, or NULL: global h*/, const uint32_t* perm,
                   const uint32_t* cell_start, int64_t n_gas, const sph_params* p, const sph_grid* g,
                   const DenseList* dense, float* rho, cudaStream_t st, Shard sh) {
    if (n_gas <= 0) return SPH_OK;
    const float two_h = 2.0f * p->h;
    const float rc2 = two_h * two_h;
    const float inv_h = 1.0f / p->h;
    const unsigned blocks = shard_blocks(n_gas, sh);
    if (blocks == 0u) return SPH_OK;
    if (h_s) {
        k_density<true><<<blocks, 128, 0, st>>>(posm_s, h_s, perm, cell_start, (int)n_gas, to_dev(g), rc2, inv_h,
                                                (float)(1.0 / 3.14159265358979323846), dense ? (uint32_t)kDenseMin : 0u, sh, rho);
        SPHB_LAUNCHED();
        if (dense) SPHB_TRY(density_dense(posm_s, h_s, perm, cell_start, p, g, *dense, rho, st, sh));
    } else {
        const float norm = (float)(1.0 / (3.14159265358979323846 * (double)p->h * (double)p->h * (double)p->h));
        k_density<false><<<blocks, 128, 0, st>>>(posm_s, nullptr, perm, cell_start, (int)n_gas, to_dev(g), rc2, inv_h,
                                                 norm, dense ? (uint32_t)kDenseMin : 0u, sh, rho);
        SPHB_LAUNCHED();
        if (dense) SPHB_TRY(density_dense(posm_s, nullptr, perm, cell_start, p, g, *dense, rho, st, sh));
    }
    return SPH_OK;
}

// ---------------------------------------------------------------- (a8) EOS gather into cell order
// velr_s[s] = (v_x, v_y, v_z, rho) ; pc_s[s] = (p/rho^2, c) with p = (gamma-1) rho e (Eq. 5),
// c = sqrt(gamma p / rho) = sqrt(gamma (gamma-1) e) (L99).
__global__ void __launch_bounds__(256) k_eos_gather(const float4* __restrict__ vele, const float* __restrict__ rho,
                                                    const uint32_t* __restrict__ perm, int n, float gamma,
                                                    float4* __restrict__ velr_s, float2* __restrict__ pc_s) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint32_t i = perm[s];
    const float4 v = vele[i];
    const float r = rho[i];
    const float gm1 = gamma - 1.0f;
    velr_s[s] = make_float4(v.x, v.y, v.z, r);
    pc_s[s] = make_float2(gm1 * v.w / r, sqrtf(gamma * gm1 * v.w));
}

// ---------------------------------------------------------------- (a9) hydro force, Eqs. 10-11
// Compensated (Kahan) accumulation.  The hydro terms of one particle routinely cancel by 10^2-10^3
// and dense cells sum hundreds of them; a plain FP32 running sum loses ~sqrt(n) ulps of the GROSS
// sum, which is what broke the 2e-4 parity bar on the clumpy configs.  Cost: 3 extra FADD per add.
struct KSum {
    float s = 0.f, c = 0.f;
    __device__ __forceinline__ void add(float x) {
        const float y = __fsub_rn(x, c);
        const float t = __fadd_rn(s, y);
        c = __fsub_rn(__fsub_rn(t, s), y);
        s = t;
    }
};

// VARH: as k_density<true> — pair length h_ij = (h_i + h_j)/2 in the cutoff, in grad W_p and in mu_ij (L82, L95-97).
// CFL: the per-particle terms of Eq. 17 (s^min, c^max, mu^max) are gathered in the same walk (L125-129) and the bracket is
// formed at its end (CflArgs, common.cuh).
template <bool VARH, bool CFL>
__global__ void __launch_bounds__(128) k_forces(const float4* __restrict__ posm_s, const float4* __restrict__ velr_s,
                                                const float2* __restrict__ pc_s, const float* __restrict__ h_s,
                                                const uint32_t* __restrict__ perm, const uint32_t* __restrict__ start,
                                                int n, GridDev g, float rc2, ViscDev q, uint32_t dense_min, CflArgs cfl,
                                                Shard sh, float4* __restrict__ acc) {
    const int s = (int)((blockIdx.x * sh.world + sh.rank) * 128u + threadIdx.x);   // the rank's tiles of 128 slots
    if (s >= n) return;
    const float4 pi = posm_s[s];
    int ix, iy, iz;
    cell_of(pi, g, ix, iy, iz);
    if (own_cell_is_dense(start, g, ix, iy, iz, dense_min)) return;   // sph_dense.cu walks that cell
    const float4 vi = velr_s[s];
    const float2 ci = pc_s[s];
    const float h_i = VARH ? h_s[s] : 0.f;
    KSum ax, ay, az, de;
    float d2min = __int_as_float(0x7f800000), cmax = ci.y, mumax = 0.f;   // A22: no neighbour -> s = 2h, c_i, 0
#pragma unroll 1
    for (int r = 0; r < 9; ++r) {
        uint32_t lo, hi_;
        stencil_run(start, g, ix, iy, iz, r, lo, hi_);
        for (uint32_t t = lo; t < hi_; ++t) {
            const float4 pj = posm_s[t];
            float dx, dy, dz;
            const float d2 = dist2_f32(pi, pj, dx, dy, dz);
            float rc2p = rc2, hsum = 0.f;
            if (VARH) {
                hsum = __fadd_rn(h_i, h_s[t]);                     // 2 h_ij
                rc2p = __fmul_rn(hsum, hsum);
            }
            if (d2 < rc2p && d2 > 0.f) {   // d2 == 0: self, or a coincident pair (A9) — no contribution
                const float4 vj = velr_s[t];
                const float2 cj = pc_s[t];
                float f, rv, mu, c_ij;
                if (VARH) {
                    f = hydro_pair_h(vi, ci, pj.w, vj, cj, dx, dy, dz, d2, hsum, q, rv, mu, c_ij);
                } else {
                    f = hydro_pair(vi, ci, pj.w, vj, cj, dx, dy, dz, d2, q, rv, mu, c_ij);
                }
                if (CFL) {
                    d2min = fminf(d2min, d2);
                    cmax = fmaxf(cmax, c_ij);
                    mumax = fmaxf(mumax, fabsf(mu));
                }
                ax.add(-f * dx);
                ay.add(-f * dy);
                az.add(-f * dz);
                de.add(0.5f * f * rv);                             // 1/2 m_j Pi dv . grad W_p   (Eq. 11)
            }
        }
    }
    const uint32_t i = perm[s];
    const float4 a_own = make_float4(ax.s, ay.s, az.s, de.s);
    if (acc) acc[i] = a_own;
    if (CFL) {
        const float bound = cfl_bracket(d2min, d2min == __int_as_float(0x7f800000), VARH ? 2.0f * h_i : 2.0f * q.h, cmax, mumax,
                                        q.alpha, q.beta, cfl.q_sph ? cfl.q_sph[i] : a_own, cfl.acc_grav[i]);
        if (cfl.dt_particle) cfl.dt_particle[i] = bound;
        cfl_min(cfl.c_cfl * bound, cfl.dt_bits);
    }
}

int forces_sorted(const float4* posm_s, const float4* vele, const float* rho, const float* h_s /*or NULL*/,
                  const uint32_t* perm, const uint32_t* cell_start, int64_t n_gas, const sph_params* p, const sph_grid* g,
                  const DenseList* dense, const CflArgs* cfl, float4* velr_s, float2* pc_s, float4* acc_sph,
                  cudaStream_t st, Shard sh) {
    if (n_gas <= 0) return SPH_OK;
    const int n = (int)n_gas;
    k_eos_gather<<<(unsigned)cdiv(n, 256), 256, 0, st>>>(vele, rho, perm, n, p->gamma, velr_s, pc_s);
    SPHB_LAUNCHED();
    const float two_h = 2.0f * p->h;
    ViscDev q;
    q.h = p->h;
    q.alpha = p->alpha;
    q.beta = p->beta;
    q.eta_h2 = p->eta * p->h * p->h;
    const double h = p->h;
    q.gw = (float)(-45.0 / (64.0 * 3.14159265358979323846 * h * h * h * h));   // dWp/dxi scale / h
    q.inv_h2 = (float)(1.0 / (h * h));
    q.rc2_64 = 4.0 * h * h;
    q.eta = p->eta;
    q.gw_unit = (float)(-45.0 / (64.0 * 3.14159265358979323846));
    q.inv_h = 1.0f / p->h;
    q.rc2 = two_h * two_h;
    q.two_h2 = (float)(2.0 * h * h);
    q.beta2 = 2.0f * p->beta;
    const unsigned blocks = shard_blocks(n_gas, sh);
    if (blocks == 0u) return SPH_OK;
    const GridDev gd = to_dev(g);
    const CflArgs c = cfl ? *cfl : CflArgs{};
    const uint32_t dmin = dense ? (uint32_t)kDenseMin : 0u;   // those cells are walked by sph_dense.cu
    if (h_s && cfl)
        k_forces<true, true><<<blocks, 128, 0, st>>>(posm_s, velr_s, pc_s, h_s, perm, cell_start, n, gd, q.rc2, q, dmin, c, sh, acc_sph);
    else if (h_s)
        k_forces<true, false><<<blocks, 128, 0, st>>>(posm_s, velr_s, pc_s, h_s, perm, cell_start, n, gd, q.rc2, q, dmin, c, sh, acc_sph);
    else if (cfl)
        k_forces<false, true><<<blocks, 128, 0, st>>>(posm_s, velr_s, pc_s, nullptr, perm, cell_start, n, gd, q.rc2, q, dmin, c, sh, acc_sph);
    else
        k_forces<false, false><<<blocks, 128, 0, st>>>(posm_s, velr_s, pc_s, nullptr, perm, cell_start, n, gd, q.rc2, q, dmin, c, sh, acc_sph);
    SPHB_LAUNCHED();
    if (dmin) SPHB_TRY(forces_dense(posm_s, velr_s, pc_s, h_s, perm, cell_start, g, q.rc2, q, *dense, cfl, acc_sph, st, sh));
    return SPH_OK;
}

// ---------------------------------------------------------------- (NEXT-1) modified CFL step, Eq. 17
// The terms of Eq. 17 are gathered by the forces kernels themselves (template flag CFL above, and in sph_dense.cu); the
// global minimum is an atomicMin on the float bit pattern (positive floats order like unsigned integers), hence exact
// and order-independent.  This sets its starting value: the ceiling dt_max of the step, +inf for none.
__global__ void k_cfl_init(float* dt_out, float dt_max) { *dt_out = dt_max; }

int cfl_init(float* dt_dev, float dt_max, cudaStream_t st) {
    k_cfl_init<<<1, 1, 0, st>>>(dt_dev, dt_max);
    SPHB_LAUNCHED();
    return SPH_OK;
}

}  // namespace sphb
