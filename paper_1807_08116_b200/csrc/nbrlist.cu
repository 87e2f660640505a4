// nbrlist.cu — sph_neighbour_lists: explicit neighbour sets in CSR form (test helper of the
// boundary, include/sph_b200.h).  Same walk and same FP32 predicate (A8) as the density kernel.
#include "common.cuh"

namespace sphb {

__device__ __forceinline__ float nl_d2(const float4 a, const float4 b) {
    const float dx = __fsub_rn(a.x, b.x), dy = __fsub_rn(a.y, b.y), dz = __fsub_rn(a.z, b.z);
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

// PASS 0: count.  PASS 1: write original indices of the neighbours at nbr_offset[i].
template <int PASS>
__global__ void __launch_bounds__(128) k_nbr(const float4* __restrict__ posm_s, const uint32_t* __restrict__ perm,
                                             const uint32_t* __restrict__ start, int n, GridDev g, float rc2,
                                             const float* __restrict__ h_s /*cell order, or NULL (global h)*/,
                                             uint32_t* __restrict__ cnt, const uint64_t* __restrict__ off,
                                             uint32_t* __restrict__ idx) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const float4 pi = posm_s[s];
    const int ix = (int)fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(pi.x, g.ox), g.inv_cell)), 0.f), g.fx);
    const int iy = (int)fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(pi.y, g.oy), g.inv_cell)), 0.f), g.fy);
    const int iz = (int)fminf(fmaxf(floorf(__fmul_rn(__fsub_rn(pi.z, g.oz), g.inv_cell)), 0.f), g.fz);
    const uint32_t i = perm[s];
    uint32_t c = 0;
    uint64_t base = PASS ? off[i] : 0;
    for (int r = 0; r < 9; ++r) {
        const int cy = iy + (r % 3) - 1, cz = iz + (r / 3) - 1;
        if (cy < 0 || cy >= g.my || cz < 0 || cz >= g.mz) continue;
        const int64_t row = (int64_t)g.mx * (cy + (int64_t)g.my * cz);
        const uint32_t lo = start[row + max(ix - 1, 0)], hi = start[row + min(ix + 1, g.mx - 1) + 1];
        for (uint32_t t = lo; t < hi; ++t) {
            if ((int)t == s) continue;
            float lim = rc2;
            if (h_s) {   // reading A24: pair cutoff fl(fl(h_i + h_j)^2)
                const float hsum = __fadd_rn(h_s[s], h_s[t]);
                lim = __fmul_rn(hsum, hsum);
            }
            if (nl_d2(pi, posm_s[t]) < lim) {
                if (PASS) idx[base + c] = perm[t];
                ++c;
            }
        }
    }
    if (!PASS) cnt[i] = c;
}

// one CTA: exclusive scan of cnt[n] into off[n+1] (64-bit), chunks of 1024 with a carry
__global__ void __launch_bounds__(1024) k_nbr_scan(const uint32_t* __restrict__ cnt, int n, uint64_t* __restrict__ off) {
    __shared__ uint64_t wsum[32];
    __shared__ uint64_t carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int base = 0; base < n; base += 1024) {
        const int i = base + threadIdx.x;
        const uint64_t v = i < n ? cnt[i] : 0;
        uint64_t inc = v;
        for (int o = 1; o < 32; o <<= 1) {
            uint64_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) wsum[w] = inc;
        __syncthreads();
        if (w == 0) {
            uint64_t sv = wsum[lane];
            for (int o = 1; o < 32; o <<= 1) {
                uint64_t t = __shfl_up_sync(0xffffffffu, sv, o);
                if (lane >= o) sv += t;
            }
            wsum[lane] = sv;
        }
        __syncthreads();
        const uint64_t carry = carry_s;
        const uint64_t ex = carry + (w ? wsum[w - 1] : 0) + inc - v;
        if (i < n) off[i] = ex;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = carry + wsum[31];
        __syncthreads();
    }
    if (threadIdx.x == 0) off[n] = carry_s;
}

// each list ascending in original index: in-place insertion sort, one thread per list (test helper)
__global__ void __launch_bounds__(128) k_nbr_sort(const uint64_t* __restrict__ off, int n, uint32_t* __restrict__ idx) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint64_t a = off[i], b = off[i + 1];
    for (uint64_t q = a + 1; q < b; ++q) {
        const uint32_t v = idx[q];
        uint64_t r = q;
        while (r > a && idx[r - 1] > v) {
            idx[r] = idx[r - 1];
            --r;
        }
        idx[r] = v;
    }
}

}  // namespace sphb

using namespace sphb;

extern "C" int sph_neighbour_lists_h(const float* posm, const float* hsml, int64_t n_gas, float h, const sph_grid* g,
                                     const uint32_t* perm, const uint32_t* cell_start, uint32_t* nbr_count,
                                     uint64_t* nbr_offset, uint32_t* nbr_index, uint64_t nbr_capacity, void* ws,
                                     size_t ws_bytes, void* stream) {
    if (n_gas < 0 || n_gas >= (1ll << 31) || !(h > 0.f) || !nbr_offset) return SPH_ERR_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    if (n_gas == 0) {
        SPHB_CUDA(cudaMemsetAsync(nbr_offset, 0, sizeof(uint64_t), st));
        SPHB_CUDA(cudaStreamSynchronize(st));
        return SPH_OK;
    }
    if (!posm || !perm || !cell_start || !nbr_count || !ws || !aligned16(posm) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, h));
    Workspace w = carve(ws, n_gas, n_gas, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    const int n = (int)n_gas;
    const float two_h = 2.0f * h;
    const float rc2 = two_h * two_h;
    const GridDev gd = to_dev(g);
    SPHB_TRY(gather_sorted_pos(reinterpret_cast<const float4*>(posm), perm, n_gas, w.posm_s, st));
    const float* h_s = nullptr;
    if (hsml) {
        SPHB_TRY(gather_sorted_h(hsml, perm, n_gas, h, w.status, w.h_s, st));
        h_s = w.h_s;
    }
    k_nbr<0><<<(unsigned)cdiv(n, 128), 128, 0, st>>>(w.posm_s, perm, cell_start, n, gd, rc2, h_s, nbr_count, nullptr,
                                                    nullptr);
    SPHB_LAUNCHED();
    k_nbr_scan<<<1, 1024, 0, st>>>(nbr_count, n, nbr_offset);
    SPHB_LAUNCHED();
    uint64_t total = 0;
    SPHB_CUDA(cudaMemcpyAsync(&total, nbr_offset + n, sizeof(total), cudaMemcpyDeviceToHost, st));
    SPHB_CUDA(cudaStreamSynchronize(st));
    if (total > nbr_capacity || (total > 0 && !nbr_index)) return SPH_ERR_WORKSPACE;
    if (total > 0) {
        k_nbr<1><<<(unsigned)cdiv(n, 128), 128, 0, st>>>(w.posm_s, perm, cell_start, n, gd, rc2, h_s, nbr_count, nbr_offset,
                                                        nbr_index);
        SPHB_LAUNCHED();
        k_nbr_sort<<<(unsigned)cdiv(n, 128), 128, 0, st>>>(nbr_offset, n, nbr_index);
        SPHB_LAUNCHED();
    }
    SPHB_CUDA(cudaStreamSynchronize(st));
    return SPH_OK;
}

extern "C" int sph_neighbour_lists(const float* posm, int64_t n_gas, float h, const sph_grid* g, const uint32_t* perm,
                                   const uint32_t* cell_start, uint32_t* nbr_count, uint64_t* nbr_offset,
                                   uint32_t* nbr_index, uint64_t nbr_capacity, void* ws, size_t ws_bytes, void* stream) {
    return sph_neighbour_lists_h(posm, nullptr, n_gas, h, g, perm, cell_start, nbr_count, nbr_offset, nbr_index,
                                 nbr_capacity, ws, ws_bytes, stream);
}
