// grid.cu — (a1-a6) the grid-sort neighbour search of PAPER.md L156-207, re-designed for sm_100a.
//
// Paper (Kepler): K0 zero, K1 key + atomic histogram, K2 Hillis-Steele scan per block + O(G^2)
// atomics on block totals, K3 add block offsets, K4 atomic scatter (order inside a cell left to
// the atomics: neither stable nor deterministic, L204).
// Here:
//   zero      cudaMemsetAsync of count[M]
//   k_key_hist  per particle: cell number (A7, bit-exact FP32 op sequence) and
//               rank_u[i] = atomicAdd(&count[k], 1) — the histogram atomics already hand every
//               particle a unique (unstable) slot in its cell, so no second cursor array / pass;
//               four particles per thread, their loads and atomics in flight together.  On the
//               sparse galaxy grids (N_g <= M / 8) the particles also gather the totals of the
//               scan's tiles of 4096 cells, through a per-CTA histogram in shared memory
//   k_scan_*    two-level exclusive scan ("in-block then across blocks", L171-172) with warp
//               shuffles, 16 cells per thread through uint4 loads.  Up to 8192 tiles (33.5 M cells)
//               k_scan_apply adds up the totals of the tiles before its own by itself and, where
//               k_key_hist gathered the totals, is the only pass over the cells: 4 B read + 4 B
//               written per cell.  Otherwise k_scan_tile_sums (4 B read per cell more) and, above
//               8192 tiles, k_scan_tile_offsets
//   k_scatter   tmp[start[k_i] + rank_u[i]] = i                          (unstable, like K4)
//   k_stable    stable fix-up: slot s holding i moves to start[k] + #{t in cell : tmp[t] < i},
//               i.e. ascending original index inside each cell (A16).  The count costs O(n_c)
//               reads per particle, never more than the density pass's own-cell pair tests, so
//               it is safe for any cell population.  Fused with (a6): writes perm and the
//               cell-ordered copy posm_s.
// All results are deterministic (integer atomics commute; the fix-up removes the only order
// the atomics decide).
#include "sph_dev.cuh"

namespace sphb {

// ---------------------------------------------------------------- bounding box (A7)
__device__ __forceinline__ void atomic_min_f(float* addr, float v) {
    // order-preserving for all finite floats: signed compare for >= 0, unsigned reversed for < 0
    if (v >= 0.f) atomicMin(reinterpret_cast<int*>(addr), __float_as_int(v));
    else atomicMax(reinterpret_cast<unsigned int*>(addr), __float_as_uint(v));
}
__device__ __forceinline__ void atomic_max_f(float* addr, float v) {
    if (v >= 0.f) atomicMax(reinterpret_cast<int*>(addr), __float_as_int(v));
    else atomicMin(reinterpret_cast<unsigned int*>(addr), __float_as_uint(v));
}

__global__ void k_bbox_init(float* bb) {
    if (threadIdx.x < 3) bb[threadIdx.x] = __int_as_float(0x7f7fffff);        // +FLT_MAX
    else if (threadIdx.x < 6) bb[threadIdx.x] = __int_as_float(0xff7fffff);   // -FLT_MAX
}

__global__ void __launch_bounds__(256) k_bbox(const float4* __restrict__ posm, int n, float* bb) {
    float lo[3] = {3.4e38f, 3.4e38f, 3.4e38f}, hi[3] = {-3.4e38f, -3.4e38f, -3.4e38f};
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        float4 p = posm[i];
        lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
        lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
        lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            atomic_min_f(bb + a, lo[a]);
            atomic_max_f(bb + 3 + a, hi[a]);
        }
    }
}

int bbox_gas(const float4* posm, int64_t n_gas, float* bb, cudaStream_t st) {
    k_bbox_init<<<1, 32, 0, st>>>(bb);
    SPHB_LAUNCHED();
    int blocks = (int)(cdiv(n_gas, 256) < (int64_t)num_sms() * 8 ? cdiv(n_gas, 256) : (int64_t)num_sms() * 8);
    k_bbox<<<blocks, 256, 0, st>>>(posm, (int)n_gas, bb);
    SPHB_LAUNCHED();
    return SPH_OK;
}

// ---------------------------------------------------------------- (a1) cell number, (a2) histogram
__device__ __forceinline__ int cell_coord(float x, float o, float inv_cell, float fmax_) {
    float c = __fmul_rn(__fsub_rn(x, o), inv_cell);   // two RN FP32 ops, never contracted (A7)
    c = fminf(fmaxf(floorf(c), 0.0f), fmax_);         // clamp in float before the cast
    return (int)c;
}
__device__ __forceinline__ uint32_t cell_key(const float4 p, const GridDev g) {
    int ix = cell_coord(p.x, g.ox, g.inv_cell, g.fx);
    int iy = cell_coord(p.y, g.oy, g.inv_cell, g.fy);
    int iz = cell_coord(p.z, g.oz, g.inv_cell, g.fz);
    return (uint32_t)ix + (uint32_t)g.mx * ((uint32_t)iy + (uint32_t)g.my * (uint32_t)iz);
}

// Both particle passes below are bound by the latency of their scattered accesses (an atomic with its return value; a
// gather of start[] and a scattered store), not by bandwidth: a thread takes kPassItems particles, a CTA-stride apart
// (coalesced), and issues their loads, then their atomics / gathers, back to back — kPassItems requests in flight per
// thread instead of one.
constexpr int kPassItems = 4;
constexpr int kPassBatch = 256 * kPassItems;   // particles a CTA takes at a time
// The scan's tile of cells (k_scan_*: 4096 cells per CTA) and the largest number of tiles for which the tile totals are
// gathered here, by the particles, instead of by a pass over count[M] (k_scan_tile_sums): every CTA keeps a private
// histogram over the tiles in shared memory (<= 32 KB) and adds its non-zero entries to tile_sums[] at the end — one
// global atomic per (CTA, tile it touched), so a galaxy core or a clump does not pile its atomics on a few words (one
// more GLOBAL atomic per particle did, and measured slower).  This drops one of the two reads of count[M].
constexpr int kTileShift = 12;
constexpr int kFuseTiles = 8192;
__global__ void __launch_bounds__(256) k_key_hist(const float4* __restrict__ posm, int n, GridDev g,
                                                  uint32_t* __restrict__ key, uint32_t* __restrict__ rank_u,
                                                  uint32_t* __restrict__ count, uint32_t* __restrict__ tile_sums,
                                                  int n_tiles /*0: no tile totals*/, unsigned int* dense_ctl) {
    extern __shared__ uint32_t sh_tiles[];
    if (dense_ctl && blockIdx.x == 0 && threadIdx.x == 0) *dense_ctl = 0u;   // the work list k_scan_apply is about to write
    for (int t = threadIdx.x; t < n_tiles; t += 256) sh_tiles[t] = 0u;
    if (n_tiles) __syncthreads();
    for (int64_t b0 = (int64_t)blockIdx.x * kPassBatch; b0 < n; b0 += (int64_t)gridDim.x * kPassBatch) {
        const int i0 = (int)b0 + threadIdx.x;
        float4 p[kPassItems];
#pragma unroll
        for (int q = 0; q < kPassItems; ++q) {
            const int i = i0 + 256 * q;
            p[q] = i < n ? posm[i] : make_float4(0.f, 0.f, 0.f, 0.f);
        }
        uint32_t k[kPassItems], r[kPassItems];
#pragma unroll
        for (int q = 0; q < kPassItems; ++q) {
            k[q] = cell_key(p[q], g);
            r[q] = (i0 + 256 * q < n) ? atomicAdd(count + k[q], 1u) : 0u;
        }
#pragma unroll
        for (int q = 0; q < kPassItems; ++q) {
            const int i = i0 + 256 * q;
            if (i < n) {
                key[i] = k[q];
                rank_u[i] = r[q];
                if (n_tiles) atomicAdd(sh_tiles + (k[q] >> kTileShift), 1u);
            }
        }
    }
    if (n_tiles) {
        __syncthreads();
        for (int t = threadIdx.x; t < n_tiles; t += 256) {
            const uint32_t v = sh_tiles[t];
            if (v) atomicAdd(tile_sums + t, v);
        }
    }
}

// ---------------------------------------------------------------- (a3) two-level exclusive scan
constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;   // 4096 cells per CTA
static_assert(kScanTile == 1 << kTileShift, "k_key_hist's tile totals");

// tile layout: thread t owns cells [tile*4096 + 16 t, +16) — four uint4 loads, fully coalesced per warp
__device__ __forceinline__ void load_items(const uint32_t* __restrict__ count, int64_t base, int64_t M,
                                           uint32_t (&c)[kScanItems]) {
    if (base + kScanItems <= M && ((reinterpret_cast<uintptr_t>(count + base) & 15u) == 0)) {
        const uint4* p = reinterpret_cast<const uint4*>(count + base);
#pragma unroll
        for (int q = 0; q < kScanItems / 4; ++q) {
            uint4 v = p[q];
            c[4 * q] = v.x; c[4 * q + 1] = v.y; c[4 * q + 2] = v.z; c[4 * q + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int q = 0; q < kScanItems; ++q) c[q] = (base + q < M) ? count[base + q] : 0u;
    }
}

__global__ void __launch_bounds__(kScanThreads) k_scan_tile_sums(const uint32_t* __restrict__ count, int64_t M,
                                                                 uint32_t* __restrict__ tile_sums) {
    __shared__ uint32_t ws[kScanThreads / 32];
    uint32_t c[kScanItems];
    load_items(count, (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems, M, c);
    uint32_t s = 0;
#pragma unroll
    for (int q = 0; q < kScanItems; ++q) s += c[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
#pragma unroll
        for (int q = 0; q < kScanThreads / 32; ++q) t += ws[q];
        tile_sums[blockIdx.x] = t;
    }
}

// one CTA of 1024 threads: exclusive scan of the tile sums in place.  Thread t owns the contiguous
// slice [t*per, (t+1)*per): local sum, one block scan over the 1024 slice sums, local rescan —
// a single pass whatever n_tiles is (the chunked version needed n_tiles/256 dependent block scans).
constexpr int kOffThreads = 1024;
__global__ void __launch_bounds__(kOffThreads) k_scan_tile_offsets(uint32_t* tile_sums, int n_tiles) {
    __shared__ uint32_t ws[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int per = (n_tiles + kOffThreads - 1) / kOffThreads;
    const int lo = min(threadIdx.x * per, n_tiles), hi = min(lo + per, n_tiles);
    uint32_t s = 0;
    for (int i = lo; i < hi; ++i) s += tile_sums[i];
    uint32_t inc = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) ws[w] = inc;
    __syncthreads();
    if (w == 0) {
        uint32_t v = ws[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += t;
        }
        ws[lane] = v;
    }
    __syncthreads();
    uint32_t run = (w > 0 ? ws[w - 1] : 0u) + inc - s;
    for (int i = lo; i < hi; ++i) {
        const uint32_t v = tile_sums[i];
        tile_sums[i] = run;
        run += v;
    }
}

// TOTALS: tile_offsets[] holds the tiles' TOTALS (k_key_hist gathered them, <= kFuseTiles of them) and the CTA adds up
// the ones before its own itself — at most 32 KB of L2-resident reads per CTA, against one more kernel on the path.
template <bool TOTALS>
__global__ void __launch_bounds__(kScanThreads, TOTALS ? 6 : 4) k_scan_apply(const uint32_t* __restrict__ count, int64_t M,
                                                                const uint32_t* __restrict__ tile_offsets,
                                                                uint32_t* __restrict__ start, uint32_t n_gas,
                                                                unsigned int* dense_ctl, DenseItem* dense_items) {
    constexpr int kWarps = kScanThreads / 32;
    __shared__ uint32_t ws[kWarps], wv[kWarps];   // per warp: its cells' total; its share of the totals of the tiles before this one
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t c[kScanItems];
    const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    load_items(count, base, M, c);
    uint32_t v = 0;
    if (TOTALS) {
        // (16-byte loads, at most kFuseTiles / 1024 of them per thread, all in flight together with the cells' loads;
        // tile_offsets[] is 256-byte aligned and padded to a multiple of 4 words by the caller's allocation of n_tiles + 1
        // words rounded up to 256 bytes)
#pragma unroll
        for (int j = 0; j < kFuseTiles / (4 * kScanThreads); ++j) {
            const int t = 4 * (threadIdx.x + kScanThreads * j), nb = (int)blockIdx.x;
            if (t < nb) {
                const uint4 q = *reinterpret_cast<const uint4*>(tile_offsets + t);
                v += q.x + (t + 1 < nb ? q.y : 0u) + (t + 2 < nb ? q.z : 0u) + (t + 3 < nb ? q.w : 0u);
            }
        }
    }
    const uint32_t off = TOTALS ? 0u : tile_offsets[blockIdx.x];   // (every thread: the load is in flight with the cells')
    uint32_t s = 0;
#pragma unroll
    for (int q = 0; q < kScanItems; ++q) s += c[q];
    // ONE barrier: inclusive scan of s inside the warp, the warp's sum of v; then every thread adds up the (at most 8 + 8)
    // per-warp words it needs
    uint32_t inc = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 31) ws[w] = inc;
    if (lane == 0) wv[w] = v;
    __syncthreads();
    uint32_t part = lane < kWarps ? ((lane < w ? ws[lane] : 0u) + wv[lane]) : 0u;
#pragma unroll
    for (int o = kWarps / 2; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    part = __shfl_sync(0xffffffffu, part, 0);
    uint32_t run = off + part + inc - s;
    uint32_t out[kScanItems];
#pragma unroll
    for (int q = 0; q < kScanItems; ++q) {
        out[q] = run;
        run += c[q];
    }
    if (base + kScanItems <= M && ((reinterpret_cast<uintptr_t>(start + base) & 15u) == 0)) {
        uint4* p = reinterpret_cast<uint4*>(start + base);
#pragma unroll
        for (int q = 0; q < kScanItems / 4; ++q) p[q] = make_uint4(out[4 * q], out[4 * q + 1], out[4 * q + 2], out[4 * q + 3]);
    } else {
#pragma unroll
        for (int q = 0; q < kScanItems; ++q)
            if (base + q < M) start[base + q] = out[q];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) start[M] = n_gas;   // A13: start[M] = N_g
    // the densely populated cells go on the work list of sph_dense.cu (the counts are in registers here)
    if (dense_ctl && s >= (uint32_t)kDenseMin) {
#pragma unroll
        for (int q = 0; q < kScanItems; ++q)
            if (c[q] >= (uint32_t)kDenseMin) dense_append((uint32_t)(base + q), c[q], dense_ctl, dense_items);
    }
}

// ---------------------------------------------------------------- (a4) scatter and stable fix-up
__global__ void __launch_bounds__(256) k_scatter(const uint32_t* __restrict__ key, const uint32_t* __restrict__ rank_u,
                                                 const uint32_t* __restrict__ start, int n, uint32_t* __restrict__ tmp) {
    const int i0 = blockIdx.x * (256 * kPassItems) + threadIdx.x;
    uint32_t k[kPassItems], r[kPassItems], a[kPassItems];
#pragma unroll
    for (int q = 0; q < kPassItems; ++q) {
        const int i = i0 + 256 * q;
        k[q] = i < n ? key[i] : 0u;
        r[q] = i < n ? rank_u[i] : 0u;
    }
#pragma unroll
    for (int q = 0; q < kPassItems; ++q) a[q] = start[k[q]];
#pragma unroll
    for (int q = 0; q < kPassItems; ++q) {
        const int i = i0 + 256 * q;
        if (i < n) tmp[a[q] + r[q]] = (uint32_t)i;
    }
}

// slot s of the unstable order holds i = tmp[s]; its stable slot is start[k] + #{t in cell k : tmp[t] < i}.
// Consecutive threads share a cell, so the reads of tmp[a..b) are warp-broadcast / L1 hits.
// The cell number is recomputed from posm[i] (needed anyway for the reorder) instead of gathering key[i]:
// one random 32-byte sector less per particle.
__global__ void __launch_bounds__(256) k_stable(const uint32_t* __restrict__ tmp, const GridDev g,
                                                const uint32_t* __restrict__ start, const float4* __restrict__ posm,
                                                int n, uint32_t* __restrict__ perm, float4* __restrict__ posm_s) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint32_t i = tmp[s];
    const float4 p = posm[i];
    const uint32_t k = cell_key(p, g);
    const uint32_t a = start[k], b = start[k + 1];
    uint32_t r = 0, t = a;
    // tmp is 16-byte aligned (workspace carve): scalar head to a multiple of 4, uint4 body, scalar tail
    for (; t < b && (t & 3u); ++t) r += (tmp[t] < i) ? 1u : 0u;
    for (; t + 4u <= b; t += 4u) {
        const uint4 v = *reinterpret_cast<const uint4*>(tmp + t);
        r += (v.x < i ? 1u : 0u) + (v.y < i ? 1u : 0u) + (v.z < i ? 1u : 0u) + (v.w < i ? 1u : 0u);
    }
    for (; t < b; ++t) r += (tmp[t] < i) ? 1u : 0u;
    perm[a + r] = i;
    if (posm_s) posm_s[a + r] = p;
}

__global__ void __launch_bounds__(256) k_gather_pos(const float4* __restrict__ posm, const uint32_t* __restrict__ perm,
                                                    int n, float4* __restrict__ posm_s) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) posm_s[s] = posm[perm[s]];
}

int gather_sorted_pos(const float4* posm, const uint32_t* perm, int64_t n_gas, float4* posm_s, cudaStream_t st) {
    if (n_gas <= 0) return SPH_OK;
    k_gather_pos<<<(unsigned)cdiv(n_gas, 256), 256, 0, st>>>(posm, perm, (int)n_gas, posm_s);
    SPHB_LAUNCHED();
    return SPH_OK;
}

// ---------------------------------------------------------------- host side
int check_grid(const sph_grid* g, float h) {
    if (!g) return SPH_ERR_ARG;
    double m = 1.0;
    for (int a = 0; a < 3; ++a) {
        if (g->dims[a] < 1 || g->dims[a] > 4096) return SPH_ERR_GRID;
        m *= g->dims[a];
    }
    if (m >= 2147483648.0) return SPH_ERR_GRID;
    if (!(g->cell > 0.f) || !(g->inv_cell > 0.f)) return SPH_ERR_GRID;
    if (h > 0.f && g->cell < 2.0f * h) return SPH_ERR_GRID;   // 3x3x3 stencil needs cell >= 2h
    return SPH_OK;
}

GridDev to_dev(const sph_grid* g) {
    GridDev d;
    d.ox = g->origin[0]; d.oy = g->origin[1]; d.oz = g->origin[2];
    d.inv_cell = g->inv_cell;
    d.mx = g->dims[0]; d.my = g->dims[1]; d.mz = g->dims[2];
    d.fx = (float)(g->dims[0] - 1); d.fy = (float)(g->dims[1] - 1); d.fz = (float)(g->dims[2] - 1);
    return d;
}

int grid_build(const float4* posm, int64_t n_gas, const sph_grid* g, uint32_t* key, uint32_t* perm,
               uint32_t* cell_count, uint32_t* cell_start, uint32_t* rank_u, uint32_t* tmp, uint32_t* tile_sums,
               float4* posm_s, const DenseList* dense, cudaStream_t st) {
    const int64_t M = grid_cells(g);
    const int n = (int)n_gas;
    const int n_tiles = (int)cdiv(M, kScanTile);
    // Few tiles (M <= 33.5 M cells): k_scan_apply adds up the totals of the tiles before its own by itself, one kernel less
    // on the path; and where the particles are few against the cells (the galaxy grids: N_g <= M / 8) they gather the tile
    // totals themselves in k_key_hist, which drops the pass that reads count[M] only to add it up.
    const bool own_offsets = n_tiles <= kFuseTiles;
    const bool by_particles = own_offsets && (int64_t)n * 8 <= M;
    unsigned int* ctl = dense ? dense->ctl : nullptr;
    DenseItem* items = dense ? dense->items : nullptr;
    {   // K0; tile_sums[] lies right behind count[M] in a workspace (step.cu: carve): one memset then zeroes both
        const char* c_end = reinterpret_cast<const char*>(cell_count + M);
        const char* t_beg = reinterpret_cast<const char*>(tile_sums);
        const char* t_end = reinterpret_cast<const char*>(tile_sums + n_tiles);
        if (by_particles && t_beg >= c_end && t_beg - c_end < 4096) {
            SPHB_CUDA(cudaMemsetAsync(cell_count, 0, (size_t)(t_end - reinterpret_cast<const char*>(cell_count)), st));
        } else {
            SPHB_CUDA(cudaMemsetAsync(cell_count, 0, (size_t)M * sizeof(uint32_t), st));
            if (by_particles) SPHB_CUDA(cudaMemsetAsync(tile_sums, 0, (size_t)n_tiles * sizeof(uint32_t), st));
        }
    }
    {
        const int64_t batches = cdiv(n, kPassBatch), cap = (int64_t)num_sms() * 8;
        const unsigned blocks = (unsigned)(batches < 1 ? 1 : (by_particles && batches > cap ? cap : batches));
        k_key_hist<<<blocks, 256, by_particles ? (size_t)n_tiles * sizeof(uint32_t) : 0, st>>>(
            posm, n, to_dev(g), key, rank_u, cell_count, tile_sums, by_particles ? n_tiles : 0, ctl);   // K1
        SPHB_LAUNCHED();
    }
    if (!by_particles) {
        k_scan_tile_sums<<<n_tiles, kScanThreads, 0, st>>>(cell_count, M, tile_sums);          // K2 (in-block)
        SPHB_LAUNCHED();
    }
    if (own_offsets) {
        k_scan_apply<true><<<n_tiles, kScanThreads, 0, st>>>(cell_count, M, tile_sums, cell_start, (uint32_t)n, ctl, items);   // K2 (across blocks) + K3
        SPHB_LAUNCHED();
    } else {
        k_scan_tile_offsets<<<1, kOffThreads, 0, st>>>(tile_sums, n_tiles);                     // K2 (across blocks)
        SPHB_LAUNCHED();
        k_scan_apply<false><<<n_tiles, kScanThreads, 0, st>>>(cell_count, M, tile_sums, cell_start, (uint32_t)n, ctl, items);   // K3
        SPHB_LAUNCHED();
    }
    if (n > 0) {
        k_scatter<<<(unsigned)cdiv(n, 256 * kPassItems), 256, 0, st>>>(key, rank_u, cell_start, n, tmp);                 // K4
        SPHB_LAUNCHED();
        k_stable<<<(unsigned)cdiv(n, 256), 256, 0, st>>>(tmp, to_dev(g), cell_start, posm, n, perm, posm_s);
        SPHB_LAUNCHED();
    }
    return SPH_OK;
}

// ---------------------------------------------------------------- (a5) ranges
__global__ void __launch_bounds__(256) k_cell_range(const uint32_t* __restrict__ start, int64_t M,
                                                    uint2* __restrict__ range) {
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < M) range[k] = make_uint2(start[k], start[k + 1]);
}

__global__ void __launch_bounds__(256) k_particle_runs(const uint32_t* __restrict__ key,
                                                       const uint32_t* __restrict__ start, int n, int mx, int my, int mz,
                                                       uint2* __restrict__ runs) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t k = key[i];
    int ix = (int)(k % (uint32_t)mx), iy = (int)((k / (uint32_t)mx) % (uint32_t)my), iz = (int)(k / ((uint32_t)mx * my));
    int x0 = max(ix - 1, 0), x1 = min(ix + 1, mx - 1);
#pragma unroll
    for (int r = 0; r < 9; ++r) {
        int cy = iy + (r % 3) - 1, cz = iz + (r / 3) - 1;
        uint2 v = make_uint2(0u, 0u);
        if (cy >= 0 && cy < my && cz >= 0 && cz < mz) {
            int64_t row = (int64_t)mx * (cy + (int64_t)my * cz);
            v = make_uint2(start[row + x0], start[row + x1 + 1]);
        }
        runs[(size_t)i * 9 + r] = v;
    }
}

}  // namespace sphb

using namespace sphb;

extern "C" int sph_neighbour_ranges(const sph_grid* g, const uint32_t* key, const uint32_t* cell_start, int64_t n_gas,
                                    uint32_t* cell_range, uint32_t* particle_runs, void* stream) {
    if (!g || !cell_start || n_gas < 0 || n_gas >= (1ll << 31)) return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, 0.f));
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t M = grid_cells(g);
    if (cell_range) {
        k_cell_range<<<(unsigned)cdiv(M, 256), 256, 0, st>>>(cell_start, M, reinterpret_cast<uint2*>(cell_range));
        SPHB_LAUNCHED();
    }
    if (particle_runs && n_gas > 0) {
        if (!key) return SPH_ERR_ARG;
        k_particle_runs<<<(unsigned)cdiv(n_gas, 256), 256, 0, st>>>(key, cell_start, (int)n_gas, g->dims[0], g->dims[1],
                                                                    g->dims[2], reinterpret_cast<uint2*>(particle_runs));
        SPHB_LAUNCHED();
    }
    return SPH_OK;
}
