// sph_dense_dev.cuh — what the two dense-cell walks share (sph_dense.cu: hydro force, warp per target; sph_dense_rho.cu:
// density, thread per target): the slot boundaries of the 9 stencil rows of a cell, the octant bins of a staged row and
// their boxes, and the counting sort of a staged chunk by bin.  Internal to libsph_b200; nothing here is shared with
// the oracle.
#pragma once
#include "sph_dev.cuh"
#include "tma_dev.cuh"

namespace sphb {
namespace dense {

constexpr int kBins = 24;   // (sz, sy) sub-row x (cell of the row, sx): bin = (2 sz + sy) 6 + 2 c + sx — x fastest

// Row r of the stencil of cell (ix, iy, iz): the cells (ix-1, ix, ix+1) at (iy + r%3 - 1, iz + r/3 - 1) are ONE slot range
// (x-fastest cell order, L160/L203/L207); runs[4 r .. 4 r + 3] = its boundaries b0 <= b1 <= b2 <= b3 (all 0 outside the grid).
__device__ __forceinline__ void row_bounds(const uint32_t* __restrict__ start, const GridDev g, int ix, int iy, int iz, int r,
                                           uint32_t* runs) {
    const int cy = iy + (r % 3) - 1, cz = iz + (r / 3) - 1;
    uint32_t b0 = 0, b1 = 0, b2 = 0, b3 = 0;
    if (cy >= 0 && cy < g.my && cz >= 0 && cz < g.mz) {
        const uint32_t row = (uint32_t)g.mx * ((uint32_t)cy + (uint32_t)g.my * (uint32_t)cz);
        b1 = start[row + (uint32_t)ix];
        b2 = start[row + (uint32_t)ix + 1u];
        b0 = ix > 0 ? start[row + (uint32_t)ix - 1u] : b1;
        b3 = ix + 1 < g.mx ? start[row + (uint32_t)ix + 2u] : b2;
    }
    runs[4 * r] = b0;
    runs[4 * r + 1] = b1;
    runs[4 * r + 2] = b2;
    runs[4 * r + 3] = b3;
}

// mid-planes of the three cells of a row and of the row itself
struct RowGeom {
    float xm0, xm1, xm2, ym, zm;
    int cy, cz;
};
__device__ __forceinline__ RowGeom row_geom(const GridDev g, float cell, int ix, int iy, int iz, int r) {
    RowGeom q;
    q.cy = iy + (r % 3) - 1;
    q.cz = iz + (r / 3) - 1;
    q.xm0 = fmaf((float)(ix - 1) + 0.5f, cell, g.ox);
    q.xm1 = q.xm0 + cell;
    q.xm2 = q.xm1 + cell;
    q.ym = fmaf((float)q.cy + 0.5f, cell, g.oy);
    q.zm = fmaf((float)q.cz + 0.5f, cell, g.oz);
    return q;
}

// bin of the candidate in slot `slot` of the row (b1, b2: where the cells ix and ix+1 start)
__device__ __forceinline__ uint32_t bin_of(const float4 p, uint32_t slot, uint32_t b1, uint32_t b2, const RowGeom& q) {
    const uint32_t c = (slot >= b1 ? 1u : 0u) + (slot >= b2 ? 1u : 0u);
    const float xm = c == 0u ? q.xm0 : (c == 1u ? q.xm1 : q.xm2);
    return ((p.z >= q.zm ? 2u : 0u) + (p.y >= q.ym ? 1u : 0u)) * 6u + 2u * c + (p.x >= xm ? 1u : 0u);
}

// Box of bin bb: the octant, pulled out by eps = 2^-8 cell (the rounding of the cell assignment, A7, and of the faces);
// open-ended on the outside of a boundary cell, where the particles clamped into the grid sit; out of reach altogether
// where the row has no such cell.  (xl, xh, yl, yh), (zl, zh, -, -).
__device__ __forceinline__ void bin_box(int bb, const GridDev g, float cell, int ix, const RowGeom& q, float4& b0, float4& b1) {
    const float eps = cell * 0.00390625f, half = 0.5f * cell, big = 3.0e38f;
    const int k = bb % 6, sr = bb / 6, c = k >> 1, sx = k & 1, sy = sr & 1, sz = sr >> 1;
    const int cx = ix - 1 + c;
    const float xm = c == 0 ? q.xm0 : (c == 1 ? q.xm1 : q.xm2);
    float xl = (sx ? xm : xm - half) - eps, xh = (sx ? xm + half : xm) + eps;
    float yl = (sy ? q.ym : q.ym - half) - eps, yh = (sy ? q.ym + half : q.ym) + eps;
    float zl = (sz ? q.zm : q.zm - half) - eps, zh = (sz ? q.zm + half : q.zm) + eps;
    if (cx == 0 && !sx) xl = -big;
    if (cx == g.mx - 1 && sx) xh = big;
    if (cx < 0 || cx >= g.mx) xl = big;   // no such cell (the row ends here)
    if (q.cy <= 0 && !sy) yl = -big;
    if (q.cy >= g.my - 1 && sy) yh = big;
    if (q.cz <= 0 && !sz) zl = -big;
    if (q.cz >= g.mz - 1 && sz) zh = big;
    b0 = make_float4(xl, xh, yl, yh);
    b1 = make_float4(zl, zh, 0.f, 0.f);
}

// Stable counting sort of a staged chunk by bin (slot order inside a bin), all THREADS threads of the CTA:
//   raw[roff + i], i < ncand, is the candidate of slot cs + i;  move(src raw index, dst sorted index, bin) copies its payload;
//   bstart[b] = first sorted index of bin b (bstart[24..31] = ncand);  box[2 b], box[2 b + 1] = the bins' boxes.
// hist: [ROUNDS][THREADS/32][kBins] words, ZERO on entry (the caller zeroes it once, each call leaves it zeroed).  `wait` is
// called first (the bulk copy's mbarrier), `extra` by one thread between the barriers (per-chunk resets of the caller).  PAD_EVEN: every bin starts at
// an even sorted index — a bin of odd population is followed by one filler slot, which pad(dst) fills (a caller that
// reads the sorted chunk two slots at a time).  Ends with a barrier: the sorted chunk is complete and the landing zone
// is free.
template <int THREADS, int ROUNDS, bool PAD_EVEN, class Wait, class Extra, class Move, class Pad>
__device__ __forceinline__ void bin_chunk(const float4* r_pos, uint32_t roff, uint32_t ncand, uint32_t cs, uint32_t b1,
                                          uint32_t b2, const GridDev g, float cell, int ix, const RowGeom& q, uint32_t* hist,
                                          uint32_t* bstart, float4* box, Wait&& wait, Extra&& extra, Move&& move, Pad&& pad) {
    constexpr int WARPS = THREADS / 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    wait();   // (every thread waits for the copy itself; the histogram was zeroed before the last barrier of the previous call)
    uint32_t my_bin[ROUNDS], my_rank[ROUNDS];
#pragma unroll
    for (int rd = 0; rd < ROUNDS; ++rd) {
        const uint32_t i = (uint32_t)(rd * THREADS + tid);
        uint32_t bin = 31u;   // past the end of the chunk
        if (i < ncand) bin = bin_of(r_pos[roff + i], cs + i, b1, b2, q);
        const unsigned peers = __match_any_sync(0xffffffffu, bin);
        my_bin[rd] = bin;
        my_rank[rd] = __popc(peers & lt_mask);
        if (bin < (uint32_t)kBins && my_rank[rd] == 0u) hist[(rd * WARPS + warp) * kBins + bin] = __popc(peers);
    }
    __syncthreads();   // counts complete; every warp is past the previous chunk's candidates
    if (tid < 32) {
        // lane b: exclusive prefix of bin b over (round, warp), then the bins' starts
        // (all the loads first: the other warps wait at the barrier below for this one)
        uint32_t run = 0u;
        if (lane < kBins) {
            uint32_t v[ROUNDS * WARPS];
#pragma unroll
            for (int j = 0; j < ROUNDS * WARPS; ++j) v[j] = hist[j * kBins + lane];
#pragma unroll
            for (int j = 0; j < ROUNDS * WARPS; ++j) {
                hist[j * kBins + lane] = run;
                run += v[j];
            }
        }
        const uint32_t len = PAD_EVEN ? (run + 1u) & ~1u : run;
        uint32_t inc = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += v;
        }
        bstart[lane] = inc - len;   // lanes >= kBins: the end of the sorted chunk
        if (PAD_EVEN && len != run) pad(inc - 1u);
        if (lane == 0) extra();
    }
    if (tid >= 32 && tid < 32 + kBins) {   // warp 1, after the barrier above: no warp still reads the previous chunk's boxes
        float4 b0, b1_;
        bin_box(tid - 32, g, cell, ix, q, b0, b1_);
        box[2 * (tid - 32)] = b0;
        box[2 * (tid - 32) + 1] = b1_;
    }
    __syncthreads();
#pragma unroll
    for (int rd = 0; rd < ROUNDS; ++rd) {
        const uint32_t i = (uint32_t)(rd * THREADS + tid);
        if (i < ncand) move(roff + i, bstart[my_bin[rd]] + hist[(rd * WARPS + warp) * kBins + my_bin[rd]] + my_rank[rd], my_bin[rd]);
    }
    __syncwarp();
    // zero the histogram for the next call: a warp reads only its own rows of it above
#pragma unroll
    for (int rd = 0; rd < ROUNDS; ++rd)
        if (lane < kBins) hist[(rd * WARPS + warp) * kBins + lane] = 0u;
    __syncthreads();   // the sorted chunk is complete, the landing zone is free
}

// The reachable bins of a target, in bin order, are its candidate list: flat position v = 0 .. T-1.  Along a (sz, sy)
// sub-row the distance to the 6 x-slabs falls and rises once, so the reachable bins of a sub-row are consecutive: one
// slot range per sub-row, from its first to its last reachable bin (if a bin in between were out of reach after all,
// testing its candidates costs time, not correctness).  A range is described by the flat position where it ends and
// the offset from a flat position to a slot, both in BYTES of the float4 array (x16), so a candidate's address is one
// add.  `reach`: bit b set = bin b reachable (a ballot: uniform); bstart: the bins' starts inside the segment, which
// begins at sorted index `first`.  All lanes compute the same four ranges: bit operations and 8 broadcast loads.
struct Groups {
    uint2 g0, g1, g2, g3;
    uint32_t T;
};
__device__ __forceinline__ Groups candidate_groups(unsigned reach, const uint32_t* bstart, uint32_t first) {
    Groups G;
    uint32_t end = 0;
    uint2* g[4] = {&G.g0, &G.g1, &G.g2, &G.g3};
#pragma unroll
    for (int sr = 0; sr < 4; ++sr) {
        const unsigned m6 = (reach >> (6 * sr)) & 63u;
        uint32_t lo = 0, hi = 0;
        if (m6) {
            lo = bstart[6 * sr + __ffs(m6) - 1];
            hi = bstart[6 * sr + 32 - __clz(m6)];
        }
        const uint32_t off = first + lo - end;   // flat position end .. end + (hi - lo) -> slots first + lo ..
        end += hi - lo;
        *g[sr] = make_uint2(16u * end, 16u * off);
    }
    G.T = end;
    return G;
}
// flat position (x16) -> byte offset of the candidate in the sorted float4 array
__device__ __forceinline__ uint32_t candidate_offset(const Groups& G, uint32_t v16) {
    uint32_t rel = v16 + G.g3.y;
    rel = v16 < G.g2.x ? v16 + G.g2.y : rel;
    rel = v16 < G.g1.x ? v16 + G.g1.y : rel;
    rel = v16 < G.g0.x ? v16 + G.g0.y : rel;
    return rel;
}

}  // namespace dense
}  // namespace sphb
