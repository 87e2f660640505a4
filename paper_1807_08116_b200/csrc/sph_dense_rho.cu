// sph_dense_rho.cu — (a7) density, Eq. 7-8, for DENSELY populated cells (>= kDenseMin particles per cell).
//
// The density pair term is ~15 instructions: nothing is won by compacting accepted pairs (the warp-per-target walk of
// sph_dense.cu, tried on the density, lost to the thread-per-slot walk); the cost is the NUMBER of candidates tested —
// all 27 cells of the stencil, 6 per neighbour — and the instructions per test.  Per work item (one cell, <= 384 targets):
//   * the item's targets are ordered by the octant of their cell they lie in, so a group of 8 consecutive targets covers
//     one or two octants and has a small bounding box;
//   * each stencil row is staged by TMA bulk copies and re-ordered by octant bin in shared memory (sph_dense_dev.cuh), as
//     for the forces — positions only, and written as PAIRS (x0,x1,y0,y1)(z0,z1,m0,m1), every bin padded to an even
//     number of slots, for the packed arithmetic below;
//   * a work unit is one group of 8 targets on one warp, 4 lanes per target: the warp tests the bins against the GROUP's
//     bounding box — lane b the box of bin b — and walks only the reachable ones (~65 % of the stencil; 83 % for a group
//     of 32, 39 % for a single target, 100 % without bins); the 4 lanes of a target take the candidate pairs of a range
//     in turn, so a warp reads 4 consecutive pairs per step — two LDS.128 of 4 distinct addresses, no bank conflict — and
//     the 4 partial sums are added by two shuffles in a fixed order.  (2 and 8 lanes per target measured slower: 23.0
//     and 26.2 ms against 20.9 at config 4.)
//   * the arithmetic of a pair of candidates is packed FP32 (sub/mul/fma.f32x2, as in the gravity kernels): 14 packed
//     operations + 2 MUFU.SQRT + 4 FMNMX + 2 LDS.128 + 3 of loop control for two candidates — 25 instructions per step
//     of 64 lane tests; the loop is issue-bound, and packing halves the slots;
//   * a CTA's 12 warps draw the units of a chunk from a counter; a target's running sum lives in shared memory between
//     chunks and is touched by one warp per chunk, in chunk order.
// Kernel value: W = 1/4 (2 - xi)_+^3 - (1 - xi)_+^3 with xi from MUFU.SQRT (sph_dev.cuh), d2 formed by the same mul, fma,
// fma as everywhere; the clamped cubes stand in for the cutoff test (see the loop).  Fixed order: bitwise reproducible.
#include "sph_dense_dev.cuh"
#include "grav_dev.cuh"   // the packed-FP32 helpers pk2 / upk2 / fma2 / mul2 / sub2

namespace sphb {

namespace {

using dense::kBins;
constexpr int kRhoThreads = 384;
constexpr int kRhoWarps = kRhoThreads / 32;
constexpr int kRhoCtasPerSm = 3;
constexpr int kRhoTT = 3 * kDenseTT;                        // targets per item: three consecutive entries of the work list
constexpr int kRhoL = 4;                                    // lanes per target: each takes every kRhoL-th candidate pair
constexpr int kRhoG = 32 / kRhoL;                           // targets per work unit (one warp)
constexpr int kRhoK = 1152;                                 // candidate slots per staged chunk
constexpr int kRhoKS = kRhoK + kBins;                       // sorted: + one filler per bin at most
static_assert(kRhoTT == kRhoThreads, "a thread per target of the item");
constexpr int kRhoRounds = (kRhoK + kRhoThreads - 1) / kRhoThreads;

// VARH (per-particle smoothing lengths, L82): the pairs also carry (h0, h1), every bin its largest length, every target
// its own and every group of targets its largest
template <bool VARH>
struct RhoLayout {
    static constexpr int raw_pos = 0;                                   // float4 [K]     landing zone of the bulk copies
    static constexpr int pk = raw_pos + kRhoK * 16;                     // float4 [KS/2][2] the chunk in bin order, as pairs
    static constexpr int hp = pk + kRhoKS * 16;                         // float2 [KS/2]  VARH: the pairs' lengths
    static constexpr int th = hp + (VARH ? kRhoKS * 4 : 0);             // float [TT]     VARH: the targets' lengths, octant order
    static constexpr int hmax = th + (VARH ? kRhoTT * 4 : 0);           // uint32 [32]    VARH: bits of the largest length in bin b
    static constexpr int tpos = hmax + (VARH ? 32 * 4 : 0);             // float4 [TT]    the item's targets in octant order
    static constexpr int tslot = tpos + kRhoTT * 16;                    // uint32 [TT]    their sorted slots
    static constexpr int part = tslot + kRhoTT * 4;                     // float [TT]     the targets' running sums
    static constexpr int bbox = part + kRhoTT * 4;                      // float [TT/G][8] bounding boxes of the target groups
    static constexpr int runs = bbox + (kRhoTT / kRhoG) * 32;           // uint32 [9][4]
    static constexpr int hist = runs + 9 * 4 * 4;                       // uint32 [rounds][warps][bins]
    static constexpr int bstart = hist + kRhoRounds * kRhoWarps * kBins * 4;   // uint32 [32]
    static constexpr int box = bstart + 32 * 4;                         // float4 [bins][2]
    static constexpr int ocnt = box + kBins * 32;                       // uint32 [warps][8] octant counts
    static constexpr int bar = ocnt + kRhoWarps * 8 * 4;                // uint64
    static constexpr int item = bar + 8;                                // uint32
    static constexpr int unext = bar + 12;                              // uint32: next work unit of the chunk
    static constexpr int bytes = bar + 16;
};
static_assert((RhoLayout<false>::bytes + 1024) * kRhoCtasPerSm <= 227 * 1024, "shared memory per SM");
static_assert((RhoLayout<true>::bytes + 1024) * kRhoCtasPerSm <= 227 * 1024, "shared memory per SM");

// VARH: W(|dr| / h_ij, h_ij) with h_ij = (h_i + h_j)/2 carries its own 1/(pi h_ij^3) (readings A24-A26 as in
// k_density<true>); norm is then 8/pi (1/h_ij^3 = 8/(h_i + h_j)^3).  A group's sphere reaches a bin iff the distance of
// the boxes is below (the group's largest length) + (the bin's largest length) — the paper's hmaxCell (L164, L207) at the
// granularity of the octant bins.
template <bool VARH>
__global__ void __launch_bounds__(kRhoThreads, kRhoCtasPerSm)
    k_dense_density(const float4* __restrict__ posm_s, const float* __restrict__ h_s, const uint32_t* __restrict__ perm,
                    const uint32_t* __restrict__ start, GridDev g, float cell, float rc2, float neg_inv_h, float norm, Shard sh,
                    unsigned int* __restrict__ ctl, const DenseItem* __restrict__ items, float* __restrict__ rho) {
    using L = RhoLayout<VARH>;
    extern __shared__ __align__(128) unsigned char smem[];
    float4* r_pos = reinterpret_cast<float4*>(smem + L::raw_pos);
    float* c_pk = reinterpret_cast<float*>(smem + L::pk);
    float* c_hp = reinterpret_cast<float*>(smem + L::hp);
    float* t_h = reinterpret_cast<float*>(smem + L::th);
    uint32_t* s_hmax = reinterpret_cast<uint32_t*>(smem + L::hmax);
    float4* t_pos = reinterpret_cast<float4*>(smem + L::tpos);
    uint32_t* t_slot = reinterpret_cast<uint32_t*>(smem + L::tslot);
    float* s_part = reinterpret_cast<float*>(smem + L::part);
    float4* s_bbox = reinterpret_cast<float4*>(smem + L::bbox);
    uint32_t* s_runs = reinterpret_cast<uint32_t*>(smem + L::runs);
    uint32_t* s_hist = reinterpret_cast<uint32_t*>(smem + L::hist);
    uint32_t* s_bstart = reinterpret_cast<uint32_t*>(smem + L::bstart);
    float4* s_box = reinterpret_cast<float4*>(smem + L::box);
    uint32_t* s_ocnt = reinterpret_cast<uint32_t*>(smem + L::ocnt);
    uint64_t* s_bar = reinterpret_cast<uint64_t*>(smem + L::bar);
    uint32_t* s_item = reinterpret_cast<uint32_t*>(smem + L::item);
    uint32_t* s_unext = reinterpret_cast<uint32_t*>(smem + L::unext);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    const uint32_t sbase = smem_u32(smem);
    const uint32_t a_pk = sbase + L::pk;
    const uint32_t a_hp_pk = sbase + L::hp - (a_pk >> 2);   // a pair at byte address pa of the pk array has its lengths at a_hp_pk + pa / 4
    const uint32_t sub = (uint32_t)lane % kRhoL, tl = (uint32_t)lane / kRhoL;   // this lane's share and target within a unit
    const uint32_t n_items = ctl[0];
    if (blockIdx.x >= n_items) return;   // uniform per CTA
    if (tid == 0) {
        mbar_init(s_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < kRhoRounds * kRhoWarps * kBins; i += kRhoThreads) s_hist[i] = 0u;   // dense::bin_chunk keeps it zeroed
    uint32_t n_staged = 0;
    const float big = 3.0e38f;
    const u64 ninvh2 = pk2(neg_inv_h, neg_inv_h), two2 = pk2(2.0f, 2.0f), one2 = pk2(1.0f, 1.0f), q25 = pk2(0.25f, 0.25f);

    auto issue = [&](uint32_t cs, uint32_t ce) {   // positions only: 16-byte slots, no alignment padding needed
        mbar_expect_tx(s_bar, (ce - cs) * 16u);
        bulk_g2s(r_pos, posm_s + cs, (ce - cs) * 16u, s_bar);
    };
    auto skip_empty = [&](int& r, uint32_t& cs) {
        while (r < 9 && s_runs[4 * r] >= s_runs[4 * r + 3]) ++r;
        if (r < 9) cs = s_runs[4 * r];
    };
    auto next_chunk = [&](int& r, uint32_t& cs) {
        cs += kRhoK;
        if (cs >= s_runs[4 * r + 3]) {
            ++r;
            skip_empty(r, cs);
        }
    };

    for (;;) {
        __syncthreads();   // the previous item's shared memory is no longer read
        if (tid == 0) *s_item = atomicAdd(ctl + 1, 1u);   // items from a counter (zeroed before the launch)
        __syncthreads();
        const uint32_t item = *s_item;
        if (item >= n_items) break;
        const DenseItem it = items[item];
        if (it.chunk % 3u != 0u) continue;   // an item here is three entries of the list: kRhoTT targets of the cell
        const uint32_t mx = (uint32_t)g.mx, my = (uint32_t)g.my;
        const int ix = (int)(it.key % mx), iy = (int)((it.key / mx) % my), iz = (int)(it.key / (mx * my));
        const uint32_t ts = start[it.key] + it.chunk * kDenseTT;
        if (!sh.owns(ts)) continue;   // another rank's targets (common.cuh: Shard)
        const uint32_t nt = min(start[it.key + 1u] - ts, (uint32_t)kRhoTT);
        if (tid < 9) dense::row_bounds(start, g, ix, iy, iz, tid, s_runs);

        // ---- the item's targets into octant order (stable): a warp of 32 then covers one or two octants ----
        float4 mine = make_float4(big, big, big, 0.f);
        float mine_h = 0.f;
        uint32_t oct = 8u;
        if ((uint32_t)tid < nt) {
            mine = posm_s[ts + tid];
            if (VARH) mine_h = h_s[ts + tid];
            const float xm = fmaf((float)ix + 0.5f, cell, g.ox), ym = fmaf((float)iy + 0.5f, cell, g.oy),
                        zm = fmaf((float)iz + 0.5f, cell, g.oz);
            oct = (mine.x >= xm ? 1u : 0u) + (mine.y >= ym ? 2u : 0u) + (mine.z >= zm ? 4u : 0u);
        }
        const unsigned opeers = __match_any_sync(0xffffffffu, oct);
        const uint32_t orank = __popc(opeers & lt_mask);
        if (lane < 8) s_ocnt[warp * 8 + lane] = 0u;
        __syncwarp();
        if (oct < 8u && orank == 0u) s_ocnt[warp * 8 + oct] = __popc(opeers);
        for (int i = tid; i < kRhoTT; i += kRhoThreads) s_part[i] = 0.f;
        __syncthreads();
        if (oct < 8u) {
            uint32_t dst = orank;
            for (uint32_t o = 0; o <= oct; ++o)
                for (int w = 0; w < kRhoWarps; ++w)
                    if (o < oct || w < warp) dst += s_ocnt[w * 8 + o];
            t_pos[dst] = mine;
            t_slot[dst] = ts + (uint32_t)tid;
            if (VARH) t_h[dst] = mine_h;
        }
        __syncthreads();
        // bounding box of every group of kRhoG consecutive targets (the threads' targets: kRhoTT == kRhoThreads)
        if ((uint32_t)(warp * 32) < nt) {
            const uint32_t t = (uint32_t)(warp * 32 + lane);
            const bool has = t < nt;
            const float4 p = has ? t_pos[t] : make_float4(0.f, 0.f, 0.f, 0.f);
            float lo[3] = {has ? p.x : big, has ? p.y : big, has ? p.z : big};
            float hi[3] = {has ? p.x : -big, has ? p.y : -big, has ? p.z : -big};
            float hg = (VARH && has) ? t_h[t] : 0.f;   // the group's largest length
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int o = kRhoG / 2; o > 0; o >>= 1) {
                    lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
                    hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
                }
            if (VARH) {
#pragma unroll
                for (int o = kRhoG / 2; o > 0; o >>= 1) hg = fmaxf(hg, __shfl_xor_sync(0xffffffffu, hg, o));
            }
            if (lane % kRhoG == 0) {
                s_bbox[2 * (t / kRhoG)] = make_float4(lo[0], hi[0], lo[1], hi[1]);
                s_bbox[2 * (t / kRhoG) + 1] = make_float4(lo[2], hi[2], hg, 0.f);
            }
        }
        __syncthreads();
        const uint32_t n_units = (nt + kRhoG - 1u) / kRhoG;   // unit u: targets u kRhoG .. u kRhoG + kRhoG - 1

        int r = 0;
        uint32_t cs = 0;
        skip_empty(r, cs);
        if (tid == 0 && r < 9) issue(cs, min(cs + kRhoK, s_runs[4 * r + 3]));
        while (r < 9) {
            const uint32_t ce = min(cs + kRhoK, s_runs[4 * r + 3]);
            const uint32_t ncand = ce - cs;
            const uint32_t b1 = s_runs[4 * r + 1], b2 = s_runs[4 * r + 2];
            const dense::RowGeom rg = dense::row_geom(g, cell, ix, iy, iz, r);
            // sorted slot d -> pair d / 2, half d % 2 of (x0, x1, y0, y1), (z0, z1, m0, m1)
            auto put = [&](uint32_t d, const float4 p) {
                float* q = c_pk + (size_t)(d >> 1) * 8u + (d & 1u);
                q[0] = p.x;
                q[2] = p.y;
                q[4] = p.z;
                q[6] = p.w;
            };
            dense::bin_chunk<kRhoThreads, kRhoRounds, true>(
                r_pos, 0u, ncand, cs, b1, b2, g, cell, ix, rg, s_hist, s_bstart, s_box,
                [&]() {
                    mbar_wait(s_bar, n_staged & 1u);
                    ++n_staged;
                },
                [&]() {   // one thread, after every warp has left the previous chunk and before the moves
                    *s_unext = 0u;
                    if (VARH) {
#pragma unroll
                        for (int bq = 0; bq < 32; ++bq) s_hmax[bq] = 0u;
                    }
                },
                [&](uint32_t src, uint32_t dst, uint32_t bin) {
                    put(dst, r_pos[src]);
                    if (VARH) {   // the length straight from global memory (L2), and the bin's largest (positive floats order like their bits)
                        const float hj = h_s[cs + src];
                        c_hp[dst] = hj;
                        atomicMax(s_hmax + bin, __float_as_uint(hj));
                    }
                },
                [&](uint32_t dst) {   // a filler: out of reach, no mass
                    put(dst, make_float4(big, big, big, 0.f));
                    if (VARH) c_hp[dst] = 1.0f;
                });
            int rn = r;
            uint32_t csn = cs;
            next_chunk(rn, csn);
            if (tid == 0 && rn < 9) issue(csn, min(csn + kRhoK, s_runs[4 * rn + 3]));

            const float4 bx0 = lane < kBins ? s_box[2 * lane] : make_float4(big, big, big, big);
            const float4 bx1 = lane < kBins ? s_box[2 * lane + 1] : make_float4(big, big, 0.f, 0.f);
            // units are handed to the warps from a counter (their work differs with the group's position in the cell); a
            // target's sum is touched by one warp per chunk, chunk after chunk in a fixed order
            for (;;) {
                uint32_t u = 0;
                if (lane == 0) u = atomicAdd(s_unext, 1u);
                u = __shfl_sync(0xffffffffu, u, 0);
                if (u >= n_units) break;
                // lane b: can any target of the group reach bin b?  distance between the two boxes, a lower bound
                const float4 w0 = s_bbox[2 * u], w1 = s_bbox[2 * u + 1];   // (xlo, xhi, ylo, yhi), (zlo, zhi)
                const float ex = fmaxf(fmaxf(bx0.x - w0.y, w0.x - bx0.y), 0.f);
                const float ey = fmaxf(fmaxf(bx0.z - w0.w, w0.z - bx0.w), 0.f);
                const float ez = fmaxf(fmaxf(bx1.x - w1.y, w1.x - bx1.y), 0.f);
                float rcb2 = rc2;
                if (VARH) {
                    const float rcb = w1.z + __uint_as_float(s_hmax[lane]);
                    rcb2 = rcb * rcb;
                }
                const bool reach_b = fmaf(ez, ez, fmaf(ey, ey, ex * ex)) < rcb2;
                const unsigned reach = __ballot_sync(0xffffffffu, reach_b) & ((1u << kBins) - 1u);
                if (reach == 0u) continue;
                const uint32_t t = u * kRhoG + tl;
                const float4 pi = t < nt ? t_pos[t] : make_float4(big, big, big, 0.f);
                const u64 xi = pk2(pi.x, pi.x), yi = pk2(pi.y, pi.y), zi = pk2(pi.z, pi.z);
                const float h_i = (VARH && t < nt) ? t_h[t] : 1.0f;
                const u64 hi2 = pk2(h_i, h_i), m2 = pk2(-2.0f, -2.0f);
                u64 sum2 = 0ull;   // includes the self term m_i W(0): j = i passes the predicate with d2 = 0 (A5)
                // one range of pairs per (sz, sy) sub-row, from its first to its last reachable bin (sph_dense_dev.cuh);
                // the kRhoL lanes of a target take the pairs of a range in turn
#pragma unroll
                for (int sr = 0; sr < 4; ++sr) {
                    const unsigned m6 = (reach >> (6 * sr)) & 63u;
                    if (m6 == 0u) continue;   // uniform
                    // byte addresses of the pairs: sorted slot d is in pair d / 2 (every bin starts even), 32 bytes a pair
                    const uint32_t hi = a_pk + 16u * s_bstart[6 * sr + 32 - __clz(m6)];
                    for (uint32_t pa = a_pk + 16u * s_bstart[6 * sr + __ffs(m6) - 1] + 32u * sub; pa < hi; pa += 32u * kRhoL) {
                        const float4 A = lds_f4(pa), B = lds_f4(pa + 16u);
                        const u64 dx = sub2(xi, pk2(A.x, A.y)), dy = sub2(yi, pk2(A.z, A.w)), dz = sub2(zi, pk2(B.x, B.y));
                        const u64 d2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));   // per half: the mul, fma, fma of the cutoff (A8)
                        float d2a, d2b;
                        upk2(d2, d2a, d2b);
                        const u64 rr = pk2(sqrt_approx(d2a), sqrt_approx(d2b));
                        float a0, a1, c0, c1;
                        u64 rh = 0ull;   // VARH: 1 / (h_i + h_j) = 1 / (2 h_ij)
                        if (VARH) {
                            const float2 H = lds_f2(a_hp_pk + (pa >> 2));
                            float s0_, s1_;
                            upk2(add2(hi2, pk2(H.x, H.y)), s0_, s1_);
                            rh = pk2(rcp_approx(s0_), rcp_approx(s1_));
                            const u64 t2 = mul2(rr, rh);            // xi / 2
                            upk2(fma2(t2, m2, two2), a0, a1);       // 2 - xi
                            upk2(fma2(t2, m2, one2), c0, c1);       // 1 - xi
                        } else {
                            upk2(fma2(rr, ninvh2, two2), a0, a1);   // 2 - xi
                            upk2(fma2(rr, ninvh2, one2), c0, c1);   // 1 - xi
                        }
                        const u64 a = pk2(fmaxf(a0, 0.f), fmaxf(a1, 0.f)), c = pk2(fmaxf(c0, 0.f), fmaxf(c1, 0.f));
                        const u64 c3 = mul2(mul2(c, c), c);
                        const u64 w = sub2(mul2(mul2(mul2(a, a), a), q25), c3);   // 1/4 (2 - xi)_+^3 - (1 - xi)_+^3
                        // no test of the cutoff: beyond 2h the clamped cubes are 0, and where the rounding of MUFU.SQRT and of the
                        // fma puts 2 - xi on the other side of 0 than d2 < fl(fl(2h)^2) (A8), the term is <= (2^-22)^3 / 4 of the
                        // self term m_i W(0) that every sum holds: it does not reach the sum's last bit
                        if (VARH)
                            sum2 = fma2(mul2(pk2(B.z, B.w), mul2(mul2(rh, rh), rh)), w, sum2);   // m_j W / (h_i + h_j)^3; 8/pi at the end
                        else
                            sum2 = fma2(pk2(B.z, B.w), w, sum2);
                    }
                }
                float s0, s1;
                upk2(sum2, s0, s1);
                float sum = s0 + s1;
#pragma unroll
                for (int o = kRhoL / 2; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
                if (sub == 0u && t < nt) s_part[t] += sum;
            }
            r = rn;
            cs = csn;
            // the barrier after the wait at the top of the next chunk's sort (or the one below) separates this chunk's
            // reads of the sorted tile from the next re-ordering
        }
        __syncthreads();
        if ((uint32_t)tid < nt) {
            rho[perm[t_slot[tid]]] = s_part[tid] * norm;
        }
    }
}

}  // namespace

int density_dense(const float4* posm_s, const float* h_s /*cell order, or NULL*/, const uint32_t* perm, const uint32_t* cell_start,
                  const sph_params* p, const sph_grid* g, const DenseList& dl, float* rho, cudaStream_t st, Shard sh) {
    int dev = 0;
    SPHB_CUDA(cudaGetDevice(&dev));
    static std::atomic<bool> opted[64];   // per device: the dynamic shared-memory opt-in
    if (dev < 0 || dev >= 64) return SPH_ERR_UNSUPPORTED;
    if (!opted[dev].load(std::memory_order_acquire)) {
        SPHB_CUDA(cudaFuncSetAttribute(k_dense_density<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, RhoLayout<false>::bytes));
        SPHB_CUDA(cudaFuncSetAttribute(k_dense_density<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, RhoLayout<true>::bytes));
        opted[dev].store(true, std::memory_order_release);
    }
    const float two_h = 2.0f * p->h;
    SPHB_CUDA(cudaMemsetAsync(dl.ctl + 1, 0, sizeof(unsigned int), st));   // the item counter
    const unsigned grid = (unsigned)(kRhoCtasPerSm * num_sms());
    if (h_s) {
        k_dense_density<true><<<grid, kRhoThreads, RhoLayout<true>::bytes, st>>>(
            posm_s, h_s, perm, cell_start, to_dev(g), 1.0f / g->inv_cell, two_h * two_h, 0.f, (float)(8.0 / 3.14159265358979323846), sh,
            dl.ctl, dl.items, rho);
    } else {
        const float norm = (float)(1.0 / (3.14159265358979323846 * (double)p->h * (double)p->h * (double)p->h));
        k_dense_density<false><<<grid, kRhoThreads, RhoLayout<false>::bytes, st>>>(
            posm_s, nullptr, perm, cell_start, to_dev(g), 1.0f / g->inv_cell, two_h * two_h, -(1.0f / p->h), norm, sh, dl.ctl, dl.items, rho);
    }
    SPHB_LAUNCHED();
    return SPH_OK;
}

}  // namespace sphb
