// sph_dense.cu — (a9) hydro force / energy rate for DENSELY populated cells (>= kDenseMin particles per cell).
//
// The thread-per-slot walk of sph.cu suits the sparse galaxy grids (a handful of neighbours, latency bound).  In a
// clump (config 4: up to ~570 particles per cell, ~2000 neighbours, one candidate in five to six accepted) its
// ~100-instruction pair term runs at 14 active lanes per instruction and waits on global gathers.  Here, per work item
// (one cell, <= kDenseTT targets):
//   * the candidates of each of the 9 stencil rows — ONE contiguous slot range per row, which is what the x-fastest cell
//     order buys (L160, L203, L207) — are staged in shared memory by TMA bulk copies (cp.async.bulk + mbarrier), in
//     chunks of kDenseK slots, once for all the item's targets; a chunk holds a piece of one row or, where the rows are
//     short, several whole rows (a target's queue of accepted pairs and its partial sums then live across them, and the
//     per-chunk costs are paid once); the copy of the next chunk runs under the work on this one;
//   * the CTA re-orders each staged chunk in shared memory by SUB-CELL (a stable counting sort over 24 bins: the
//     three cells of the row x 2x2x2 octants, x fastest), so that the candidates a target can reach are a few contiguous
//     ranges: a 2h sphere meets ~84 octants of h^3 against the 27 x 8 = 216 of the whole stencil — 2.6 candidates per
//     neighbour instead of 6.  The order is internal to this kernel: the exported keys / perm (A7, A16) are untouched;
//   * a WARP takes a target: lane b finds out whether the sphere reaches bin b (distance to the octant's box, pulled out
//     by eps and open-ended on the outside of boundary cells, where clamped particles sit); the reachable bins, in bin
//     order, are the target's candidate list, addressed by a flat position through at most four slot ranges, so the 32
//     lanes test 64 candidates per step (two per lane) with every lane busy whatever the bins' sizes;
//   * accepted candidates are compacted by ballot + popc into a per-warp ring queue and the pair term (sph_dev.cuh:
//     hydro_pair_fast; hydro_pair_h with per-particle lengths) runs on full warps, its operands read from the staged tile;
//   * a lane's partial sum over one chunk (<= kDenseK/32 candidates) is plain FP32; the 32 partials are added across the
//     warp in FP64 (one butterfly for the four sums) and accumulated per target in FP64 shared memory, so a target's sum
//     has a fixed order (bitwise reproducible) and is at least as accurate as the compensated FP32 sum of the sparse walk.
// Work items come from the list the grid build writes (grid.cu: k_scan_apply) — or k_dense_list for the stand-alone
// calls — and are drawn from a counter by a persistent grid (kDenseCtasPerSm CTAs per SM).
// The density pass (a7) of these cells is sph_dense_rho.cu: the same staging and binning, but four lanes per target and
// no compaction — its pair term is ~15 instructions.
#include <type_traits>
#include "sph_dense_dev.cuh"

namespace sphb {

namespace {

constexpr int kDenseThreads = 384;
constexpr int kDenseWarps = kDenseThreads / 32;
constexpr int kDenseCtasPerSm = 2;
constexpr int kMaxSeg = 6;                // pieces of stencil rows ("segments") a chunk may hold
using dense::kBins;
constexpr int kQueue = 128;               // ring queue entries per warp: <= 31 left over + 64 pushed by a step

// VARH (per-particle smoothing lengths, L82): the sorted chunk also holds the candidates' lengths and every bin its
// largest one, so the chunk is a little smaller
template <bool VARH>
struct DenseLayout {
    static constexpr int kDenseK = VARH ? 992 : 1088;                   // candidate slots per staged chunk
    static constexpr int kDenseKS = kDenseK + 2 * kMaxSeg;              // + the even-slot alignment of the float2 array, per segment
    static constexpr int kRounds = (kDenseK + kDenseThreads - 1) / kDenseThreads;
    // byte offsets inside the dynamic shared memory block (all multiples of 16)
    static constexpr int raw_pos = 0;                                   // float4 [KS]   landing zone of the bulk copies
    static constexpr int raw_vel = raw_pos + kDenseKS * 16;             // float4 [KS]
    static constexpr int raw_pc = raw_vel + kDenseKS * 16;              // float2 [KS]
    static constexpr int pos = raw_pc + kDenseKS * 8;                   // float4 [K]    the chunk in bin order: (x, y, z, m)
    static constexpr int vel = pos + kDenseK * 16;                      // float4 [K]    (v, rho)
    static constexpr int pc = vel + kDenseK * 16;                       // float2 [K]    (p/rho^2, c)
    static constexpr int hh = pc + kDenseK * 8;                         // float [K]     VARH: the candidates' smoothing lengths
    static constexpr int tpos = hh + (VARH ? kDenseK * 4 : 0);          // float4 [TT]   the item's targets
    static constexpr int tvel = tpos + kDenseTT * 16;                   // float4 [TT]
    static constexpr int tpc = tvel + kDenseTT * 16;                    // float2 [TT]
    static constexpr int acc = tpc + kDenseTT * 8;                      // double [TT][4]
    static constexpr int cfl = acc + kDenseTT * 8 * 4;                  // float [TT][4]: min d2, c^max, mu^max of Eq. 17, -
    static constexpr int runs = cfl + kDenseTT * 16;                    // uint32 [9][4]
    static constexpr int hist = runs + 9 * 4 * 4;                       // uint32 [rounds][warps][bins]
    static constexpr int bstart = hist + kRounds * kDenseWarps * kBins * 4;   // uint32 [seg][32]: start of bin b inside its segment
    static constexpr int box = bstart + kMaxSeg * 32 * 4;               // float [seg][bins][8]: xl, xh, yl, yh, zl, zh, -, -
    static constexpr int hmax = box + kMaxSeg * kBins * 8 * 4;          // uint32 [seg][32]: VARH: bits of the largest length in bin b
    static constexpr int th = hmax + (VARH ? kMaxSeg * 32 * 4 : 0);     // float [TT]: VARH: the targets' lengths
    static constexpr int queue = th + (VARH ? kDenseTT * 4 : 0);        // uint32 [warps][kQueue]
    static constexpr int seg = queue + kDenseWarps * kQueue * 4;        // uint4 [2][seg]: (row, first slot, end slot, raw base) of the
                                                                        // chunk being worked on and of the one being copied
    static constexpr int nseg = seg + 2 * kMaxSeg * 16;                 // uint32 [2] segments of those chunks, [2] (row, slot) the producer is at
    static constexpr int bar = nseg + 16;                               // uint64
    static constexpr int item = bar + 8;                                // uint32: the work item the CTA has drawn
    static constexpr int tnext = bar + 12;                              // uint32: next target of the chunk to hand to a warp
    static constexpr int bytes = bar + 16;
};
static_assert((DenseLayout<false>::bytes + 1024) * kDenseCtasPerSm <= 227 * 1024, "shared memory per SM");
static_assert((DenseLayout<true>::bytes + 1024) * kDenseCtasPerSm <= 227 * 1024, "shared memory per SM");

// CFL: the terms of Eq. 17 (s^min, c^max, mu^max; L125-129) are reduced in the same walk, as in k_forces (sph.cu).
// VARH: per-particle smoothing lengths h_s[] in cell order (L82; readings A24-A26 as in k_forces<true>): the pair is a
// neighbour pair iff d2 < fl(fl(h_i + h_j)^2), the pair term uses h_ij = (h_i + h_j)/2, and a target's sphere reaches a
// bin iff its distance to the bin's box is below h_i + (the largest length in that bin) — the paper's hmaxCell (L164,
// L207) at the granularity of the octant bins, gathered while the chunk is binned.
template <bool CFL, bool VARH>
__global__ void __launch_bounds__(kDenseThreads, kDenseCtasPerSm)
    k_dense_forces(const float4* __restrict__ posm_s, const float4* __restrict__ velr_s, const float2* __restrict__ pc_s,
            const float* __restrict__ h_s, const uint32_t* __restrict__ perm, const uint32_t* __restrict__ start, GridDev g,
            float cell, float rc2, ViscDev q, CflArgs cfl, Shard sh, unsigned int* __restrict__ ctl,
            const DenseItem* __restrict__ items, float4* __restrict__ acc_out) {
    using L = DenseLayout<VARH>;
    constexpr int kDenseK = L::kDenseK, kRounds = L::kRounds;
    extern __shared__ __align__(128) unsigned char smem[];
    float4* r_pos = reinterpret_cast<float4*>(smem + L::raw_pos);
    float4* r_vel = reinterpret_cast<float4*>(smem + L::raw_vel);
    float2* r_pc = reinterpret_cast<float2*>(smem + L::raw_pc);
    float4* c_pos = reinterpret_cast<float4*>(smem + L::pos);
    float4* c_vel = reinterpret_cast<float4*>(smem + L::vel);
    float2* c_pc = reinterpret_cast<float2*>(smem + L::pc);
    float* c_h = reinterpret_cast<float*>(smem + L::hh);
    float* t_h = reinterpret_cast<float*>(smem + L::th);
    uint32_t* s_hmax = reinterpret_cast<uint32_t*>(smem + L::hmax);
    float4* t_pos = reinterpret_cast<float4*>(smem + L::tpos);
    float4* t_vel = reinterpret_cast<float4*>(smem + L::tvel);
    float2* t_pc = reinterpret_cast<float2*>(smem + L::tpc);
    double* s_acc = reinterpret_cast<double*>(smem + L::acc);
    float4* s_cfl = reinterpret_cast<float4*>(smem + L::cfl);
    uint32_t* s_runs = reinterpret_cast<uint32_t*>(smem + L::runs);
    uint32_t* s_hist = reinterpret_cast<uint32_t*>(smem + L::hist);
    uint32_t* s_bstart = reinterpret_cast<uint32_t*>(smem + L::bstart);
    float4* s_box = reinterpret_cast<float4*>(smem + L::box);
    uint4* s_seg = reinterpret_cast<uint4*>(smem + L::seg);
    uint32_t* s_nseg = reinterpret_cast<uint32_t*>(smem + L::nseg);
    uint64_t* s_bar = reinterpret_cast<uint64_t*>(smem + L::bar);
    uint32_t* s_item = reinterpret_cast<uint32_t*>(smem + L::item);
    uint32_t* s_tnext = reinterpret_cast<uint32_t*>(smem + L::tnext);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned lt_mask = (1u << lane) - 1u;
    const uint32_t sbase = smem_u32(smem);
    const uint32_t a_pos = sbase + L::pos, a_vel = sbase + L::vel, a_pc = sbase + L::pc, a_h = sbase + L::hh;
    const uint32_t a_tpos = sbase + L::tpos, a_tvel = sbase + L::tvel, a_tpc = sbase + L::tpc;
    const uint32_t a_q = sbase + L::queue + 4u * kQueue * (uint32_t)warp;
    const uint32_t n_items = ctl[0];
    if (blockIdx.x >= n_items) return;   // uniform per CTA

    if (tid == 0) {
        mbar_init(s_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < kRounds * kDenseWarps * kBins; i += kDenseThreads) s_hist[i] = 0u;   // dense::bin_chunk keeps it zeroed
    uint32_t n_staged = 0;   // chunks this CTA has waited for so far: the barrier's phase parity
    uint32_t n_chunk = 0;    // chunks this CTA has described so far: the descriptor set in use is n_chunk & 1

    // The producer (thread 0): describe the next chunk of the item — rows in order from (s_nseg[2], s_nseg[3]); a row that
    // does not fit what is left of the chunk starts a new one unless the chunk is empty (then it is cut) — and start
    // its bulk copies.  Bulk copies need 16-byte alignment and the float2 array gives it on even slots only, so every
    // segment is staged from the even slot at or below its first one, at an even raw index.
    auto produce = [&](uint32_t set) {
        uint32_t r = s_nseg[2], cs = s_nseg[3], ns = 0, used = 0, raw = 0;
        while (r < 9u && ns < (uint32_t)kMaxSeg) {
            const uint32_t left = s_runs[4 * r + 3] - cs;
            if (left > (uint32_t)kDenseK - used && used > 0u) break;
            const uint32_t len = min(left, (uint32_t)kDenseK - used);
            const uint32_t base = cs & ~1u, cnt = (cs + len - base + 1u) & ~1u;
            s_seg[set * kMaxSeg + ns] = make_uint4(r, cs, cs + len, raw);
            raw += cnt;
            used += len;
            ++ns;
            cs += len;
            if (cs >= s_runs[4 * r + 3]) {
                ++r;
                while (r < 9u && s_runs[4 * r] >= s_runs[4 * r + 3]) ++r;
                if (r < 9u) cs = s_runs[4 * r];
            }
            if (used == (uint32_t)kDenseK) break;
        }
        s_nseg[set] = ns;
        s_nseg[2] = r;
        s_nseg[3] = cs;
        if (ns == 0u) return;
        mbar_expect_tx(s_bar, raw * 40u);
        for (uint32_t i = 0; i < ns; ++i) {
            const uint4 sg = s_seg[set * kMaxSeg + i];
            const uint32_t base = sg.y & ~1u, cnt = (sg.z - base + 1u) & ~1u;
            bulk_g2s(r_pos + sg.w, posm_s + base, cnt * 16u, s_bar);
            bulk_g2s(r_vel + sg.w, velr_s + base, cnt * 16u, s_bar);
            bulk_g2s(r_pc + sg.w, pc_s + base, cnt * 8u, s_bar);
        }
    };

    const float big = 3.0e38f;

    for (;;) {
        // items are handed out by a counter (ctl[1], zeroed before the launch): they differ by 100x in work, and a
        // target's sum does not depend on which CTA takes its item
        __syncthreads();   // the previous item's shared memory is no longer read
        if (tid == 0) *s_item = atomicAdd(ctl + 1, 1u);
        __syncthreads();
        const uint32_t item = *s_item;
        if (item >= n_items) break;
        const DenseItem it = items[item];
        const uint32_t mx = (uint32_t)g.mx, my = (uint32_t)g.my;
        const int ix = (int)(it.key % mx), iy = (int)((it.key / mx) % my), iz = (int)(it.key / (mx * my));
        const uint32_t ts = start[it.key] + it.chunk * kDenseTT;
        if (!sh.owns(ts)) continue;   // another rank's targets (common.cuh: Shard)
        const uint32_t nt = min(start[it.key + 1u] - ts, (uint32_t)kDenseTT);
        if (tid < 9) dense::row_bounds(start, g, ix, iy, iz, tid, s_runs);
        for (uint32_t t = tid; t < nt; t += kDenseThreads) {
            t_pos[t] = posm_s[ts + t];
            t_vel[t] = velr_s[ts + t];
            const float2 pc = pc_s[ts + t];
            t_pc[t] = pc;
#pragma unroll
            for (int c = 0; c < 4; ++c) s_acc[4 * t + c] = 0.0;
            if (CFL) s_cfl[t] = make_float4(__int_as_float(0x7f800000), pc.y, 0.f, 0.f);   // A22: no neighbour -> c_i, 0
            if (VARH) t_h[t] = h_s[ts + t];
        }
        __syncthreads();
        if (tid == 0) {
            uint32_t r = 0;
            while (r < 9u && s_runs[4 * r] >= s_runs[4 * r + 3]) ++r;
            s_nseg[2] = r;
            s_nseg[3] = r < 9u ? s_runs[4 * r] : 0u;
            produce(n_chunk & 1u);
        }
        __syncthreads();

        for (;;) {
            const uint32_t set = n_chunk & 1u;
            const uint32_t nseg = s_nseg[set];
            if (nseg == 0u) break;
            ++n_chunk;
            // ---- every segment of the chunk: counting sort by octant bin, stable: raw -> sorted (sph_dense_dev.cuh) ----
            uint32_t soff = 0;   // sorted index where the segment starts
            for (uint32_t sgi = 0; sgi < nseg; ++sgi) {
                const uint4 sg = s_seg[set * kMaxSeg + sgi];   // (row, first slot, end slot, raw base)
                const int r = (int)sg.x;
                const dense::RowGeom rg = dense::row_geom(g, cell, ix, iy, iz, r);
                if (VARH && tid < 32) s_hmax[32u * sgi + tid] = 0u;   // (ordered before the moves by bin_chunk's barriers)
                dense::bin_chunk<kDenseThreads, kRounds, false>(
                    r_pos, sg.w + (sg.y & 1u), sg.z - sg.y, sg.y, s_runs[4 * r + 1], s_runs[4 * r + 2], g, cell, ix, rg, s_hist,
                    s_bstart + 32u * sgi, s_box + 2u * kBins * sgi,
                    [&]() {
                        if (sgi == 0u) {
                            mbar_wait(s_bar, n_staged & 1u);
                            ++n_staged;
                        }
                    },
                    [&]() { *s_tnext = 0u; },
                    [&](uint32_t src, uint32_t dst, uint32_t bin) {
                        c_pos[soff + dst] = r_pos[src];
                        c_vel[soff + dst] = r_vel[src];
                        c_pc[soff + dst] = r_pc[src];
                        if (VARH) {   // the length straight from global memory (L2), and the bin's largest (positive floats order like their bits)
                            const float hj = h_s[sg.y + (src - (sg.w + (sg.y & 1u)))];
                            c_h[soff + dst] = hj;
                            atomicMax(s_hmax + 32u * sgi + bin, __float_as_uint(hj));
                        }
                    },
                    [&](uint32_t) {});
                soff += sg.z - sg.y;
            }
            if (tid == 0) produce(n_chunk & 1u);   // the landing zone is free: the next chunk's copies run under the work below

            // ---- the item's targets against the chunk ----
            // (shared memory by 32-bit address from here on: byte offsets in registers, no generic-address arithmetic)
            // targets are handed to the warps one at a time from a counter: their work differs (position in the cell, the
            // chunk's population), and the CTA waits for its slowest warp at the end of every chunk.  Which warp takes a
            // target does not enter its sum: a target meets the chunks in a fixed order, one warp per chunk.
            for (;;) {
                uint32_t t = 0;
                if (lane == 0) t = atomicAdd(s_tnext, 1u);
                t = __shfl_sync(0xffffffffu, t, 0);
                if (t >= nt) break;
                const float4 pi = lds_f4(a_tpos + 16u * t);
                const float4 vi = lds_f4(a_tvel + 16u * t);
                const float2 ci = lds_f2(a_tpc + 8u * t);
                const float h_i = VARH ? t_h[t] : 0.f;
                float ax = 0.f, ay = 0.f, az = 0.f, de = 0.f;
                float d2min = __int_as_float(0x7f800000), cmax = 0.f, mumax = 0.f;
                uint32_t qh = 0, qt = 0;   // ring queue of accepted candidates (byte offsets in the float4 arrays): head, tail x4
                auto pair_term = [&](uint32_t rel) {
                    const float4 pj = lds_f4(a_pos + rel);
                    const float4 vj = lds_f4(a_vel + rel);
                    const float2 cj = lds_f2(a_pc + (rel >> 1));
                    float dx, dy, dz, rv, mu;
                    const float d2 = dist2_f32(pi, pj, dx, dy, dz);
                    float f, c_v = 0.f;
                    if (VARH)   // the sparse walk's arithmetic (sph_dev.cuh says why); twice the term, as hydro_pair_fast's is halved below
                        f = hydro_pair_h(vi, ci, pj.w, vj, cj, dx, dy, dz, d2, __fadd_rn(h_i, lds_f32(a_h + (rel >> 2))), q, rv, mu, c_v);
                    else
                        f = hydro_pair_fast(vi, ci, pj.w, vj, cj, dx, dy, dz, d2, q, rv, mu);
                    ax = fmaf(-f, dx, ax);
                    ay = fmaf(-f, dy, ay);
                    az = fmaf(-f, dz, az);
                    de = fmaf(f, rv, de);   // m_j Pi dv . grad W_p: twice the term of Eq. 11, halved with the warp's sum
                    if (CFL) {
                        d2min = fminf(d2min, d2);
                        cmax = fmaxf(cmax, 0.5f * (ci.y + cj.y));
                        mumax = fmaxf(mumax, fabsf(mu));
                    }
                };
                uint32_t first = 0;   // sorted index where the segment starts
                for (uint32_t sgi = 0; sgi < nseg; ++sgi) {
                    // lane b: does the 2h sphere of the target reach the box of bin b of this segment?  (a lower bound of the distance)
                    const float4 bx0 = lane < kBins ? s_box[2u * (kBins * sgi + lane)] : make_float4(big, big, big, big);
                    const float4 bx1 = lane < kBins ? s_box[2u * (kBins * sgi + lane) + 1u] : make_float4(big, big, 0.f, 0.f);
                    const uint32_t ncand = s_bstart[32u * sgi + kBins];
                    const float ex = fmaxf(fmaxf(bx0.x - pi.x, pi.x - bx0.y), 0.f);
                    const float ey = fmaxf(fmaxf(bx0.z - pi.y, pi.y - bx0.w), 0.f);
                    const float ez = fmaxf(fmaxf(bx1.x - pi.z, pi.z - bx1.y), 0.f);
                    float rcb2 = rc2;
                    if (VARH) {   // h_i + the largest length among the bin's candidates
                        const float rcb = h_i + __uint_as_float(s_hmax[32u * sgi + lane]);
                        rcb2 = rcb * rcb;
                    }
                    const bool reach_b = fmaf(ez, ez, fmaf(ey, ey, ex * ex)) < rcb2;   // lanes >= kBins: their box is out of reach
                    // the reachable bins, in bin order, are the target's candidates in this segment: four slot ranges
                    const unsigned reach = __ballot_sync(0xffffffffu, reach_b);
                    if (reach == 0u) {   // nothing of this segment in reach (with per-particle lengths: most segments)
                        first += ncand;
                        continue;
                    }
                    const dense::Groups G = dense::candidate_groups(reach, s_bstart + 32u * sgi, first);
                    first += ncand;
                    const uint32_t T = G.T;
                    if (T == 0u) continue;
                    const uint32_t T16 = 16u * T;
                    // one step: 64 flat positions, two per lane (v16 and v16 + 32 x 16): the two tests are independent
                    // instruction streams, and the loop control and the queue's bookkeeping are paid once for both.
                    // FULL: every lane's two positions are inside the list; else `in` says which are (a position past the
                    // end still reads shared memory of this CTA: nothing is done with it)
                    auto step = [&](uint32_t v16, auto full) {
                        const uint32_t rel0 = dense::candidate_offset(G, v16), rel1 = dense::candidate_offset(G, v16 + 512u);
                        float dx, dy, dz;
                        const float d20 = dist2_f32(pi, lds_f4(a_pos + rel0), dx, dy, dz);
                        const float d21 = dist2_f32(pi, lds_f4(a_pos + rel1), dx, dy, dz);
                        // d2 == 0: self, or a coincident pair (A9) — no contribution
                        float rc20 = rc2, rc21 = rc2;
                        if (VARH) {   // d2 < fl(fl(h_i + h_j)^2) (A24); a position past the end reads some length of this CTA
                            const float s0 = __fadd_rn(h_i, lds_f32(a_h + (rel0 >> 2))), s1 = __fadd_rn(h_i, lds_f32(a_h + (rel1 >> 2)));
                            rc20 = __fmul_rn(s0, s0);
                            rc21 = __fmul_rn(s1, s1);
                        }
                        const bool ok0 = (decltype(full)::value || v16 < T16) && d20 < rc20 && d20 > 0.f;
                        const bool ok1 = (decltype(full)::value || v16 + 512u < T16) && d21 < rc21 && d21 > 0.f;
                        const unsigned m0 = __ballot_sync(0xffffffffu, ok0), m1 = __ballot_sync(0xffffffffu, ok1);
                        if (ok0) sts_u32(a_q + ((qt + 4u * __popc(m0 & lt_mask)) & (4u * kQueue - 4u)), rel0);
                        qt += 4u * __popc(m0);
                        if (ok1) sts_u32(a_q + ((qt + 4u * __popc(m1 & lt_mask)) & (4u * kQueue - 4u)), rel1);
                        qt += 4u * __popc(m1);
                        while (qt - qh >= 128u) {
                            __syncwarp();
                            pair_term(lds_u32(a_q + ((qh + 4u * (uint32_t)lane) & (4u * kQueue - 4u))));
                            qh += 128u;
                        }
                    };
                    const uint32_t full16 = T16 & ~1023u;
                    uint32_t v16 = 16u * (uint32_t)lane;
                    for (; v16 < full16; v16 += 1024u) step(v16, std::true_type{});   // v16 - 16 lane < full16 for every lane: uniform
                    if (full16 != T16) step(v16, std::false_type{});
                }
                if (qt != qh) {
                    __syncwarp();
                    if (4u * (uint32_t)lane < qt - qh) pair_term(lds_u32(a_q + ((qh + 4u * (uint32_t)lane) & (4u * kQueue - 4u))));
                }
                __syncwarp();   // the queue is rewritten for the next target
                if (qt != 0u) {
                    // the four sums over the 32 lanes in FP64, as one butterfly: after the exchange over lane bit 4 a
                    // lane holds two of them, after bit 3 one; lanes 0, 8, 16, 24 end with a_x, a_y, a_z, de/dt
                    const bool hi16 = (lane & 16) != 0, hi8 = (lane & 8) != 0;
                    const double dxs = (double)ax, dys = (double)ay, dzs = (double)az, des = 0.5 * (double)de;
                    double k0 = hi16 ? dzs : dxs, k1 = hi16 ? des : dys;
                    const double s0 = hi16 ? dxs : dzs, s1 = hi16 ? dys : des;
                    k0 += __shfl_xor_sync(0xffffffffu, s0, 16);
                    k1 += __shfl_xor_sync(0xffffffffu, s1, 16);
                    double k = hi8 ? k1 : k0;
                    k += __shfl_xor_sync(0xffffffffu, hi8 ? k0 : k1, 8);
                    k += __shfl_xor_sync(0xffffffffu, k, 4);
                    k += __shfl_xor_sync(0xffffffffu, k, 2);
                    k += __shfl_xor_sync(0xffffffffu, k, 1);
                    if ((lane & 7) == 0) s_acc[4 * t + (lane >> 3)] += k;
                    if (CFL) {   // non-negative floats order like their bit patterns
                        const uint32_t m0 = __reduce_min_sync(0xffffffffu, __float_as_uint(d2min));
                        const uint32_t m1 = __reduce_max_sync(0xffffffffu, __float_as_uint(cmax));
                        const uint32_t m2 = __reduce_max_sync(0xffffffffu, __float_as_uint(mumax));
                        if (lane == 0) {
                            const float4 o = s_cfl[t];
                            s_cfl[t] = make_float4(fminf(o.x, __uint_as_float(m0)), fmaxf(o.y, __uint_as_float(m1)),
                                                   fmaxf(o.z, __uint_as_float(m2)), 0.f);
                        }
                    }
                }
            }
            __syncthreads();   // every warp is done with the sorted chunk; the next chunk's description is visible
        }
        __syncthreads();

        for (uint32_t t = tid; t < nt; t += kDenseThreads) {
            const uint32_t i = perm[ts + t];
            const float4 a_own = make_float4((float)s_acc[4 * t], (float)s_acc[4 * t + 1], (float)s_acc[4 * t + 2],
                                             (float)s_acc[4 * t + 3]);
            if (acc_out) acc_out[i] = a_own;
            if (CFL) {
                const float4 c = s_cfl[t];
                const float bound = cfl_bracket(c.x, c.x == __int_as_float(0x7f800000), 2.0f * (VARH ? t_h[t] : q.h), c.y, c.z, q.alpha, q.beta,
                                                cfl.q_sph ? cfl.q_sph[i] : a_own, cfl.acc_grav[i]);
                if (cfl.dt_particle) cfl.dt_particle[i] = bound;
                cfl_min(cfl.c_cfl * bound, cfl.dt_bits);
            }
        }
    }
}

// the work list from a caller's cell_start (stand-alone calls): one thread per cell
__global__ void __launch_bounds__(256) k_dense_list(const uint32_t* __restrict__ start, int64_t M, unsigned int* ctl,
                                                    DenseItem* items) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= M) return;
    const uint32_t c = start[k + 1] - start[k];
    if (c >= (uint32_t)kDenseMin) dense_append((uint32_t)k, c, ctl, items);
}

}  // namespace

int dense_list_from_start(const uint32_t* cell_start, const sph_grid* g, const DenseList& dl, cudaStream_t st) {
    const int64_t M = grid_cells(g);
    SPHB_CUDA(cudaMemsetAsync(dl.ctl, 0, sizeof(unsigned int), st));
    k_dense_list<<<(unsigned)cdiv(M, 256), 256, 0, st>>>(cell_start, M, dl.ctl, dl.items);
    SPHB_LAUNCHED();
    return SPH_OK;
}

int forces_dense(const float4* posm_s, const float4* velr_s, const float2* pc_s, const float* h_s /*cell order, or NULL*/,
                 const uint32_t* perm, const uint32_t* cell_start, const sph_grid* g, float rc2, const ViscDev& q,
                 const DenseList& dl, const CflArgs* cfl, float4* acc_sph, cudaStream_t st, Shard sh) {
    int dev = 0;
    SPHB_CUDA(cudaGetDevice(&dev));
    static std::atomic<bool> opted[64];   // per device: the dynamic shared-memory opt-in
    if (dev < 0 || dev >= 64) return SPH_ERR_UNSUPPORTED;
    if (!opted[dev].load(std::memory_order_acquire)) {
        SPHB_CUDA(cudaFuncSetAttribute(k_dense_forces<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DenseLayout<false>::bytes));
        SPHB_CUDA(cudaFuncSetAttribute(k_dense_forces<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DenseLayout<false>::bytes));
        SPHB_CUDA(cudaFuncSetAttribute(k_dense_forces<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, DenseLayout<true>::bytes));
        SPHB_CUDA(cudaFuncSetAttribute(k_dense_forces<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, DenseLayout<true>::bytes));
        opted[dev].store(true, std::memory_order_release);
    }
    // the faces of the cells follow the rule the keys are made with (A7: c = (x - origin) * inv_cell), so the cell
    // edge is taken from inv_cell, not from g->cell
    SPHB_CUDA(cudaMemsetAsync(dl.ctl + 1, 0, sizeof(unsigned int), st));   // the item counter
    const unsigned grid = (unsigned)(kDenseCtasPerSm * num_sms());
    const float cell = 1.0f / g->inv_cell;
    const CflArgs c = cfl ? *cfl : CflArgs{};
    const GridDev gd = to_dev(g);
    if (h_s) {
        if (cfl)
            k_dense_forces<true, true><<<grid, kDenseThreads, DenseLayout<true>::bytes, st>>>(
                posm_s, velr_s, pc_s, h_s, perm, cell_start, gd, cell, rc2, q, c, sh, dl.ctl, dl.items, acc_sph);
        else
            k_dense_forces<false, true><<<grid, kDenseThreads, DenseLayout<true>::bytes, st>>>(
                posm_s, velr_s, pc_s, h_s, perm, cell_start, gd, cell, rc2, q, c, sh, dl.ctl, dl.items, acc_sph);
    } else {
        if (cfl)
            k_dense_forces<true, false><<<grid, kDenseThreads, DenseLayout<false>::bytes, st>>>(
                posm_s, velr_s, pc_s, nullptr, perm, cell_start, gd, cell, rc2, q, c, sh, dl.ctl, dl.items, acc_sph);
        else
            k_dense_forces<false, false><<<grid, kDenseThreads, DenseLayout<false>::bytes, st>>>(
                posm_s, velr_s, pc_s, nullptr, perm, cell_start, gd, cell, rc2, q, c, sh, dl.ctl, dl.items, acc_sph);
    }
    SPHB_LAUNCHED();
    return SPH_OK;
}

}  // namespace sphb
