// gravity_sym.cu — (a10) Eq. 4 (reading A1) evaluated once per UNORDERED pair.
//
// Eq. 4 is antisymmetric: the term of source j in a_i is m_j w d and the term of source i in a_j is -m_i w d, with the
// SAME  w = (|d|^2 + delta^2)^(-3/2),  d = r_j - r_i  ("Newton's third law", which the paper invokes for its SPH terms at
// L95), so one evaluation of w and d serves two interactions.  With equal masses (every BASELINE.json config, and the
// paper's model: equal-mass particles per component) both terms are the same vector w d:
//   3 sub + 3 fma + rsqrt + 2 mul + 3 fma (a_i += w d) + 3 fma (t_j += w d)  = 14 FP32 operations + 1 MUFU per PAIR,
// i.e. 7 + 0.5 per interaction against the 11 + 1 of the one-sided kernel (gravity.cu); with unequal masses two more
// multiplications (m_j w, m_i w): 8 + 0.5 against 12 + 1.
//
// The difficulty is the second accumulator: the one-sided kernel broadcasts each source to all threads, so a
// source-side sum would need a reduction over every thread.  Here sources CIRCULATE instead (a systolic ring in
// each warp): a lane owns I targets (registers: position + packed accumulator) and, at any moment, two packed source
// pairs A and B (position + source-side accumulator, also registers).  One step evaluates the lane's I targets
// against its current pairs and passes the pairs, with their accumulators, to the next lane by SHFL; after 32 steps
// every pair has met every lane's targets and is home again.  While pair A's 12 shuffles are in flight the lane
// works on pair B, so their latency is hidden.  Per lane and step: 2 x I packed evaluations (28 FMA-pipe cycles
// each) against 24 SHFL.
//
// Work decomposition.  Particles are cut into column blocks of L = 2048 (the packed source layout of
// grav_pack_sources, one TMA bulk copy per block).  The pairs (i, j) with i < c L <= j < (c+1) L, i.e. block c
// against ALL EARLIER particles, are cut into work items of at most `rows_per_item` rows; the diagonal blocks
// (i, j in the same column block) go to the one-sided kernel (N x L interactions, 0.2 % at N = 2^20), which adds its
// FP32 sums into the same fixed-point accumulators.  One CTA of
// 4 warps takes an item: all warps hold the SAME 32 I rows and each owns a quarter of the column block, so a source
// belongs to exactly one warp (its sums live in that warp's shared-memory slots, no inter-warp traffic), and the
// target sums of the 4 warps are added through shared memory once per row tile.  Items are handed out by an atomic
// counter to a persistent grid of (SMs x resident CTAs).
//
// Accumulation and determinism.  Partial sums leave a CTA as 64-bit FIXED-POINT integers added with
// red.global.add.u64: integer addition is associative, so the result does not depend on the order in which CTAs
// finish — the evaluation is bitwise reproducible although the work is scheduled dynamically — and no [S][N] partial
// buffer is needed.  The scale 2^k is chosen on the device (grav_plan) so that the largest possible sum,
// N max_r r/(r^2+delta^2)^(3/2) = 0.385 N/delta^2, cannot overflow; the symmetric path is only taken when the
// resolution 2^-k is below 2^-26 of N m_min/R^2 (R = bounding-box diagonal: the sum's natural magnitude), otherwise —
// and for non-positive masses, delta = 0, explicit target slices or small N — the one-sided kernel runs (see gravity()).
// FP32 partials before conversion: <= 256 terms per packed half (targets: one row tile x a warp's quarter block;
// sources: 32 lanes x I rows per ring revolution, then one FP32 add per row tile of the item).
#include "grav_dev.cuh"

namespace sphb {

constexpr int kSymI = 8;                      // targets per lane
constexpr int kSymRows = 32 * kSymI;          // rows per tile (the same rows in all 4 warps)
constexpr int kSymThreads = 128;

// one packed evaluation: target k against the lane's current source pair; both sides accumulate
#define SPHB_SYM_EVAL(XJ, YJ, ZJ, MJ, TX, TY, TZ, k)                  \
    {                                                                 \
        const u64 dx = sub2(XJ, xi[k]);                               \
        const u64 dy = sub2(YJ, yi[k]);                               \
        const u64 dz = sub2(ZJ, zi[k]);                               \
        u64 r2 = fma2(dx, dx, e2);                                    \
        r2 = fma2(dy, dy, r2);                                        \
        r2 = fma2(dz, dz, r2);                                        \
        float r2a, r2b;                                               \
        upk2(r2, r2a, r2b);                                           \
        const u64 u = pk2(rsqrt_approx(r2a), rsqrt_approx(r2b));      \
        const u64 w = mul2(mul2(u, u), u);                            \
        const u64 wi = UNIFORM ? w : mul2(w, MJ);      /* m_j w */    \
        const u64 wj = UNIFORM ? w : mul2(w, mi[k]);   /* m_i w */    \
        ax[k] = fma2(wi, dx, ax[k]);                                  \
        TX = fma2(wj, dx, TX);                                        \
        ay[k] = fma2(wi, dy, ay[k]);                                  \
        TY = fma2(wj, dy, TY);                                        \
        az[k] = fma2(wi, dz, az[k]);                                  \
        TZ = fma2(wj, dz, TZ);                                        \
    }

// shared memory: [L/2 pairs][2] float4 packed sources | [L/2 pairs][3] u64 source-side sums | [4][rows][3] f32
constexpr size_t kSymSmem = (size_t)kSymL * 16 + (size_t)kSymL * 12 + 4 * kSymRows * 3 * sizeof(float);

// UNIFORM: all masses equal m_0, which is left out of the loop (applied with G in grav_reduce).  Otherwise the two sides of
// a pair differ by the mass factor: a_i += (m_j w) d, t_j += (m_i w) d — 16 operations per pair; the source masses travel
// round the ring with the positions.
template <bool UNIFORM>
__global__ void __launch_bounds__(kSymThreads, 2)
    grav_sym_kernel(const float4* __restrict__ posm, const float4* __restrict__ pk, int n_pad, int rows_per_item,
                    int n_items, int share_rank, int share_world, float eps2, long long* __restrict__ acc64,
                    GravCtl* __restrict__ ctl) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* spk = reinterpret_cast<float4*>(smem_raw);
    u64* sacc = reinterpret_cast<u64*>(smem_raw + (size_t)kSymL * 16);
    float* sred = reinterpret_cast<float*>(smem_raw + (size_t)kSymL * 28);
    __shared__ __align__(8) uint64_t bar;
    __shared__ unsigned int s_item;
    // uniform over the grid: the one-sided kernel, or the other mass variant, does this evaluation
    if (ctl->sym == 0u || (ctl->nonuniform == 0u) != UNIFORM) return;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int from = (lane + 31) & 31;   // the ring: receive from lane - 1
    const int rpi_shift = 31 - __clz(rows_per_item);
    const float scale = ctl->scale;
    const u64 e2 = pk2(eps2, eps2);
    u64* const out = reinterpret_cast<u64*>(acc64);
    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    uint32_t phase = 0;
    for (;;) {
        if (tid == 0) s_item = atomicAdd(&ctl->counter, 1u);
        __syncthreads();
        // one GPU's share of the evaluation (NEXT-4): items rank, rank + world, ... ; all of them if world == 1
        const unsigned int item = s_item * (unsigned int)share_world + (unsigned int)share_rank;
        if (s_item >= (unsigned int)n_items || item >= (unsigned int)n_items) break;
        // item -> (column block c >= 1, run): block c has ceil(c L / rows_per_item) runs of rows below c L.
        // rows_per_item is a power of two, so the division is a shift (a 64-bit division here cost 1.5-4 % of the kernel).
        int c = 1, run = (int)item;
        for (;; ++c) {
            const int runs = (int)(((unsigned int)c * (unsigned int)kSymL + (unsigned int)(rows_per_item - 1)) >> rpi_shift);
            if (run < runs) break;
            run -= runs;
        }
        const int col0 = c * kSymL;                  // < n_pad, and every row below it is a real particle
        const int row0 = run * rows_per_item;
        const int row1 = min(row0 + rows_per_item, col0);
        if (tid == 0) {
            mbar_expect_tx(&bar, (uint32_t)kSymL * 16u);
            bulk_g2s(spk, pk + (size_t)col0, (uint32_t)kSymL * 16u, &bar);
        }
        for (int q = tid; q < (kSymL / 2) * 3; q += kSymThreads) sacc[q] = 0ull;
        __syncthreads();
        mbar_wait(&bar, phase);
        phase ^= 1u;
        constexpr int pairs_w = kSymL / 8;           // source pairs per warp
        const int pbase = warp * pairs_w;

        for (int rt = row0; rt < row1; rt += kSymRows) {
            u64 xi[kSymI], yi[kSymI], zi[kSymI], mi[kSymI], ax[kSymI], ay[kSymI], az[kSymI];
#pragma unroll
            for (int k = 0; k < kSymI; ++k) {
                const float4 t = posm[rt + k * 32 + lane];
                xi[k] = pk2(t.x, t.x);
                yi[k] = pk2(t.y, t.y);
                zi[k] = pk2(t.z, t.z);
                mi[k] = pk2(t.w, t.w);
                ax[k] = ay[k] = az[k] = 0ull;
            }
            for (int ps = 0; ps < pairs_w; ps += 64) {
                const int pA = pbase + ps + lane, pB = pA + 32;
                const float4 A0 = spk[2 * pA], A1 = spk[2 * pA + 1], B0 = spk[2 * pB], B1 = spk[2 * pB + 1];
                u64 xA = pk2(A0.x, A0.y), yA = pk2(A0.z, A0.w), zA = pk2(A1.x, A1.y);
                u64 xB = pk2(B0.x, B0.y), yB = pk2(B0.z, B0.w), zB = pk2(B1.x, B1.y);
                u64 mA = pk2(A1.z, A1.w), mB = pk2(B1.z, B1.w);
                u64 tAx = 0ull, tAy = 0ull, tAz = 0ull, tBx = 0ull, tBy = 0ull, tBz = 0ull;
#pragma unroll 1
                for (int s = 0; s < 32; ++s) {
#pragma unroll
                    for (int k = 0; k < kSymI; ++k) SPHB_SYM_EVAL(xA, yA, zA, mA, tAx, tAy, tAz, k)
                    xA = shfl2(xA, from);
                    yA = shfl2(yA, from);
                    zA = shfl2(zA, from);
                    if (!UNIFORM) mA = shfl2(mA, from);
                    tAx = shfl2(tAx, from);
                    tAy = shfl2(tAy, from);
                    tAz = shfl2(tAz, from);
#pragma unroll
                    for (int k = 0; k < kSymI; ++k) SPHB_SYM_EVAL(xB, yB, zB, mB, tBx, tBy, tBz, k)
                    xB = shfl2(xB, from);
                    yB = shfl2(yB, from);
                    zB = shfl2(zB, from);
                    if (!UNIFORM) mB = shfl2(mB, from);
                    tBx = shfl2(tBx, from);
                    tBy = shfl2(tBy, from);
                    tBz = shfl2(tBz, from);
                }
                // the pairs are home again: their sums go to this warp's own shared slots
                sacc[3 * pA + 0] = add2(sacc[3 * pA + 0], tAx);
                sacc[3 * pA + 1] = add2(sacc[3 * pA + 1], tAy);
                sacc[3 * pA + 2] = add2(sacc[3 * pA + 2], tAz);
                sacc[3 * pB + 0] = add2(sacc[3 * pB + 0], tBx);
                sacc[3 * pB + 1] = add2(sacc[3 * pB + 1], tBy);
                sacc[3 * pB + 2] = add2(sacc[3 * pB + 2], tBz);
            }
            // target side: even + odd sources, then the 4 warps (same rows), then fixed point
#pragma unroll
            for (int k = 0; k < kSymI; ++k) {
                float a, b;
                float* d = sred + ((size_t)warp * kSymRows + k * 32 + lane) * 3;
                upk2(ax[k], a, b);
                d[0] = a + b;
                upk2(ay[k], a, b);
                d[1] = a + b;
                upk2(az[k], a, b);
                d[2] = a + b;
            }
            __syncthreads();
            for (int q = tid; q < kSymRows * 3; q += kSymThreads) {
                const float v = (sred[q] + sred[kSymRows * 3 + q]) + (sred[2 * kSymRows * 3 + q] + sred[3 * kSymRows * 3 + q]);
                atomicAdd(out + (size_t)rt * 3 + q, (u64)__float2ll_rn(v * scale));
            }
            __syncthreads();
        }
        // source side: d was r_j - r_i, so a_j gets MINUS the sum
        const float* sf = reinterpret_cast<const float*>(sacc);   // pair p: (x0, x1, y0, y1, z0, z1)
        for (int q = tid; q < kSymL * 3; q += kSymThreads) {
            const int j = q / 3, comp = q - 3 * j;
            const float v = sf[(j >> 1) * 6 + comp * 2 + (j & 1)];
            atomicAdd(out + (size_t)col0 * 3 + q, (u64)__float2ll_rn(-v * scale));
        }
        __syncthreads();   // before the next item overwrites the shared block
    }
}

// rows per work item: a power of two in [256, 8192], small enough for >= ~16 items per resident CTA slot
static int sym_rows_per_item(int64_t ncols, int slots) {
    const int64_t pairs_rows = ncols * (ncols - 1) / 2 * kSymL;   // sum over blocks of rows below the block
    int rpi = 8192;
    while (rpi > kSymRows && pairs_rows / rpi < (int64_t)16 * slots) rpi >>= 1;
    return rpi;
}

int gravity_sym_launch(const float4* posm, const float4* src_pk, int n_pad, int share_rank, int share_world, float eps2,
                       long long* acc64, GravCtl* ctl, cudaStream_t st) {
    // the opt-in for > 48 KB of dynamic shared memory is per device (context): set it on every launch, as gravity.cu's
    // launch_one does, and cache the occupancy per device, so that a process driving several GPUs gets it right on each
    static int occ_dev[64] = {0};
    int dev = 0;
    SPHB_CUDA(cudaGetDevice(&dev));
    SPHB_CUDA(cudaFuncSetAttribute(grav_sym_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSymSmem));
    SPHB_CUDA(cudaFuncSetAttribute(grav_sym_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSymSmem));
    int occ = (dev >= 0 && dev < 64) ? occ_dev[dev] : 0;
    if (occ == 0) {
        int o1 = 0, o2 = 0;
        SPHB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o1, grav_sym_kernel<true>, kSymThreads, kSymSmem));
        SPHB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o2, grav_sym_kernel<false>, kSymThreads, kSymSmem));
        occ = o1 < o2 ? o1 : o2;
        if (occ < 1) occ = 1;
        if (dev >= 0 && dev < 64) occ_dev[dev] = occ;
    }
    const int64_t ncols = cdiv(n_pad, kSymL);
    const int slots = num_sms() * occ;
    const int rpi = sym_rows_per_item(ncols, slots);
    int64_t items = 0;
    for (int64_t c = 1; c < ncols; ++c) items += cdiv(c * kSymL, rpi);
    const int64_t mine = items > share_rank ? cdiv(items - share_rank, share_world) : 0;   // this rank's items
    if (mine <= 0) return SPH_OK;
    const unsigned grid = (unsigned)(mine < slots ? mine : slots);
    // both mass variants, back to back: the one that does not apply returns at once; the work-item counter is only
    // touched by the one that runs
    grav_sym_kernel<true><<<grid, kSymThreads, kSymSmem, st>>>(posm, src_pk, n_pad, rpi, (int)items, share_rank, share_world,
                                                               eps2, acc64, ctl);
    SPHB_LAUNCHED();
    grav_sym_kernel<false><<<grid, kSymThreads, kSymSmem, st>>>(posm, src_pk, n_pad, rpi, (int)items, share_rank, share_world,
                                                                eps2, acc64, ctl);
    SPHB_LAUNCHED();
    return SPH_OK;
}

}  // namespace sphb
