// grav_dev.cuh — device helpers shared by the two gravity translation units (gravity.cu: one-sided kernel,
// packing, reduction; gravity_sym.cu: pair-symmetric kernel).  Internal to libsph_b200; nothing here is shared
// with the oracle.
#pragma once
#include "common.cuh"
#include "tma_dev.cuh"

namespace sphb {

typedef unsigned long long u64;

__device__ __forceinline__ u64 pk2(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(u64 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 sub2(u64 a, u64 b) {
    u64 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ u64 shfl2(u64 v, int src_lane) {   // both halves of a packed register from another lane
    float lo, hi;
    upk2(v, lo, hi);
    lo = __shfl_sync(0xffffffffu, lo, src_lane);
    hi = __shfl_sync(0xffffffffu, hi, src_lane);
    return pk2(lo, hi);
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// ---- device-side control block of one gravity evaluation (lives in the 256-byte grav_flag slot of the workspace) --
// Zeroed by a memset at the start of every evaluation; written by grav_pack_sources (nonuniform, bounding box)
// and grav_plan (sym, scale); read by every gravity kernel, which returns at once when it is not the variant the
// block selects.  No host read-back anywhere.
struct GravCtl {
    unsigned int nonuniform;   // != 0: the masses are not all equal to m_0
    unsigned int sym;          // != 0: the pair-symmetric path applies (delta > 0, positive masses, fixed-point range fits)
    unsigned int counter;      // work-item counter of the persistent pair-symmetric kernel
    float scale;               // fixed-point scale 2^k of the int64 accumulators
    double inv_scale;          // 2^-k
    unsigned int bmin_c[3];    // bounding box of all particles: max over particles of ~ord(x) (so 0 = empty)
    unsigned int bmax[3];      // max over particles of ord(x); ord() maps floats to order-preserving unsigned
    unsigned int mmin_c, mmax; // the same for the masses: max of ~ord(m), max of ord(m)
};
static_assert(sizeof(GravCtl) <= 256, "GravCtl must fit the workspace slot");

constexpr float kPadCoord = 1.0e18f;   // padded sources: mass 0 far away, contribute exactly 0 (see grav_pack_sources)
constexpr int kSymL = 2048;            // sources (columns) per work item of the pair-symmetric kernel
constexpr int kSymMinN = 32768;        // below this the one-sided kernel is used

int gravity_sym_launch(const float4* posm, const float4* src_pk, int n_pad, int share_rank, int share_world, float eps2,
                       long long* acc64, GravCtl* ctl, cudaStream_t st);

}  // namespace sphb
