// noalloc.cu — nbody_pp_gravity_static: Eq. 4 for callers that cannot allocate device memory (code under
// CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  The scratch the gravity kernels need — the
// packed sources, the per-chunk partial sums, the 64-bit fixed-point sums of the pair-symmetric path, the control block:
// what a caller of nbody_pp_gravity provides as `ws` — lives in ONE file-scope device array of fixed size, so the call
// takes inputs and outputs only and allocates nothing.
//   * The array's name is a host-side stand-in in host code, not a device address: its address is taken once per device,
//     with that device current, by cudaGetSymbolAddress below, and that pointer is what the kernels are given.
//   * Every call on a device shares the array.  It keeps the last call's contents; what must start at zero (the control
//     block and the fixed-point sums) is cleared by every evaluation on the call's stream (gravity.cu: gravity_share).
//     Calls that overlap on the GPU (two streams, two host threads on one device) RACE on it: serialise them.
//   * Every GPU that loads the library holds the array (12 MiB) until the process exits.
#include "common.cuh"

namespace sphb {
namespace {

constexpr int64_t kStaticMaxN = 65536;                       // particles: both gravity paths fit (pair-symmetric from 32768)
constexpr size_t kStaticBytes = (size_t)12 * 1024 * 1024;    // >= the gravity workspace of kStaticMaxN particles (11.6 MiB)
static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

// the array's device address on the current device (set up once per device), or NULL with *err set
void* static_scratch(cudaError_t* err) {
    static void* ptr[64];
    static std::atomic<bool> done[64];
    int dev = 0;
    *err = cudaGetDevice(&dev);
    if (*err != cudaSuccess) return nullptr;
    if (dev < 0 || dev >= 64) {
        *err = cudaErrorInvalidDevice;
        return nullptr;
    }
    if (!done[dev].load(std::memory_order_acquire)) {
        void* p = nullptr;
        *err = cudaGetSymbolAddress(&p, g_static_scratch);
        if (*err != cudaSuccess || !p) {
            if (*err == cudaSuccess) *err = cudaErrorInvalidSymbol;
            return nullptr;
        }
        ptr[dev] = p;
        done[dev].store(true, std::memory_order_release);
    }
    return ptr[dev];
}

}  // namespace
}  // namespace sphb

using namespace sphb;

extern "C" {

int64_t nbody_pp_gravity_static_max(void) { return kStaticMaxN; }

int nbody_pp_gravity_static(const float* posm, int64_t n_total, float G, float delta, float* acc_grav, void* stream) {
    if (n_total < 0) return SPH_ERR_ARG;
    if (n_total > kStaticMaxN) return SPH_ERR_WORKSPACE;   // beyond the fixed scratch: use nbody_pp_gravity with a workspace
    if (delta < 0.f) return SPH_ERR_UNSUPPORTED;
    if (n_total == 0) return SPH_OK;
    if (!posm || !acc_grav || (reinterpret_cast<uintptr_t>(posm) & 15u) || (reinterpret_cast<uintptr_t>(acc_grav) & 15u))
        return SPH_ERR_ARG;
    cudaError_t err = cudaSuccess;
    void* scratch = static_scratch(&err);
    if (!scratch) return cuda_fail(err);
    const Workspace w = carve(scratch, 0, n_total, nullptr);
    if (w.bytes > kStaticBytes) return SPH_ERR_WORKSPACE;
    return gravity(reinterpret_cast<const float4*>(posm), n_total, 0, n_total, G, delta, reinterpret_cast<float4*>(acc_grav),
                   w.src_pk, w.grav_part, w.grav_acc64, w.grav_flag, (cudaStream_t)stream);
}

}  // extern "C"
