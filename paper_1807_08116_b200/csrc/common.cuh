// common.cuh — internal declarations shared by the CUDA translation units of libsph_b200.
// Nothing here is visible at the C boundary (include/sph_b200.h) and nothing here is shared
// with the oracle.
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <stdint.h>
#include <stddef.h>
#include "../../include/sph_b200.h"

namespace sphb {

// ---- error plumbing ---------------------------------------------------------------------
extern thread_local int g_last_cuda_error;
extern std::atomic<long long> g_launch_count;   // kernels enqueued by this library (sph_launch_count)

inline int cuda_fail(cudaError_t e) {
    g_last_cuda_error = (int)e;
    return SPH_ERR_CUDA;
}
#define SPHB_CUDA(call)                                         \
    do {                                                        \
        cudaError_t e__ = (call);                               \
        if (e__ != cudaSuccess) return ::sphb::cuda_fail(e__);  \
    } while (0)
// after a kernel launch: count it and surface launch-configuration errors
#define SPHB_LAUNCHED()                                         \
    do {                                                        \
        ++::sphb::g_launch_count;                               \
        cudaError_t e__ = cudaGetLastError();                   \
        if (e__ != cudaSuccess) return ::sphb::cuda_fail(e__);  \
    } while (0)
#define SPHB_TRY(call)                 \
    do {                               \
        int rc__ = (call);             \
        if (rc__ != SPH_OK) return rc__; \
    } while (0)

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

int num_sms();

// ---- grid descriptor as the kernels see it -----------------------------------------------
struct GridDev {
    float ox, oy, oz, inv_cell;
    int mx, my, mz;
    float fx, fy, fz;   // (float)(M-1) per axis, the float clamp bound of reading A7
};
inline int64_t grid_cells(const sph_grid* g) { return (int64_t)g->dims[0] * g->dims[1] * g->dims[2]; }
int check_grid(const sph_grid* g, float h);          // SPH_OK or SPH_ERR_GRID
GridDev to_dev(const sph_grid* g);

// ---- dense-cell work list (sph_dense.cu) ----------------------------------------------------
// A cell holding at least kDenseMin particles is walked by the dense kernels, kDenseTT targets per work item; the
// thread-per-slot kernels skip its slots.  The list is written by the grid build (k_scan_apply has every cell's
// count in registers) or, for the stand-alone calls that get cell_start from the caller, by dense_list_from_start.
constexpr int kDenseMin = 32;
constexpr int kDenseTT = 128;
struct DenseItem {
    uint32_t key;     // cell number
    uint32_t chunk;   // targets [start[key] + chunk kDenseTT, ... + kDenseTT) of that cell
};
// The SPH passes shared over several GPUs (targets in slices of the sorted order over the replicated
// sorted arrays): rank `rank` of `world` takes every world-th tile of 128 sorted slots — a thread-per-slot
// CTA, or a dense work item by its first slot — and leaves the other targets' outputs untouched.  {0, 1}: everything.
struct Shard {
    uint32_t rank, world;
    __host__ __device__ bool owns(uint32_t first_slot) const { return ((first_slot >> 7) % world) == rank; }
};

struct DenseList {
    unsigned int* ctl;   // device: ctl[0] = number of items
    DenseItem* items;    // device: [dense_capacity(n_gas)]
};
inline size_t dense_capacity(int64_t n_gas) { return (size_t)(n_gas / kDenseMin + n_gas / kDenseTT + 16); }

// ---- Eq. 17 gathered inside the HFC neighbour walk (L125-129) ---------------------------------
// With a CflArgs the forces kernels also reduce, per gas particle, s^min, c^max and mu^max over the accepted pairs, form
// the bracket of Eq. 17 and take its minimum (x c_cfl) into *dt_bits by integer atomicMin on the float's bit pattern.
struct CflArgs {
    float c_cfl;
    const float4* q_sph;      // (a_sph, de/dt) by original index for |Q_i|, |E_i|, or NULL: the sums this very walk computes
    const float4* acc_grav;   // a_grav by original index
    float* dt_particle;       // [n_gas] bracket per particle (without c_cfl), or NULL
    unsigned int* dt_bits;    // the running minimum (float bits; positive floats order like unsigned integers)
};

// ---- workspace layout (device scratch carved from the caller's ws) -------------------------
struct Workspace {
    // grid sort
    uint32_t* key;         // [n_gas]   cell number of original particle i
    uint32_t* rank_u;      // [n_gas]   unstable in-cell rank from the histogram atomics
    uint32_t* tmp;         // [n_gas]   unstable scatter (original indices, cell order)
    uint32_t* perm;        // [n_gas]   stable permutation: sorted slot -> original index
    uint32_t* cell_count;  // [M]
    uint32_t* cell_start;  // [M+1]
    uint32_t* tile_sums;   // [n_scan_tiles + 1]
    // sorted (cell-order) particle data
    float4* posm_s;        // [n_gas] (x,y,z,m)
    float4* velr_s;        // [n_gas] (vx,vy,vz,rho)
    float2* pc_s;          // [n_gas] (p/rho^2, c)
    float* h_s;            // [n_gas] per-particle smoothing lengths in cell order (NEXT-2)
    DenseList dense;       // work list of the densely populated cells
    unsigned int* status;  // 256-byte block; word 0: SPH_STATUS_* bits raised by kernels (sph_workspace_status)
    // gravity
    float4* src_pk;        // [n_pad] packed source pairs
    float4* grav_part;     // [S][n_total] partial accelerations
    long long* grav_acc64;     // [n_pad][3] fixed-point accumulators of the pair-symmetric gravity kernel
    size_t grav_acc64_off;     // its byte offset in the workspace (sph_workspace_gravity_sums)
    unsigned int* grav_flag;   // 256-byte device control block of one gravity evaluation (GravCtl, grav_dev.cuh)
    // integrator
    float4* vele0;         // [n_total] v(t), e(t) saved by the predictor
    // bbox scratch
    float* bbox;           // [8]
    size_t bytes;          // total
};
// Lays the arrays out behind `base` (may be NULL to just measure).  g may be NULL if n_gas == 0.
Workspace carve(void* base, int64_t n_gas, int64_t n_total, const sph_grid* g);

// gravity decomposition (shared by carve and the launcher)
constexpr int kGravTileSrc = 2048;                 // sources per shared-memory stage
int grav_splits(int64_t n_total);                  // S: number of j-chunks
int64_t grav_padded(int64_t n_total);              // sources padded to a whole number of tiles

// ---- internal stage entry points (all enqueue on `st`, no synchronisation) -----------------
int grid_build(const float4* posm, int64_t n_gas, const sph_grid* g, uint32_t* key, uint32_t* perm,
               uint32_t* cell_count, uint32_t* cell_start, uint32_t* rank_u, uint32_t* tmp, uint32_t* tile_sums,
               float4* posm_s /*may be NULL*/, const DenseList* dense /*may be NULL*/, cudaStream_t st);
int dense_list_from_start(const uint32_t* cell_start, const sph_grid* g, const DenseList& dl, cudaStream_t st);
int gather_sorted_pos(const float4* posm, const uint32_t* perm, int64_t n_gas, float4* posm_s, cudaStream_t st);
// h_s: per-particle smoothing lengths in cell order (NEXT-2), or NULL for the one global p->h
// dense: the work list of the densely populated cells, matching cell_start (global h only; NULL: every slot is walked
// by the thread-per-slot kernel)
int density_sorted(const float4* posm_s, const float* h_s, const uint32_t* perm, const uint32_t* cell_start,
                   int64_t n_gas, const sph_params* p, const sph_grid* g, const DenseList* dense, float* rho,
                   cudaStream_t st, Shard sh = Shard{0u, 1u});
int forces_sorted(const float4* posm_s, const float4* vele, const float* rho, const float* h_s, const uint32_t* perm,
                  const uint32_t* cell_start, int64_t n_gas, const sph_params* p, const sph_grid* g,
                  const DenseList* dense, const CflArgs* cfl /*or NULL*/, float4* velr_s, float2* pc_s,
                  float4* acc_sph /*or NULL with cfl: only the step criterion is wanted*/, cudaStream_t st,
                  Shard sh = Shard{0u, 1u});
int cfl_init(float* dt_dev, float dt_max, cudaStream_t st);   // *dt_dev = dt_max (+inf: no ceiling)
int smoothing_lengths(const float4* posm, const float* rho, int64_t n_gas, float sigma, float h_max, float* hsml,
                      cudaStream_t st);
int gather_sorted_h(const float* hsml, const uint32_t* perm, int64_t n_gas, float h_max, unsigned int* status, float* h_s,
                    cudaStream_t st);
int gravity_share(const float4* posm, int64_t n_total, int64_t i0, int64_t i1, int rank, int world, bool offer_sym,
                  float G, float delta, float4* acc_grav, float4* src_pk, float4* grav_part, long long* grav_acc64,
                  unsigned int* grav_flag, cudaStream_t st);   // one GPU's share of an evaluation (gravity.cu)
int gravity_finish(const float4* posm, int64_t n_total, float G, float4* acc_grav, const long long* grav_acc64,
                   const unsigned int* grav_flag, cudaStream_t st);   // after the exchange: sums -> acc_grav, if pair-symmetric
int gravity(const float4* posm, int64_t n_total, int64_t i0, int64_t i1, float G, float delta, float4* acc_grav,
            float4* src_pk, float4* grav_part, long long* grav_acc64, unsigned int* grav_flag, cudaStream_t st);   // targets [i0, i1) against all sources
// dt_dev != NULL: the step is read from device memory (the adaptive step of Eq. 17), else it is `dt`
int update_predictor(float4* posm, float4* vele, float4* vele0, const float4* acc_sph, const float4* acc_grav,
                     int64_t n_gas, int64_t n_total, float dt, const float* dt_dev, cudaStream_t st);
int update_corrector(float4* vele, const float4* vele0, const float4* acc_sph, const float4* acc_grav,
                     int64_t n_gas, int64_t n_total, float dt, const float* dt_dev, cudaStream_t st);
int bbox_gas(const float4* posm, int64_t n_gas, float* bbox_dev /*[8]*/, cudaStream_t st);

}  // namespace sphb
