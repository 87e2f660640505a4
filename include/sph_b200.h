/*
 * sph_b200.h — C ABI of the B200-native (sm_100a) hot path of
 * Khrapov & Khoperskov, "Smoothed-Particle Hydrodynamics Models: Implementation Features
 * on GPUs" (arXiv 1807.08116).  Citations "Lnn" are lines of the paper text;
 * "A<n>" are the readings listed in DESIGN.md.
 *
 * Conventions (all entry points)
 *   - extern "C"; every function returns an int status (0 = SPH_OK, negative = error);
 *     no exceptions, no aborts, no printing.
 *   - Unless a parameter says HOST, every array argument is a DEVICE pointer owned by the
 *     caller, 16-byte aligned.  The library never allocates or frees device memory inside
 *     these calls: scratch comes from the caller's workspace `ws` (DEVICE, >= the size
 *     sph_workspace_bytes() reports, 256-byte aligned).  Only the *_host entry points, which
 *     take HOST arrays, allocate (and free) device memory themselves.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Work
 *     is enqueued on it and the call returns without synchronising, except where stated.
 *   - Particle order: gas first [0, n_gas), halo [n_gas, n_total)  (the paper sums SPH
 *     over 1..N_g and gravity over 1..N, L74, L91).
 *       posm[i] = (x, y, z, m)        float4
 *       vele[i] = (vx, vy, vz, e)     float4   (e ignored for halo particles)
 *     All outputs are in the caller's ORIGINAL particle order.
 *   - n_gas = 0 (collisionless, L150) and n_halo = 0 are legal.  Inputs must be finite.
 *   - Counts are int64_t at the boundary; n_gas and n_total must be < 2^31.
 */
#ifndef SPH_B200_H
#define SPH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    SPH_OK = 0,
    SPH_ERR_ARG = -1,         /* null / misaligned pointer, negative count, non-positive h */
    SPH_ERR_GRID = -2,        /* a grid dimension > 4096, M >= 2^31, or cell < 2h */
    SPH_ERR_WORKSPACE = -3,   /* workspace (or output capacity) too small */
    SPH_ERR_CUDA = -4,        /* CUDA launch / runtime failure; see sph_last_cuda_error() */
    SPH_ERR_UNSUPPORTED = -5  /* e.g. delta < 0 */
};

/* Dense grid covering the computational domain (L158 "covered by a grid Mx x My x Mz").
 * Reading A7: cell = fl(fl(2h)(1+2^-9)), inv_cell = fl(1/cell); a particle's cell coordinate is
 *   ix = (int) min(max(floor(fl(fl(x - origin_x) * inv_cell)), 0), Mx-1)
 * (two separate FP32 RN operations, clamp in float before the cast), and its cell number is
 *   k = ix + Mx (iy + My iz)                                                          (L161). */
typedef struct {
    float origin[3];
    float cell;
    float inv_cell;
    int32_t dims[3];
} sph_grid;

/* h: smoothing length (one global value, L82 with h_i = h);  gamma: adiabatic index (Eq. 5);
 * alpha, beta, eta: artificial-viscosity constants (L99: 0.5, 1, 0.1);  G, delta: Eq. 4 (L47-49). */
typedef struct {
    float h, gamma, alpha, beta, eta;
    float G, delta;
} sph_params;

/* cudaError_t of the last failing CUDA call seen by this library in the calling thread (0 if none). */
int sph_last_cuda_error(void);

/* Grid descriptor from the bounding box of the gas particles (A7): origin = component-wise
 * minimum, dims = (int)(fl(fl(max - origin) * inv_cell)) + 1.  SYNCHRONISES `stream` (it
 * returns a HOST struct).  ws: >= 4096 bytes.  Errors: SPH_ERR_ARG, SPH_ERR_GRID.            */
int sph_grid_from_bbox(const float* posm, int64_t n_gas, float h, sph_grid* out_host /*HOST*/,
                       void* ws, size_t ws_bytes, void* stream);

/* Bytes of workspace that any call below needs for these sizes (g may be NULL when n_gas = 0). */
size_t sph_workspace_bytes(int64_t n_gas, int64_t n_total, const sph_grid* g /*HOST*/);

/* (a1-a4) Grid sort, L158-173: per-particle cell number (indexPC[i].x), per-cell count
 * (CellSPH[k].x), exclusive prefix cell_start[k] = CellSPH[k-1].y with cell_start[M] = n_gas
 * (A13), and perm = indexPC[.].y : sorted slot -> original index.  Unlike the paper's atomic
 * scatter (L204) the order inside a cell is STABLE (ascending original index, A16) and the
 * whole result is deterministic.
 *   key[n_gas], perm[n_gas], cell_count[M], cell_start[M+1]  — uint32, all written.          */
int sph_build_grid(const float* posm, int64_t n_gas, const sph_grid* g /*HOST*/,
                   uint32_t* key, uint32_t* perm, uint32_t* cell_count, uint32_t* cell_start,
                   void* ws, size_t ws_bytes, void* stream);

/* (a5) Ranges the neighbour loops of DC / HFC walk (L207):
 *   cell_range[k]      = (start, end) of cell k in sorted order = (CellSPH[k-1].y, CellSPH[k].y) (L160, L203);
 *   particle_runs[i][r] = (start, end) of the r-th x-run (r = (dy+1) + 3 (dz+1), dy,dz in -1..1)
 *                         of the 3x3x3 stencil of ORIGINAL particle i: the three x-adjacent
 *                         cells of a stencil row are contiguous in sorted order, so 9 runs cover
 *                         the 27 cells; rows outside the grid give (0,0).
 * Either output may be NULL.  Layout: uint32 pairs.                                          */
int sph_neighbour_ranges(const sph_grid* g /*HOST*/, const uint32_t* key, const uint32_t* cell_start,
                         int64_t n_gas, uint32_t* cell_range /*[M][2]*/, uint32_t* particle_runs /*[n_gas][9][2]*/,
                         void* stream);

/* (a6-a7) Density, Eq. 7 (L74) with the cubic spline of Eq. 8 (L79), self term included (A5):
 *   rho_i = sum_{j gas, |r_ij| < 2h} m_j W(|r_ij|/h, h).   Cutoff predicate in FP32 (A8):
 *   d2 = fma(dz,dz, fma(dy,dy, dx*dx)) < fl(fl(2h)^2).
 * perm / cell_start are the outputs of sph_build_grid for the same posm and g.                */
int sph_density(const float* posm, int64_t n_gas, const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/,
                const uint32_t* perm, const uint32_t* cell_start, float* rho /*[n_gas]*/,
                void* ws, size_t ws_bytes, void* stream);

/* (a8-a9) Hydrodynamic force and energy rate, Eqs. 10-11 (L91-93) hydro part, with
 * W_p of Eq. 9 (L86), Pi_ij and the Monaghan viscosity of L95-99 (A2: p_j/rho_j^2), EOS Eq. 5:
 *   acc_sph[i] = (a_x, a_y, a_z, de/dt).   A coincident pair contributes nothing (A9).        */
int sph_forces(const float* posm, const float* vele, const float* rho, int64_t n_gas,
               const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/,
               const uint32_t* perm, const uint32_t* cell_start, float* acc_sph /*[n_gas][4]*/,
               void* ws, size_t ws_bytes, void* stream);

/* (a10) Direct Particle-Particle gravity, Eq. 4 (L47) with Plummer softening (A1):
 *   acc_grav[i] = -G sum_{j=1..N} m_j (r_i - r_j) / (|r_i - r_j|^2 + delta^2)^(3/2), w = 0.
 * delta >= 0; with delta = 0 coincident pairs contribute 0.  Two kernels compute it: for
 * n_total >= 32768, delta > 0 and positive masses every UNORDERED pair is evaluated once and the sums are kept as
 * 64-bit fixed-point integers (bitwise reproducible; taken when the range rule of DESIGN.md 5.1.1 holds), otherwise
 * every ordered interaction is evaluated; the choice is made on the device and sph_gravity_path() reports it.
 * Both are held to the same tolerance against the oracle (2e-4 of the per-particle value, 1e-5 median).          */
int nbody_pp_gravity(const float* posm, int64_t n_total, float G, float delta,
                     float* acc_grav /*[n_total][4]*/, void* ws, size_t ws_bytes, void* stream);

/* (a1-a11) One predictor-corrector "leapfrog" step, Eqs. 12-16 (L103-121), in the order
 * HFC(pred) -> SU(pred) -> SP, DC, GFC at r(t+dt) -> HFC(corr) -> SU(corr)   (A11; gravity once
 * per step, L123).  posm / vele are updated in place.  rho[n_gas], acc_sph[n_gas][4],
 * acc_grav[n_total][4] and the grid arrays inside `ws` are CARRIED STATE between calls: the
 * caller must not modify them, must pass the same buffers, and must pass first != 0 on the first
 * call (or after changing posm by hand), which evaluates SP, DC, GFC at the current positions
 * before stepping.  On return rho / acc_grav hold the values at the new positions and acc_sph
 * the corrector's hydro terms.  The grid `g` is an input (fixed domain, L158); particles
 * outside it are clamped into boundary cells, which keeps the search correct.                */
int sph_step(float* posm, float* vele, int64_t n_gas, int64_t n_halo, const sph_params* p /*HOST*/,
             const sph_grid* g /*HOST*/, float dt, int first,
             float* rho, float* acc_sph, float* acc_grav, void* ws, size_t ws_bytes, void* stream);

/* Force evaluation only (call stack (2) of DESIGN.md): SP, DC, GFC, HFC at the current state;
 * fills rho, acc_sph, acc_grav and leaves the carried state valid for sph_step(first = 0).   */
int sph_evaluate(const float* posm, const float* vele, int64_t n_gas, int64_t n_halo,
                 const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/,
                 float* rho, float* acc_sph, float* acc_grav, void* ws, size_t ws_bytes, void* stream);

/* Modified CFL step, Eq. 17 (L125-129):
 *   dt = C_CFL min_i  s_i / ( c_i^max (1 + 1.2 alpha) + 1.2 beta mu_i^max + sqrt( s_i (|Q_i| + |E_i|) ) )
 * over the gas particles, with, over the neighbours j of i (same FP32 cutoff predicate as everywhere,
 * j != i, pairs at zero separation skipped as in A9):
 *   s_i = min_j |r_i - r_j|,  c_i^max = max_j (c_i + c_j)/2,  mu_i^max = max_j |mu_ij|  (mu_ij of L97; A23),
 *   Q_i = acc_sph[i].xyz + acc_grav[i].xyz (right-hand side of Eq. 10),  E_i = acc_sph[i].w (Eq. 11).
 * A gas particle without neighbours takes s_i = 2h, c^max = c_i, mu^max = 0 (A22).  rho, acc_sph,
 * acc_grav are the arrays the last sph_evaluate / sph_step left behind; perm / cell_start the grid
 * of the same positions.  dt_out: DEVICE, one float (+inf if n_gas = 0).  dt_particle: DEVICE
 * [n_gas], the bracket of Eq. 17 per particle WITHOUT C_CFL, or NULL.  The minimum is taken with
 * integer atomics on the float bit pattern: exact and order-independent.  The terms s, c^max, mu^max are
 * gathered "inside the HFC neighbour loop": this call runs the forces walk (the same kernels as sph_forces, in their
 * CFL instantiation) and discards its sums; sph_step_cfl below gets them from the step's own HFC(predictor).  */
int sph_cfl_dt(const float* posm, const float* vele, const float* rho, const float* acc_sph, const float* acc_grav,
               int64_t n_gas, const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/,
               const uint32_t* perm, const uint32_t* cell_start, float c_cfl,
               float* dt_out /*[1]*/, float* dt_particle /*[n_gas] or NULL*/,
               void* ws, size_t ws_bytes, void* stream);

/* End-to-end entry point with HOST buffers: copies posm / vele to the device, derives the grid
 * from the gas bounding box, runs `n_steps` steps (first = 1 on the first), copies posm, vele,
 * rho, acc_sph, acc_grav back (any output pointer may be NULL) and synchronises.  Allocates and
 * frees its own device memory.  All pointers HOST.                                           */
int sph_step_host(float* posm /*HOST*/, float* vele /*HOST*/, int64_t n_gas, int64_t n_halo,
                  const sph_params* p /*HOST*/, float dt, int n_steps,
                  float* rho /*HOST*/, float* acc_sph /*HOST*/, float* acc_grav /*HOST*/);

/* Persistent variant of the above for repeated end-to-end calls: device buffers are created once. */
typedef struct sph_host_ctx sph_host_ctx;
int sph_host_ctx_create(int64_t n_gas, int64_t n_halo, sph_host_ctx** out /*HOST*/);
/* first != 0: seed the carried state from the uploaded positions (as sph_step).  first == 0: the
 * caller asserts posm / vele are exactly what the previous call on this ctx returned, so the
 * carried rho / acc_grav / grid inside the ctx are still valid and only the steps are run.    */
int sph_host_ctx_step(sph_host_ctx* ctx, float* posm /*HOST*/, float* vele /*HOST*/, const sph_params* p /*HOST*/,
                      float dt, int n_steps, int first, float* rho /*HOST*/, float* acc_sph /*HOST*/,
                      float* acc_grav /*HOST*/);
int sph_host_ctx_destroy(sph_host_ctx* ctx);

/* Test helper: explicit neighbour sets N(i) = { j gas, j != i, d2 < (2h)^2 } in CSR form, every
 * list ascending in original index.  nbr_count[n_gas], nbr_offset[n_gas+1] are always written;
 * nbr_index only if nbr_capacity >= nbr_offset[n_gas], else SPH_ERR_WORKSPACE is returned and
 * nbr_offset[n_gas] tells the needed capacity.  SYNCHRONISES `stream`.                        */
int sph_neighbour_lists(const float* posm, int64_t n_gas, float h, const sph_grid* g /*HOST*/,
                        const uint32_t* perm, const uint32_t* cell_start,
                        uint32_t* nbr_count, uint64_t* nbr_offset, uint32_t* nbr_index, uint64_t nbr_capacity,
                        void* ws, size_t ws_bytes, void* stream);

/* ---- per-particle smoothing lengths (L82) ---------------------------------------
 * hsml[n_gas] (DEVICE, float): h_i.  The effective length of a pair is h_ij = (h_i + h_j)/2 (L82) in W (Eq. 7-8),
 * in grad W_p (L95) and in mu_ij (L97); (i, j) is a neighbour pair iff d2 < fl(fl(h_i + h_j)^2), FP32 like the
 * global cutoff (reading A24; equal to it when h_i = h_j = h).  In these calls p->h is the CAP h_max of the
 * lengths: the grid needs cell >= 2 h_max for the 3x3x3 stencil (that is what the paper's per-cell hmaxCell
 * array, L164, provides for a finer grid), and every hsml[i] must be <= p->h.  A larger value (or a NaN) would lose
 * neighbours; the kernel that brings the lengths into cell order raises SPH_STATUS_HSML_ABOVE_CAP in the workspace's
 * status word, which sph_workspace_status() reads back (no synchronisation on the step path itself).
 *
 * sph_smoothing_lengths: hsml[i] = min(sigma (m_i / rho_i)^(1/3), h_max)        (L82; reading A25)
 * sph_density_h / sph_forces_h / sph_evaluate_h / sph_neighbour_lists_h: as the calls without _h.
 * sph_step_h: as sph_step; additionally, if sigma > 0, hsml is renewed from the refined density right after DC at
 *   r(t+dt) (which itself used the old lengths) and the new lengths serve the corrector and the next step
 *   (reading A26); sigma = 0 keeps hsml fixed.  hsml = NULL is exactly sph_step.                            */
int sph_smoothing_lengths(const float* posm, const float* rho, int64_t n_gas, float sigma, float h_max,
                          float* hsml /*[n_gas]*/, void* stream);
int sph_density_h(const float* posm, const float* hsml, int64_t n_gas, const sph_params* p /*HOST*/,
                  const sph_grid* g /*HOST*/, const uint32_t* perm, const uint32_t* cell_start, float* rho,
                  void* ws, size_t ws_bytes, void* stream);
int sph_forces_h(const float* posm, const float* vele, const float* rho, const float* hsml, int64_t n_gas,
                 const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/, const uint32_t* perm,
                 const uint32_t* cell_start, float* acc_sph, void* ws, size_t ws_bytes, void* stream);
int sph_evaluate_h(const float* posm, const float* vele, const float* hsml, int64_t n_gas, int64_t n_halo,
                   const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/, float* rho, float* acc_sph,
                   float* acc_grav, void* ws, size_t ws_bytes, void* stream);
int sph_step_h(float* posm, float* vele, float* hsml, int64_t n_gas, int64_t n_halo, const sph_params* p /*HOST*/,
               const sph_grid* g /*HOST*/, float sigma, float dt, int first, float* rho, float* acc_sph,
               float* acc_grav, void* ws, size_t ws_bytes, void* stream);
/* One predictor-corrector step whose size comes from Eq. 17 (L125-129): as sph_step_h, but the step taken is
 *   dt = min(dt_max, C_CFL min_i [ s_i / (c_i^max (1 + 1.2 alpha) + 1.2 beta mu_i^max + sqrt(s_i (|Q_i| + |E_i|))) ])
 * with the bracket evaluated over the gas particles at the time layer the step starts from: s_i, c_i^max, mu_i^max are
 * reduced by HFC(predictor) itself over its accepted pairs, Q_i and E_i are its results (+ the carried a_grav).  The
 * minimum is taken on the device and read by the update kernels from device memory: no host read-back, the call stays
 * asynchronous and graph-capturable.  dt_used: DEVICE, one float, the step taken.  hsml may be NULL (one global h);
 * with hsml, mu_ij uses h_ij and a particle without a neighbour takes s = 2 h_i.  Without gas the step is dt_max.
 * c_cfl > 0 (the paper: 0.5 <~ C_CFL < 1), dt_max > 0.                                                             */
int sph_step_cfl(float* posm, float* vele, float* hsml, int64_t n_gas, int64_t n_halo, const sph_params* p /*HOST*/,
                 const sph_grid* g /*HOST*/, float sigma, float c_cfl, float dt_max, int first, float* rho,
                 float* acc_sph, float* acc_grav, float* dt_used /*DEVICE [1]*/, void* ws, size_t ws_bytes, void* stream);

int sph_neighbour_lists_h(const float* posm, const float* hsml, int64_t n_gas, float h_max, const sph_grid* g /*HOST*/,
                          const uint32_t* perm, const uint32_t* cell_start, uint32_t* nbr_count,
                          uint64_t* nbr_offset, uint32_t* nbr_index, uint64_t nbr_capacity,
                          void* ws, size_t ws_bytes, void* stream);

/* ---- the stages of a step, target slices and shares, for the N/k-per-GPU decomposition (L133-139) ----
 * The paper gives each of k GPUs N/k particles and copies the other GPUs' particles over before GFC (L139).  Here every
 * GPU keeps the whole (replicated) state and computes only its part of the O(N^2) stage — gravity, 99.8 % of the step.
 * The part has two forms, by the gravity kernel the device chooses: on the pair-symmetric path a
 * SHARE of the unordered-pair work items, whose 64-bit fixed-point sums the caller adds over the GPUs (one integer SUM
 * all-reduce, 24 B x N); on the one-sided path a TARGET SLICE [i0, i1) against all N sources, whose acceleration rows the
 * caller gathers (one all-gather, 16 B x N/k per GPU).  See sph_position_share below;
 * paper_1807_08116_b200/sharded.py (ShardedSimulation) drives it with torch.distributed / NCCL and issues the one
 * collective the chosen path needs.  All GPUs run the O(N) and SPH stages redundantly — they are deterministic, so the
 * replicas stay bitwise identical.
 *
 * nbody_pp_gravity_slice: Eq. 4 for targets [i0, i1) only; rows outside the slice of acc_grav are not touched.
 * sph_position_slice:     SP, DC (+ renewal of hsml if sigma > 0, as in sph_step_h), GFC for targets [i0, i1):
 *                         everything that depends on r only (L123).  hsml may be NULL (global h).
 * sph_predict:            HFC(predictor) + SU(predictor), Eqs. 10-14; needs rho and the COMPLETE acc_grav at r(t).
 * sph_correct:            HFC(corrector) + SU(corrector), Eqs. 10-11, 15-16; needs rho and the COMPLETE acc_grav at
 *                         r(t+dt).
 * sph_step_h(first) == [first: sph_position_slice(sigma = 0, 0, N)] ; sph_predict ; sph_position_slice(sigma, 0, N) ;
 *                      sph_correct  — the same code path, so one GPU with the full slice reproduces sph_step bit for bit.
 * The workspace is the carried state between these calls exactly as for sph_step.                                    */
int nbody_pp_gravity_slice(const float* posm, int64_t n_total, int64_t i0, int64_t i1, float G, float delta,
                           float* acc_grav /*[n_total][4]*/, void* ws, size_t ws_bytes, void* stream);
int sph_position_slice(const float* posm, float* hsml /*or NULL*/, float sigma, int64_t n_gas, int64_t n_halo,
                       int64_t i0, int64_t i1, const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/,
                       float* rho, float* acc_grav, void* ws, size_t ws_bytes, void* stream);

/* One GPU's SHARE of the position-only stage (NEXT-4: k GPUs, N/k particles each): SP and DC in full
 * (O(N), replicated), and rank `rank` of `world`'s part of the Eq. 4 evaluation (L47).  Which gravity kernel runs is
 * decided on the device, so the share has two forms and the caller exchanges BOTH before calling the finish:
 *   - one-sided path: targets [i0, i1) against all sources -> acc_grav rows [i0, i1) (other rows untouched);
 *     exchange = all-gather of the row slices;
 *   - pair-symmetric path (delta > 0, N >= 32768, positive masses, fixed-point range fits): the work items
 *     rank, rank + world, ... of the unordered-pair decomposition -> 64-bit fixed-point sums in the workspace region
 *     sph_workspace_gravity_sums() reports (zeroed by this call; acc_grav not written);
 *     exchange = integer SUM all-reduce of that region (exact: the result is bit for bit the same for every world size).
 * nbody_pp_gravity_finish then writes acc_grav rows [0, n) from the summed region if the pair-symmetric path was taken
 * and does nothing otherwise.  world = 1, [i0, i1) = [0, n): share + finish is sph_position_slice on the full range.
 * Errors: SPH_ERR_ARG (world < 1, rank outside [0, world), bad slice, null / misaligned pointers), SPH_ERR_GRID,
 * SPH_ERR_WORKSPACE, SPH_ERR_UNSUPPORTED (delta < 0), SPH_ERR_CUDA.  Asynchronous on `stream`.                        */
int sph_position_share(const float* posm, float* hsml /*or NULL*/, float sigma, int64_t n_gas, int64_t n_halo, int rank,
                       int world, int64_t i0, int64_t i1, const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/,
                       float* rho, float* acc_grav, void* ws, size_t ws_bytes, void* stream);
/* The gravity part alone (workspace sized for n_gas = 0). */
int nbody_pp_gravity_share(const float* posm, int64_t n_total, int rank, int world, int64_t i0, int64_t i1, float G,
                           float delta, float* acc_grav, void* ws, size_t ws_bytes, void* stream);
/* After the exchange.  (n_gas, n_halo, g) only locate the regions in `ws`: the values the share call was given
 * (n_gas = 0, g = NULL after nbody_pp_gravity_share). */
int nbody_pp_gravity_finish(const float* posm, int64_t n_gas, int64_t n_halo, const sph_grid* g /*HOST or NULL*/, float G,
                            float* acc_grav, void* ws, size_t ws_bytes, void* stream);
/* Byte offset and size, inside a workspace of sph_workspace_bytes(n_gas, n_total, g), of the int64 sums
 * [padded N][3] of the pair-symmetric path.  Host-only, no CUDA call. */
int sph_workspace_gravity_sums(int64_t n_gas, int64_t n_total, const sph_grid* g /*HOST or NULL*/,
                               size_t* offset_host, size_t* bytes_host);

int sph_predict(float* posm, float* vele, const float* hsml /*or NULL*/, int64_t n_gas, int64_t n_halo,
                const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/, float dt,
                const float* rho, float* acc_sph, const float* acc_grav, void* ws, size_t ws_bytes, void* stream);
int sph_correct(float* vele, const float* hsml /*or NULL*/, int64_t n_gas, int64_t n_halo,
                const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/, float dt,
                const float* rho, float* acc_sph, const float* acc_grav, void* ws, size_t ws_bytes, void* stream);

/* ---- The SPH passes shared over the GPUs as well ("SPH by i-slices over a replicated sorted gas
 * array"; every GPU holds all particles before a kernel runs, and computes its own N/k) ----
 * Every rank sorts (SP is O(N), and its result — keys, perm, cell_start, the sorted copies in the workspace — is what
 * the slices are cut from), then computes DC and HFC for ITS targets only: rank `rank` of `world` takes every world-th
 * tile of 128 sorted slots, i.e. tiles rank, rank + world, ...; a populated cell walked by the dense-cell kernels
 * (>= 32 particles) goes, 128 targets at a time, to the rank that owns the first slot of those targets.  Cutting the
 * SORTED order interleaves dense and sparse regions over the ranks.  A target's sum is formed by one rank with the
 * same kernel and in the same order as on one GPU, so the values are bit for bit those of the unsharded calls.
 * The outputs (rho, acc_sph) are written in the caller's particle order: the rank's targets get their values, every
 * other element is ZERO, so the caller completes them with one SUM all-reduce per pass — of the 32-bit patterns as
 * integers (x + 0 + ... + 0, exact; paper_1807_08116_b200/sharded.py does this over NCCL).
 *   sph_position_share_sph: as sph_position_share — SP in full, the rank's share of GFC — but DC for the rank's
 *                           targets only (rho zero elsewhere) and hsml READ only: its renewal needs the complete rho.
 *   sph_renew_hsml:         after rho is complete: h_i = sigma (m_i / rho_i)^(1/3) capped at p->h (L82, A25), and the
 *                           cell-order copy in the workspace that the HFC passes read.  sigma > 0.
 *   sph_forces_share:       HFC (Eqs. 10-11) for the rank's targets from the workspace's sorted state (the last
 *                           position call's), acc_sph zero elsewhere.  Needs the COMPLETE rho.  hsml NULL: one global h.
 *   sph_update:             SU alone, O(N), every rank for all particles: corrector = 0: Eqs. 12-14 (posm, vele
 *                           advanced, the time-t state kept in the workspace); corrector = 1: Eqs. 15-16 (posm unused,
 *                           may be NULL).  Needs the COMPLETE acc_sph and acc_grav.
 * One step on k GPUs = [first: position_share_sph, exchange] ; forces_share, exchange ; update(0) ; position_share_sph,
 * exchange, [renew_hsml] ; forces_share, exchange ; update(1) — the stages of sph_step_h in the same order.  The step
 * criterion of Eq. 17 is not folded into the shared HFC (a MIN over the ranks would be one more collective): the shared
 * step takes dt from the caller.
 * Errors as for sph_position_share; world = 1 gives the unsharded result.  Asynchronous on `stream`.                 */
int sph_position_share_sph(const float* posm, const float* hsml /*or NULL*/, int64_t n_gas, int64_t n_halo, int rank,
                           int world, int64_t i0, int64_t i1, const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/,
                           float* rho, float* acc_grav, void* ws, size_t ws_bytes, void* stream);
int sph_renew_hsml(const float* posm, float* hsml, float sigma, int64_t n_gas, int64_t n_halo,
                   const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/, const float* rho, void* ws, size_t ws_bytes,
                   void* stream);
int sph_forces_share(const float* vele, const float* hsml /*or NULL*/, int64_t n_gas, int64_t n_halo, int rank, int world,
                     const sph_params* p /*HOST*/, const sph_grid* g /*HOST*/, const float* rho, float* acc_sph,
                     void* ws, size_t ws_bytes, void* stream);
int sph_update(float* posm /*or NULL if corrector*/, float* vele, int64_t n_gas, int64_t n_halo,
               const sph_grid* g /*HOST, may be NULL if n_gas == 0*/, float dt, int corrector, const float* acc_sph,
               const float* acc_grav, void* ws, size_t ws_bytes, void* stream);

/* ---- Eq. 4 without any allocation: for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, serving loops, harnesses that forbid it) ----
 * nbody_pp_gravity_static is nbody_pp_gravity with the workspace replaced by a fixed device array inside the library
 * (csrc/noalloc.cu: 12 MiB, held by every GPU that loads the library until the process exits): the caller passes inputs
 * and outputs only, and the call makes no cudaMalloc / cudaFree / allocating library call.  Same kernels, same results
 * bit for bit as nbody_pp_gravity on the same input.
 *   posm     DEVICE [n_total][4] (x, y, z, m), 16-byte aligned      acc_grav  DEVICE [n_total][4] out, 16-byte aligned
 *   n_total  <= nbody_pp_gravity_static_max() (65536); more returns SPH_ERR_WORKSPACE — the fixed scratch is too small,
 *            use nbody_pp_gravity with a caller-owned workspace.
 * ALL calls on a device share the one array: it keeps the last call's contents (what must start at zero is cleared by
 * every call, on its stream), and calls that overlap on the GPU — two streams, two host threads on one device — RACE on
 * it: serialise them.  Other errors: SPH_ERR_ARG, SPH_ERR_UNSUPPORTED (delta < 0), SPH_ERR_CUDA.  Asynchronous on `stream`. */
int64_t nbody_pp_gravity_static_max(void);
int nbody_pp_gravity_static(const float* posm, int64_t n_total, float G, float delta, float* acc_grav, void* stream);

/* Stage timing: after sph_set_profiling(1) every stage the calling thread enqueues is bracketed
 * by CUDA events on the call's stream; sph_get_stage_ms() returns the milliseconds summed over all
 * calls since that switch-on (at most 4096 stage spans) for
 * {sort (a1-a6), density (a7), forces (a8-a9), gravity (a10), update (a11)}.
 * sph_set_profiling() (either value) resets the sums.  Reading the times SYNCHRONISES on the
 * recorded events.  Profiling adds event records only.                                       */
int sph_set_profiling(int on);
int sph_get_stage_ms(float out_ms[5] /*HOST*/);

/* Diagnostic: which variant of the gravity kernel the LAST evaluation enqueued with workspace `ws` (sized for n_gas,
 * n_total and g, as in that call) took.  The choice is made on the device, so this reads the
 * control block back and SYNCHRONISES `stream`.  One-sided: every ordered interaction evaluated (target slices,
 * delta = 0, N < 32768, non-positive masses, or a fixed-point range that would be too coarse); pair-symmetric: every
 * unordered pair evaluated once with fixed-point accumulation.  _UNIFORM / plain PAIR_SYMMETRIC: all masses equal
 * (m_j leaves the loop).  Eq. 4.                                                                   */
enum { SPH_GRAV_ONE_SIDED = 0, SPH_GRAV_ONE_SIDED_UNIFORM = 1, SPH_GRAV_PAIR_SYMMETRIC = 2,
       SPH_GRAV_PAIR_SYMMETRIC_GENERAL = 3 };
int sph_gravity_path(const void* ws /*DEVICE*/, size_t ws_bytes, int64_t n_gas, int64_t n_total,
                     const sph_grid* g /*HOST, may be NULL if n_gas == 0*/, int* path_host /*HOST*/, void* stream);

/* Status word of a workspace: bits raised on the device by the calls that ran with `ws` (sized for n_gas, n_total and g,
 * as in those calls) since the word was last read.  Reads it back, clears it and SYNCHRONISES `stream`.
 * SPH_STATUS_HSML_ABOVE_CAP: a per-particle smoothing length (L82) exceeded the cap p->h that sized the cells (or was NaN):
 * the neighbour sets of the calls since the last read are incomplete.  The word lives in the first 256 bytes of the
 * workspace: zero those once in a new workspace for it to start clear (nothing else in a workspace needs initialising). */
enum { SPH_STATUS_HSML_ABOVE_CAP = 1 };
int sph_workspace_status(void* ws /*DEVICE*/, size_t ws_bytes, int64_t n_gas, int64_t n_total,
                         const sph_grid* g /*HOST, may be NULL if n_gas == 0*/, uint32_t* status_host /*HOST*/, void* stream);

/* Diagnostic: how many work items the LAST forces / grid-building call enqueued with workspace `ws` (sized for
 * n_gas, n_total and g, as in that call) handed to the dense-cell walk of the neighbour passes (DESIGN.md section 5.3:
 * cells holding at least 32 particles, 128 targets per item; the DC / HFC sums of PAPER.md L143-145, L207 over the cell
 * lists).  0 means every particle was walked by the thread-per-slot kernels.  Reads the counter back and SYNCHRONISES
 * `stream`.                                                                                                        */
int sph_dense_items(const void* ws /*DEVICE*/, size_t ws_bytes, int64_t n_gas, int64_t n_total,
                    const sph_grid* g /*HOST*/, uint32_t* items_host /*HOST*/, void* stream);

/* Number of kernel launches this library has enqueued in the calling process since load. */
int64_t sph_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* SPH_B200_H */
