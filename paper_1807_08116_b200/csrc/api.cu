// api.cu — the extern "C" boundary declared in include/sph_b200.h: argument checks, workspace
// carving, stage sequencing and optional per-stage CUDA-event timing.  No arithmetic of the method.
#include "common.cuh"

using namespace sphb;

namespace {

// ---- per-stage timing (sph_set_profiling) -------------------------------------------------------
enum Stage { ST_SORT = 0, ST_DENSITY, ST_FORCES, ST_GRAVITY, ST_UPDATE, ST_COUNT };
constexpr int kMaxSpans = 4096;   // spans accumulate over calls until sph_set_profiling() resets them
struct Prof {
    bool on = false;
    cudaEvent_t ev[2 * kMaxSpans];
    int made = 0;                 // events created so far (lazily, two per span)
    int n = 0;
    int stage[kMaxSpans];
};
thread_local Prof g_prof;

struct Span {
    cudaStream_t st;
    int idx = -1;
    Span(int stage, cudaStream_t s) : st(s) {
        Prof& p = g_prof;
        if (!p.on || p.n >= kMaxSpans) return;
        while (p.made < 2 * (p.n + 1)) cudaEventCreate(&p.ev[p.made++]);
        idx = p.n++;
        p.stage[idx] = stage;
        cudaEventRecord(p.ev[2 * idx], st);
    }
    ~Span() {
        if (idx >= 0) cudaEventRecord(g_prof.ev[2 * idx + 1], st);
    }
};

bool bad_count(int64_t n) { return n < 0 || n >= (1ll << 31); }

int check_params(const sph_params* p, bool need_h) {
    if (!p) return SPH_ERR_ARG;
    if (need_h && !(p->h > 0.f)) return SPH_ERR_ARG;
    if (p->delta < 0.f) return SPH_ERR_UNSUPPORTED;
    return SPH_OK;
}

// SP + DC + GFC at the current positions: everything that depends on r only (L123, A11).
// hsml != NULL (NEXT-2): per-particle smoothing lengths; with sigma > 0 they are renewed from the refined density
// right after DC, h_i = min(sigma (m_i/rho_i)^(1/3), p->h) (L82, readings A25/A26), and re-gathered into cell order.
// world == 0: a one-GPU call (targets [i0, i1), complete on return).  world >= 1: rank's SHARE of the gravity evaluation
// (gravity_share); the caller exchanges and then calls nbody_pp_gravity_finish.
int position_only(const float4* posm, float* hsml, float sigma, int64_t n_gas, int64_t n_total, int64_t i0, int64_t i1,
                  const sph_params* p, const sph_grid* g, float* rho, float4* acc_grav, const Workspace& w,
                  cudaStream_t st, int rank = 0, int world = 0, bool share_dc = false) {
    // share_dc: DC for the rank's targets only (common.cuh: Shard), rho = 0 for the others — the caller adds rho over the ranks
    const Shard sh = share_dc ? Shard{(uint32_t)rank, (uint32_t)world} : Shard{0u, 1u};
    if (n_gas > 0) {
        {
            Span sp(ST_SORT, st);
            SPHB_TRY(grid_build(posm, n_gas, g, w.key, w.perm, w.cell_count, w.cell_start, w.rank_u, w.tmp, w.tile_sums,
                                w.posm_s, &w.dense, st));
            if (hsml) SPHB_TRY(gather_sorted_h(hsml, w.perm, n_gas, p->h, w.status, w.h_s, st));
        }
        {
            Span sp(ST_DENSITY, st);
            if (sh.world > 1u) SPHB_CUDA(cudaMemsetAsync(rho, 0, (size_t)n_gas * sizeof(float), st));
            SPHB_TRY(density_sorted(w.posm_s, hsml ? w.h_s : nullptr, w.perm, w.cell_start, n_gas, p, g, &w.dense, rho, st, sh));
            if (hsml && sigma > 0.f) {
                SPHB_TRY(smoothing_lengths(posm, rho, n_gas, sigma, p->h, hsml, st));
                SPHB_TRY(gather_sorted_h(hsml, w.perm, n_gas, p->h, w.status, w.h_s, st));
            }
        }
    }
    {
        Span sp(ST_GRAVITY, st);
        if (world == 0)
            SPHB_TRY(gravity(posm, n_total, i0, i1, p->G, p->delta, acc_grav, w.src_pk, w.grav_part, w.grav_acc64, w.grav_flag, st));   // GFC
        else
            SPHB_TRY(gravity_share(posm, n_total, i0, i1, rank, world, true, p->G, p->delta, acc_grav, w.src_pk, w.grav_part,
                                   w.grav_acc64, w.grav_flag, st));
    }
    return SPH_OK;
}

int hydro(const float4* vele, const float* rho, bool varh, int64_t n_gas, const sph_params* p, const sph_grid* g,
          float4* acc_sph, const Workspace& w, cudaStream_t st, const CflArgs* cfl = nullptr, Shard sh = Shard{0u, 1u}) {
    if (n_gas <= 0) return SPH_OK;
    Span sp(ST_FORCES, st);
    if (sh.world > 1u) SPHB_CUDA(cudaMemsetAsync(acc_sph, 0, (size_t)n_gas * sizeof(float4), st));
    return forces_sorted(w.posm_s, vele, rho, varh ? w.h_s : nullptr, w.perm, w.cell_start, n_gas, p, g, &w.dense, cfl,
                         w.velr_s, w.pc_s, acc_sph, st, sh);
}

int check_state_args(const void* posm, const void* vele, int64_t n_gas, int64_t n_halo, const sph_params* p,
                     const sph_grid* g, const void* rho, const void* acc_sph, const void* acc_grav, void* ws,
                     size_t ws_bytes) {
    if (bad_count(n_gas) || bad_count(n_halo) || bad_count(n_gas + n_halo)) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, n_gas > 0));
    if (n_gas + n_halo > 0 && (!posm || !vele || !acc_grav || !aligned16(posm) || !aligned16(vele) || !aligned16(acc_grav)))
        return SPH_ERR_ARG;
    if (n_gas > 0) {
        if (!rho || !acc_sph || !aligned16(acc_sph)) return SPH_ERR_ARG;
        SPHB_TRY(check_grid(g, p->h));
    }
    if (!ws || (reinterpret_cast<uintptr_t>(ws) & 255u)) return SPH_ERR_ARG;
    if (ws_bytes < carve(nullptr, n_gas, n_gas + n_halo, n_gas > 0 ? g : nullptr).bytes) return SPH_ERR_WORKSPACE;
    return SPH_OK;
}

}  // namespace

extern "C" {

int sph_last_cuda_error(void) { return g_last_cuda_error; }
int64_t sph_launch_count(void) { return g_launch_count; }

int sph_set_profiling(int on) {
    g_prof.on = on != 0;
    g_prof.n = 0;
    return SPH_OK;
}

int sph_get_stage_ms(float out_ms[5]) {
    if (!out_ms) return SPH_ERR_ARG;
    for (int s = 0; s < ST_COUNT; ++s) out_ms[s] = 0.f;
    Prof& p = g_prof;
    for (int i = 0; i < p.n; ++i) {
        SPHB_CUDA(cudaEventSynchronize(p.ev[2 * i + 1]));
        float ms = 0.f;
        SPHB_CUDA(cudaEventElapsedTime(&ms, p.ev[2 * i], p.ev[2 * i + 1]));
        out_ms[p.stage[i]] += ms;
    }
    return SPH_OK;
}

size_t sph_workspace_bytes(int64_t n_gas, int64_t n_total, const sph_grid* g) {
    if (bad_count(n_gas) || bad_count(n_total) || n_gas > n_total) return 0;
    if (n_gas > 0 && (!g || check_grid(g, 0.f) != SPH_OK)) return 0;
    size_t b = carve(nullptr, n_gas, n_total, n_gas > 0 ? g : nullptr).bytes;
    return b < 4096 ? 4096 : b;
}

int sph_grid_from_bbox(const float* posm, int64_t n_gas, float h, sph_grid* out, void* ws, size_t ws_bytes,
                       void* stream) {
    if (!posm || !out || !ws || n_gas <= 0 || bad_count(n_gas) || !(h > 0.f) || !aligned16(posm)) return SPH_ERR_ARG;
    if (ws_bytes < 256 + 8 * sizeof(float)) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    float* bb = reinterpret_cast<float*>(static_cast<char*>(ws) + 256);   // behind the status block (Workspace::bbox)
    SPHB_TRY(bbox_gas(reinterpret_cast<const float4*>(posm), n_gas, bb, st));
    float host[6];
    SPHB_CUDA(cudaMemcpyAsync(host, bb, sizeof(host), cudaMemcpyDeviceToHost, st));
    SPHB_CUDA(cudaStreamSynchronize(st));
    // A7, FP32 with one rounding per operation (volatile keeps the host compiler from fusing)
    volatile float two_h = 2.0f * h;
    volatile float cell = two_h * 1.001953125f;   // 1 + 2^-9
    volatile float inv = 1.0f / cell;
    double m = 1.0;
    for (int a = 0; a < 3; ++a) {
        volatile float ext = host[3 + a] - host[a];
        volatile float c = ext * inv;
        if (!(c < 4096.0f)) return SPH_ERR_GRID;
        out->origin[a] = host[a];
        out->dims[a] = (int32_t)c + 1;
        if (out->dims[a] > 4096) return SPH_ERR_GRID;
        m *= out->dims[a];
    }
    if (m >= 2147483648.0) return SPH_ERR_GRID;
    out->cell = cell;
    out->inv_cell = inv;
    return SPH_OK;
}

int sph_build_grid(const float* posm, int64_t n_gas, const sph_grid* g, uint32_t* key, uint32_t* perm,
                   uint32_t* cell_count, uint32_t* cell_start, void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas) || !g || !cell_count || !cell_start || !ws) return SPH_ERR_ARG;
    if (n_gas > 0 && (!posm || !key || !perm || !aligned16(posm))) return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, 0.f));
    if (reinterpret_cast<uintptr_t>(ws) & 255u) return SPH_ERR_ARG;
    Workspace w = carve(ws, n_gas, n_gas, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    Span sp(ST_SORT, st);
    return grid_build(reinterpret_cast<const float4*>(posm), n_gas, g, key, perm, cell_count, cell_start, w.rank_u, w.tmp,
                      w.tile_sums, nullptr, &w.dense, st);
}

int sph_density(const float* posm, int64_t n_gas, const sph_params* p, const sph_grid* g, const uint32_t* perm,
                const uint32_t* cell_start, float* rho, void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas)) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, true));
    if (n_gas == 0) return SPH_OK;
    if (!posm || !perm || !cell_start || !rho || !ws || !aligned16(posm) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, p->h));
    Workspace w = carve(ws, n_gas, n_gas, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    SPHB_TRY(gather_sorted_pos(reinterpret_cast<const float4*>(posm), perm, n_gas, w.posm_s, st));
    SPHB_TRY(dense_list_from_start(cell_start, g, w.dense, st));
    Span sp(ST_DENSITY, st);
    return density_sorted(w.posm_s, nullptr, perm, cell_start, n_gas, p, g, &w.dense, rho, st);
}

int sph_forces(const float* posm, const float* vele, const float* rho, int64_t n_gas, const sph_params* p,
               const sph_grid* g, const uint32_t* perm, const uint32_t* cell_start, float* acc_sph, void* ws,
               size_t ws_bytes, void* stream) {
    if (bad_count(n_gas)) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, true));
    if (n_gas == 0) return SPH_OK;
    if (!posm || !vele || !rho || !perm || !cell_start || !acc_sph || !ws || !aligned16(posm) || !aligned16(vele) ||
        !aligned16(acc_sph) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, p->h));
    Workspace w = carve(ws, n_gas, n_gas, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    SPHB_TRY(gather_sorted_pos(reinterpret_cast<const float4*>(posm), perm, n_gas, w.posm_s, st));
    SPHB_TRY(dense_list_from_start(cell_start, g, w.dense, st));
    Span sp(ST_FORCES, st);
    return forces_sorted(w.posm_s, reinterpret_cast<const float4*>(vele), rho, nullptr, perm, cell_start, n_gas, p, g, &w.dense,
                         nullptr, w.velr_s, w.pc_s, reinterpret_cast<float4*>(acc_sph), st);
}

int sph_cfl_dt(const float* posm, const float* vele, const float* rho, const float* acc_sph, const float* acc_grav,
               int64_t n_gas, const sph_params* p, const sph_grid* g, const uint32_t* perm, const uint32_t* cell_start,
               float c_cfl, float* dt_out, float* dt_particle, void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas) || !dt_out || !(c_cfl > 0.f)) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, n_gas > 0));
    cudaStream_t st = (cudaStream_t)stream;
    SPHB_TRY(cfl_init(dt_out, __builtin_inff(), st));
    if (n_gas == 0) return SPH_OK;
    if (!posm || !vele || !rho || !acc_sph || !acc_grav || !perm || !cell_start || !ws || !aligned16(posm) ||
        !aligned16(vele) || !aligned16(acc_sph) || !aligned16(acc_grav) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, p->h));
    Workspace w = carve(ws, n_gas, n_gas, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    SPHB_TRY(gather_sorted_pos(reinterpret_cast<const float4*>(posm), perm, n_gas, w.posm_s, st));
    SPHB_TRY(dense_list_from_start(cell_start, g, w.dense, st));
    // the forces walk in its CFL mode, its own sums discarded: |Q_i| and |E_i| come from the caller's arrays
    const CflArgs cfl{c_cfl, reinterpret_cast<const float4*>(acc_sph), reinterpret_cast<const float4*>(acc_grav), dt_particle,
                      reinterpret_cast<unsigned int*>(dt_out)};
    return forces_sorted(w.posm_s, reinterpret_cast<const float4*>(vele), rho, nullptr, perm, cell_start, n_gas, p, g, &w.dense,
                         &cfl, w.velr_s, w.pc_s, nullptr, st);
}

int nbody_pp_gravity_slice(const float* posm, int64_t n_total, int64_t i0, int64_t i1, float G, float delta,
                           float* acc_grav, void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_total) || i0 < 0 || i1 < i0 || i1 > n_total) return SPH_ERR_ARG;
    if (delta < 0.f) return SPH_ERR_UNSUPPORTED;
    if (n_total == 0) return SPH_OK;
    if (!posm || !acc_grav || !ws || !aligned16(posm) || !aligned16(acc_grav) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    Workspace w = carve(ws, 0, n_total, nullptr);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    Span sp(ST_GRAVITY, st);
    return gravity(reinterpret_cast<const float4*>(posm), n_total, i0, i1, G, delta, reinterpret_cast<float4*>(acc_grav),
                   w.src_pk, w.grav_part, w.grav_acc64, w.grav_flag, st);
}

int sph_gravity_path(const void* ws, size_t ws_bytes, int64_t n_gas, int64_t n_total, const sph_grid* g, int* path_host,
                     void* stream) {
    if (!ws || !path_host || bad_count(n_total) || bad_count(n_gas) || (n_gas > 0 && !g)) return SPH_ERR_ARG;
    Workspace w = carve(const_cast<void*>(ws), n_gas, n_total, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    unsigned int ctl[2] = {0u, 0u};   // GravCtl: nonuniform, sym
    cudaStream_t st = (cudaStream_t)stream;
    SPHB_CUDA(cudaMemcpyAsync(ctl, w.grav_flag, sizeof(ctl), cudaMemcpyDeviceToHost, st));
    SPHB_CUDA(cudaStreamSynchronize(st));
    *path_host = ctl[1] != 0u ? (ctl[0] != 0u ? SPH_GRAV_PAIR_SYMMETRIC_GENERAL : SPH_GRAV_PAIR_SYMMETRIC)
                              : (ctl[0] != 0u ? SPH_GRAV_ONE_SIDED : SPH_GRAV_ONE_SIDED_UNIFORM);
    return SPH_OK;
}

int sph_workspace_status(void* ws, size_t ws_bytes, int64_t n_gas, int64_t n_total, const sph_grid* g, uint32_t* status_host,
                         void* stream) {
    if (!ws || !status_host || bad_count(n_total) || bad_count(n_gas) || n_gas > n_total || (n_gas > 0 && !g)) return SPH_ERR_ARG;
    Workspace w = carve(ws, n_gas, n_total, n_gas > 0 ? g : nullptr);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    SPHB_CUDA(cudaMemcpyAsync(status_host, w.status, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    SPHB_CUDA(cudaMemsetAsync(w.status, 0, sizeof(uint32_t), st));
    SPHB_CUDA(cudaStreamSynchronize(st));
    return SPH_OK;
}

int sph_dense_items(const void* ws, size_t ws_bytes, int64_t n_gas, int64_t n_total, const sph_grid* g, uint32_t* items_host,
                    void* stream) {
    if (!ws || !items_host || bad_count(n_total) || bad_count(n_gas) || n_gas <= 0 || !g) return SPH_ERR_ARG;
    Workspace w = carve(const_cast<void*>(ws), n_gas, n_total, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    SPHB_CUDA(cudaMemcpyAsync(items_host, w.dense.ctl, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
    SPHB_CUDA(cudaStreamSynchronize(st));
    return SPH_OK;
}

int nbody_pp_gravity(const float* posm, int64_t n_total, float G, float delta, float* acc_grav, void* ws,
                     size_t ws_bytes, void* stream) {
    return nbody_pp_gravity_slice(posm, n_total, 0, n_total, G, delta, acc_grav, ws, ws_bytes, stream);
}

int sph_evaluate_h(const float* posm, const float* vele, const float* hsml, int64_t n_gas, int64_t n_halo,
                   const sph_params* p, const sph_grid* g, float* rho, float* acc_sph, float* acc_grav, void* ws,
                   size_t ws_bytes, void* stream) {
    SPHB_TRY(check_state_args(posm, vele, n_gas, n_halo, p, g, rho, acc_sph, acc_grav, ws, ws_bytes));
    const int64_t n = n_gas + n_halo;
    if (n == 0) return SPH_OK;
    Workspace w = carve(ws, n_gas, n, n_gas > 0 ? g : nullptr);
    cudaStream_t st = (cudaStream_t)stream;
    float* hs = n_gas > 0 ? const_cast<float*>(hsml) : nullptr;   // sigma = 0: never written
    SPHB_TRY(position_only(reinterpret_cast<const float4*>(posm), hs, 0.f, n_gas, n, 0, n, p, g, rho,
                           reinterpret_cast<float4*>(acc_grav), w, st));
    return hydro(reinterpret_cast<const float4*>(vele), rho, hs != nullptr, n_gas, p, g, reinterpret_cast<float4*>(acc_sph),
                 w, st);
}

int sph_evaluate(const float* posm, const float* vele, int64_t n_gas, int64_t n_halo, const sph_params* p,
                 const sph_grid* g, float* rho, float* acc_sph, float* acc_grav, void* ws, size_t ws_bytes,
                 void* stream) {
    return sph_evaluate_h(posm, vele, nullptr, n_gas, n_halo, p, g, rho, acc_sph, acc_grav, ws, ws_bytes, stream);
}

// ---- the three stages of a step (exposed so that a caller owning several GPUs can put its
// exchange of acc_grav between them); sph_step_h is their composition on one GPU.
int sph_position_slice(const float* posm, float* hsml, float sigma, int64_t n_gas, int64_t n_halo, int64_t i0,
                       int64_t i1, const sph_params* p, const sph_grid* g, float* rho, float* acc_grav, void* ws,
                       size_t ws_bytes, void* stream) {
    if (bad_count(n_gas) || bad_count(n_halo) || bad_count(n_gas + n_halo)) return SPH_ERR_ARG;
    const int64_t n = n_gas + n_halo;
    if (i0 < 0 || i1 < i0 || i1 > n || sigma < 0.f) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, n_gas > 0));
    if (n == 0) return SPH_OK;
    if (!posm || !acc_grav || !aligned16(posm) || !aligned16(acc_grav) || (n_gas > 0 && !rho)) return SPH_ERR_ARG;
    if (n_gas > 0) SPHB_TRY(check_grid(g, p->h));
    if (!ws || (reinterpret_cast<uintptr_t>(ws) & 255u)) return SPH_ERR_ARG;
    Workspace w = carve(ws, n_gas, n, n_gas > 0 ? g : nullptr);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    return position_only(reinterpret_cast<const float4*>(posm), n_gas > 0 ? hsml : nullptr, sigma, n_gas, n, i0, i1, p, g,
                         rho, reinterpret_cast<float4*>(acc_grav), w, (cudaStream_t)stream);
}

int sph_position_share(const float* posm, float* hsml, float sigma, int64_t n_gas, int64_t n_halo, int rank, int world,
                       int64_t i0, int64_t i1, const sph_params* p, const sph_grid* g, float* rho, float* acc_grav,
                       void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas) || bad_count(n_halo) || bad_count(n_gas + n_halo)) return SPH_ERR_ARG;
    const int64_t n = n_gas + n_halo;
    if (world < 1 || rank < 0 || rank >= world || i0 < 0 || i1 < i0 || i1 > n || sigma < 0.f) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, n_gas > 0));
    if (n == 0) return SPH_OK;
    if (!posm || !acc_grav || !aligned16(posm) || !aligned16(acc_grav) || (n_gas > 0 && !rho)) return SPH_ERR_ARG;
    if (n_gas > 0) SPHB_TRY(check_grid(g, p->h));
    if (!ws || (reinterpret_cast<uintptr_t>(ws) & 255u)) return SPH_ERR_ARG;
    Workspace w = carve(ws, n_gas, n, n_gas > 0 ? g : nullptr);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    return position_only(reinterpret_cast<const float4*>(posm), n_gas > 0 ? hsml : nullptr, sigma, n_gas, n, i0, i1, p, g,
                         rho, reinterpret_cast<float4*>(acc_grav), w, (cudaStream_t)stream, rank, world);
}

int nbody_pp_gravity_share(const float* posm, int64_t n_total, int rank, int world, int64_t i0, int64_t i1, float G,
                           float delta, float* acc_grav, void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_total) || world < 1 || rank < 0 || rank >= world || i0 < 0 || i1 < i0 || i1 > n_total) return SPH_ERR_ARG;
    if (delta < 0.f) return SPH_ERR_UNSUPPORTED;
    if (n_total == 0) return SPH_OK;
    if (!posm || !acc_grav || !ws || !aligned16(posm) || !aligned16(acc_grav) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    Workspace w = carve(ws, 0, n_total, nullptr);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    Span sp(ST_GRAVITY, st);
    return gravity_share(reinterpret_cast<const float4*>(posm), n_total, i0, i1, rank, world, true, G, delta,
                         reinterpret_cast<float4*>(acc_grav), w.src_pk, w.grav_part, w.grav_acc64, w.grav_flag, st);
}

int nbody_pp_gravity_finish(const float* posm, int64_t n_gas, int64_t n_halo, const sph_grid* g, float G, float* acc_grav,
                            void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas) || bad_count(n_halo) || bad_count(n_gas + n_halo) || (n_gas > 0 && !g)) return SPH_ERR_ARG;
    const int64_t n = n_gas + n_halo;
    if (n == 0) return SPH_OK;
    if (!posm || !acc_grav || !ws || !aligned16(posm) || !aligned16(acc_grav) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    Workspace w = carve(ws, n_gas, n, n_gas > 0 ? g : nullptr);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    Span sp(ST_GRAVITY, st);
    return gravity_finish(reinterpret_cast<const float4*>(posm), n, G, reinterpret_cast<float4*>(acc_grav), w.grav_acc64,
                          w.grav_flag, st);
}

// ---- the SPH passes shared as well ----
int sph_position_share_sph(const float* posm, const float* hsml, int64_t n_gas, int64_t n_halo, int rank, int world,
                           int64_t i0, int64_t i1, const sph_params* p, const sph_grid* g, float* rho, float* acc_grav,
                           void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas) || bad_count(n_halo) || bad_count(n_gas + n_halo)) return SPH_ERR_ARG;
    const int64_t n = n_gas + n_halo;
    if (world < 1 || rank < 0 || rank >= world || i0 < 0 || i1 < i0 || i1 > n) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, n_gas > 0));
    if (n == 0) return SPH_OK;
    if (!posm || !acc_grav || !aligned16(posm) || !aligned16(acc_grav) || (n_gas > 0 && !rho)) return SPH_ERR_ARG;
    if (n_gas > 0) SPHB_TRY(check_grid(g, p->h));
    if (!ws || (reinterpret_cast<uintptr_t>(ws) & 255u)) return SPH_ERR_ARG;
    Workspace w = carve(ws, n_gas, n, n_gas > 0 ? g : nullptr);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    // sigma = 0: hsml is read only (its renewal needs the complete rho: sph_renew_hsml, after the exchange)
    return position_only(reinterpret_cast<const float4*>(posm), n_gas > 0 ? const_cast<float*>(hsml) : nullptr, 0.f, n_gas, n,
                         i0, i1, p, g, rho, reinterpret_cast<float4*>(acc_grav), w, (cudaStream_t)stream, rank, world, true);
}

int sph_renew_hsml(const float* posm, float* hsml, float sigma, int64_t n_gas, int64_t n_halo, const sph_params* p,
                   const sph_grid* g, const float* rho, void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas) || bad_count(n_halo) || bad_count(n_gas + n_halo) || !(sigma > 0.f)) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, n_gas > 0));
    if (n_gas == 0) return SPH_OK;
    if (!posm || !hsml || !rho || !aligned16(posm) || !ws || (reinterpret_cast<uintptr_t>(ws) & 255u)) return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, p->h));
    Workspace w = carve(ws, n_gas, n_gas + n_halo, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    Span sp(ST_DENSITY, st);
    SPHB_TRY(smoothing_lengths(reinterpret_cast<const float4*>(posm), rho, n_gas, sigma, p->h, hsml, st));
    return gather_sorted_h(hsml, w.perm, n_gas, p->h, w.status, w.h_s, st);
}

int sph_forces_share(const float* vele, const float* hsml, int64_t n_gas, int64_t n_halo, int rank, int world,
                     const sph_params* p, const sph_grid* g, const float* rho, float* acc_sph, void* ws, size_t ws_bytes,
                     void* stream) {
    if (bad_count(n_gas) || bad_count(n_halo) || bad_count(n_gas + n_halo) || world < 1 || rank < 0 || rank >= world)
        return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, n_gas > 0));
    if (n_gas == 0) return SPH_OK;
    if (!vele || !rho || !acc_sph || !aligned16(vele) || !aligned16(acc_sph) || !ws || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, p->h));
    Workspace w = carve(ws, n_gas, n_gas + n_halo, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    return hydro(reinterpret_cast<const float4*>(vele), rho, hsml != nullptr, n_gas, p, g, reinterpret_cast<float4*>(acc_sph), w,
                 (cudaStream_t)stream, nullptr, Shard{(uint32_t)rank, (uint32_t)world});
}

int sph_update(float* posm, float* vele, int64_t n_gas, int64_t n_halo, const sph_grid* g, float dt, int corrector,
               const float* acc_sph, const float* acc_grav, void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas) || bad_count(n_halo) || bad_count(n_gas + n_halo) || (n_gas > 0 && !g)) return SPH_ERR_ARG;
    const int64_t n = n_gas + n_halo;
    if (n == 0) return SPH_OK;
    if (!vele || !acc_grav || (!corrector && !posm) || (n_gas > 0 && !acc_sph) || !aligned16(vele) || !aligned16(acc_grav) ||
        (posm && !aligned16(posm)) || (acc_sph && !aligned16(acc_sph)) || !ws || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    Workspace w = carve(ws, n_gas, n, n_gas > 0 ? g : nullptr);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    Span sp(ST_UPDATE, st);
    if (corrector)
        return update_corrector(reinterpret_cast<float4*>(vele), w.vele0, reinterpret_cast<const float4*>(acc_sph),
                                reinterpret_cast<const float4*>(acc_grav), n_gas, n, dt, nullptr, st);   // Eqs. 15-16
    return update_predictor(reinterpret_cast<float4*>(posm), reinterpret_cast<float4*>(vele), w.vele0,
                            reinterpret_cast<const float4*>(acc_sph), reinterpret_cast<const float4*>(acc_grav), n_gas, n, dt,
                            nullptr, st);                                                                 // Eqs. 12-14
}

int sph_workspace_gravity_sums(int64_t n_gas, int64_t n_total, const sph_grid* g, size_t* offset_host, size_t* bytes_host) {
    if (!offset_host || !bytes_host || bad_count(n_gas) || bad_count(n_total) || n_gas > n_total || (n_gas > 0 && !g))
        return SPH_ERR_ARG;
    Workspace w = carve(nullptr, n_gas, n_total, n_gas > 0 ? g : nullptr);
    *offset_host = w.grav_acc64_off;
    *bytes_host = (size_t)grav_padded(n_total) * 3 * sizeof(long long);
    return SPH_OK;
}

}  // extern "C"

namespace {
// HFC(predictor) + SU(predictor).  c_cfl > 0: the step is min(dt, C_CFL min_i [...]) of Eq. 17, reduced by the forces
// walk itself into *dt_dev (device), which the update kernels then read — no host read-back.
int predict(float* posm, float* vele, const float* hsml, int64_t n_gas, int64_t n_halo, const sph_params* p,
            const sph_grid* g, float dt, float c_cfl, float* dt_dev, const float* rho, float* acc_sph, const float* acc_grav,
            void* ws, size_t ws_bytes, void* stream) {
    SPHB_TRY(check_state_args(posm, vele, n_gas, n_halo, p, g, rho, acc_sph, acc_grav, ws, ws_bytes));
    const int64_t n = n_gas + n_halo;
    if (n == 0) return SPH_OK;
    Workspace w = carve(ws, n_gas, n, n_gas > 0 ? g : nullptr);
    cudaStream_t st = (cudaStream_t)stream;
    float4* as4 = reinterpret_cast<float4*>(acc_sph);
    const bool varh = hsml != nullptr && n_gas > 0;
    if (dt_dev) {
        SPHB_TRY(cfl_init(dt_dev, dt, st));
        const CflArgs cfl{c_cfl, nullptr, reinterpret_cast<const float4*>(acc_grav), nullptr, reinterpret_cast<unsigned int*>(dt_dev)};
        SPHB_TRY(hydro(reinterpret_cast<const float4*>(vele), rho, varh, n_gas, p, g, as4, w, st, &cfl));
    } else {
        SPHB_TRY(hydro(reinterpret_cast<const float4*>(vele), rho, varh, n_gas, p, g, as4, w, st));
    }
    Span sp(ST_UPDATE, st);
    return update_predictor(reinterpret_cast<float4*>(posm), reinterpret_cast<float4*>(vele), w.vele0, as4,
                            reinterpret_cast<const float4*>(acc_grav), n_gas, n, dt, dt_dev, st);   // Eqs. 12-14
}

int correct(float* vele, const float* hsml, int64_t n_gas, int64_t n_halo, const sph_params* p, const sph_grid* g, float dt,
            const float* dt_dev, const float* rho, float* acc_sph, const float* acc_grav, void* ws, size_t ws_bytes,
            void* stream) {
    SPHB_TRY(check_state_args(vele, vele, n_gas, n_halo, p, g, rho, acc_sph, acc_grav, ws, ws_bytes));
    const int64_t n = n_gas + n_halo;
    if (n == 0) return SPH_OK;
    Workspace w = carve(ws, n_gas, n, n_gas > 0 ? g : nullptr);
    cudaStream_t st = (cudaStream_t)stream;
    float4* as4 = reinterpret_cast<float4*>(acc_sph);
    SPHB_TRY(hydro(reinterpret_cast<const float4*>(vele), rho, hsml != nullptr && n_gas > 0, n_gas, p, g, as4, w, st));
    Span sp(ST_UPDATE, st);
    return update_corrector(reinterpret_cast<float4*>(vele), w.vele0, as4, reinterpret_cast<const float4*>(acc_grav),
                            n_gas, n, dt, dt_dev, st);                                       // Eqs. 15-16
}
}  // namespace

extern "C" {

int sph_predict(float* posm, float* vele, const float* hsml, int64_t n_gas, int64_t n_halo, const sph_params* p,
                const sph_grid* g, float dt, const float* rho, float* acc_sph, const float* acc_grav, void* ws,
                size_t ws_bytes, void* stream) {
    return predict(posm, vele, hsml, n_gas, n_halo, p, g, dt, 0.f, nullptr, rho, acc_sph, acc_grav, ws, ws_bytes, stream);
}

int sph_correct(float* vele, const float* hsml, int64_t n_gas, int64_t n_halo, const sph_params* p, const sph_grid* g,
                float dt, const float* rho, float* acc_sph, const float* acc_grav, void* ws, size_t ws_bytes,
                void* stream) {
    return correct(vele, hsml, n_gas, n_halo, p, g, dt, nullptr, rho, acc_sph, acc_grav, ws, ws_bytes, stream);
}

int sph_step_cfl(float* posm, float* vele, float* hsml, int64_t n_gas, int64_t n_halo, const sph_params* p,
                 const sph_grid* g, float sigma, float c_cfl, float dt_max, int first, float* rho, float* acc_sph,
                 float* acc_grav, float* dt_used, void* ws, size_t ws_bytes, void* stream) {
    SPHB_TRY(check_state_args(posm, vele, n_gas, n_halo, p, g, rho, acc_sph, acc_grav, ws, ws_bytes));
    if (sigma < 0.f || !(c_cfl > 0.f) || !(dt_max > 0.f) || !dt_used) return SPH_ERR_ARG;
    const int64_t n = n_gas + n_halo;
    if (n == 0) return SPH_OK;
    if (first)   // seed the carried state: SP, DC, GFC at the current positions
        SPHB_TRY(sph_position_slice(posm, hsml, 0.f, n_gas, n_halo, 0, n, p, g, rho, acc_grav, ws, ws_bytes, stream));
    SPHB_TRY(predict(posm, vele, hsml, n_gas, n_halo, p, g, dt_max, c_cfl, dt_used, rho, acc_sph, acc_grav, ws, ws_bytes, stream));
    SPHB_TRY(sph_position_slice(posm, hsml, sigma, n_gas, n_halo, 0, n, p, g, rho, acc_grav, ws, ws_bytes, stream));
    return correct(vele, hsml, n_gas, n_halo, p, g, dt_max, dt_used, rho, acc_sph, acc_grav, ws, ws_bytes, stream);
}

int sph_step_h(float* posm, float* vele, float* hsml, int64_t n_gas, int64_t n_halo, const sph_params* p,
               const sph_grid* g, float sigma, float dt, int first, float* rho, float* acc_sph, float* acc_grav, void* ws,
               size_t ws_bytes, void* stream) {
    SPHB_TRY(check_state_args(posm, vele, n_gas, n_halo, p, g, rho, acc_sph, acc_grav, ws, ws_bytes));
    if (sigma < 0.f) return SPH_ERR_ARG;
    const int64_t n = n_gas + n_halo;
    if (n == 0) return SPH_OK;
    if (first)   // seed the carried state: SP, DC, GFC at the current positions
        SPHB_TRY(sph_position_slice(posm, hsml, 0.f, n_gas, n_halo, 0, n, p, g, rho, acc_grav, ws, ws_bytes, stream));
    SPHB_TRY(sph_predict(posm, vele, hsml, n_gas, n_halo, p, g, dt, rho, acc_sph, acc_grav, ws, ws_bytes, stream));
    SPHB_TRY(sph_position_slice(posm, hsml, sigma, n_gas, n_halo, 0, n, p, g, rho, acc_grav, ws, ws_bytes, stream));
    return sph_correct(vele, hsml, n_gas, n_halo, p, g, dt, rho, acc_sph, acc_grav, ws, ws_bytes, stream);
}

int sph_step(float* posm, float* vele, int64_t n_gas, int64_t n_halo, const sph_params* p, const sph_grid* g, float dt,
             int first, float* rho, float* acc_sph, float* acc_grav, void* ws, size_t ws_bytes, void* stream) {
    return sph_step_h(posm, vele, nullptr, n_gas, n_halo, p, g, 0.f, dt, first, rho, acc_sph, acc_grav, ws, ws_bytes,
                      stream);
}

int sph_smoothing_lengths(const float* posm, const float* rho, int64_t n_gas, float sigma, float h_max, float* hsml,
                          void* stream) {
    if (bad_count(n_gas) || !(sigma > 0.f) || !(h_max > 0.f)) return SPH_ERR_ARG;
    if (n_gas == 0) return SPH_OK;
    if (!posm || !rho || !hsml || !aligned16(posm)) return SPH_ERR_ARG;
    return smoothing_lengths(reinterpret_cast<const float4*>(posm), rho, n_gas, sigma, h_max, hsml, (cudaStream_t)stream);
}

int sph_density_h(const float* posm, const float* hsml, int64_t n_gas, const sph_params* p, const sph_grid* g,
                  const uint32_t* perm, const uint32_t* cell_start, float* rho, void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas)) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, true));
    if (n_gas == 0) return SPH_OK;
    if (!posm || !hsml || !perm || !cell_start || !rho || !ws || !aligned16(posm) ||
        (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, p->h));
    Workspace w = carve(ws, n_gas, n_gas, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    SPHB_TRY(gather_sorted_pos(reinterpret_cast<const float4*>(posm), perm, n_gas, w.posm_s, st));
    SPHB_TRY(gather_sorted_h(hsml, perm, n_gas, p->h, w.status, w.h_s, st));
    Span sp(ST_DENSITY, st);
    SPHB_TRY(dense_list_from_start(cell_start, g, w.dense, st));
    return density_sorted(w.posm_s, w.h_s, perm, cell_start, n_gas, p, g, &w.dense, rho, st);
}

int sph_forces_h(const float* posm, const float* vele, const float* rho, const float* hsml, int64_t n_gas,
                 const sph_params* p, const sph_grid* g, const uint32_t* perm, const uint32_t* cell_start, float* acc_sph,
                 void* ws, size_t ws_bytes, void* stream) {
    if (bad_count(n_gas)) return SPH_ERR_ARG;
    SPHB_TRY(check_params(p, true));
    if (n_gas == 0) return SPH_OK;
    if (!posm || !vele || !rho || !hsml || !perm || !cell_start || !acc_sph || !ws || !aligned16(posm) ||
        !aligned16(vele) || !aligned16(acc_sph) || (reinterpret_cast<uintptr_t>(ws) & 255u))
        return SPH_ERR_ARG;
    SPHB_TRY(check_grid(g, p->h));
    Workspace w = carve(ws, n_gas, n_gas, g);
    if (ws_bytes < w.bytes) return SPH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    SPHB_TRY(gather_sorted_pos(reinterpret_cast<const float4*>(posm), perm, n_gas, w.posm_s, st));
    SPHB_TRY(gather_sorted_h(hsml, perm, n_gas, p->h, w.status, w.h_s, st));
    SPHB_TRY(dense_list_from_start(cell_start, g, w.dense, st));
    Span sp(ST_FORCES, st);
    return forces_sorted(w.posm_s, reinterpret_cast<const float4*>(vele), rho, w.h_s, perm, cell_start, n_gas, p, g, &w.dense,
                         nullptr, w.velr_s, w.pc_s, reinterpret_cast<float4*>(acc_sph), st);
}

}  // extern "C"
