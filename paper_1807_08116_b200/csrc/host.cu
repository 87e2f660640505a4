// host.cu — end-to-end entry points that take HOST arrays (include/sph_b200.h: sph_step_host,
// sph_host_ctx_*).  They own their device buffers and a stream, copy in, derive the grid from
// the gas bounding box, call sph_step, copy out and synchronise.  No arithmetic of the method.
#include "common.cuh"

using namespace sphb;

struct sph_host_ctx {
    int64_t n_gas = 0, n_halo = 0;
    float *posm = nullptr, *vele = nullptr, *rho = nullptr, *acc_sph = nullptr, *acc_grav = nullptr;
    void* ws = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t st = nullptr;
    sph_grid grid;          // grid of the last seeding call (first != 0)
    bool seeded = false;
};

namespace {
int ensure_ws(sph_host_ctx* c, size_t need) {
    if (need <= c->ws_bytes) return SPH_OK;
    if (c->ws) SPHB_CUDA(cudaFree(c->ws));
    c->ws = nullptr;
    c->ws_bytes = 0;
    SPHB_CUDA(cudaMalloc(&c->ws, need));
    SPHB_CUDA(cudaMemset(c->ws, 0, 256));   // the status word of a new workspace starts clear
    c->ws_bytes = need;
    return SPH_OK;
}
}  // namespace

extern "C" {

int sph_host_ctx_create(int64_t n_gas, int64_t n_halo, sph_host_ctx** out) {
    if (!out || n_gas < 0 || n_halo < 0 || n_gas + n_halo >= (1ll << 31)) return SPH_ERR_ARG;
    sph_host_ctx* c = new sph_host_ctx();
    c->n_gas = n_gas;
    c->n_halo = n_halo;
    const size_t n = (size_t)(n_gas + n_halo), ng = (size_t)n_gas;
    cudaError_t e = cudaStreamCreateWithFlags(&c->st, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaMalloc((void**)&c->posm, (n ? n : 1) * 16);
    if (e == cudaSuccess) e = cudaMalloc((void**)&c->vele, (n ? n : 1) * 16);
    if (e == cudaSuccess) e = cudaMalloc((void**)&c->acc_grav, (n ? n : 1) * 16);
    if (e == cudaSuccess) e = cudaMalloc((void**)&c->acc_sph, (ng ? ng : 1) * 16);
    if (e == cudaSuccess) e = cudaMalloc((void**)&c->rho, (ng ? ng : 1) * 4);
    if (e == cudaSuccess) e = cudaMalloc(&c->ws, 4096);
    if (e != cudaSuccess) {
        sph_host_ctx_destroy(c);
        return cuda_fail(e);
    }
    c->ws_bytes = 4096;
    *out = c;
    return SPH_OK;
}

int sph_host_ctx_destroy(sph_host_ctx* c) {
    if (!c) return SPH_OK;
    cudaFree(c->posm);
    cudaFree(c->vele);
    cudaFree(c->rho);
    cudaFree(c->acc_sph);
    cudaFree(c->acc_grav);
    cudaFree(c->ws);
    if (c->st) cudaStreamDestroy(c->st);
    delete c;
    return SPH_OK;
}

int sph_host_ctx_step(sph_host_ctx* c, float* posm, float* vele, const sph_params* p, float dt, int n_steps, int first,
                      float* rho, float* acc_sph, float* acc_grav) {
    if (!c || !posm || !vele || !p || n_steps < 0) return SPH_ERR_ARG;
    if (!first && !c->seeded) return SPH_ERR_ARG;
    const int64_t n = c->n_gas + c->n_halo;
    if (n == 0) return SPH_OK;
    cudaStream_t st = c->st;
    SPHB_CUDA(cudaMemcpyAsync(c->posm, posm, (size_t)n * 16, cudaMemcpyHostToDevice, st));
    SPHB_CUDA(cudaMemcpyAsync(c->vele, vele, (size_t)n * 16, cudaMemcpyHostToDevice, st));
    if (first) {
        sph_grid g;
        g.origin[0] = g.origin[1] = g.origin[2] = 0.f;
        g.cell = g.inv_cell = 1.f;
        g.dims[0] = g.dims[1] = g.dims[2] = 1;
        if (c->n_gas > 0) SPHB_TRY(sph_grid_from_bbox(c->posm, c->n_gas, p->h, &g, c->ws, c->ws_bytes, st));
        size_t need = sph_workspace_bytes(c->n_gas, n, c->n_gas > 0 ? &g : nullptr);
        if (need == 0) return SPH_ERR_GRID;
        SPHB_TRY(ensure_ws(c, need));
        c->grid = g;
        c->seeded = true;
    }
    const sph_grid& g = c->grid;   // fixed domain between seedings (L158); outliers are clamped
    for (int s = 0; s < n_steps; ++s)
        SPHB_TRY(sph_step(c->posm, c->vele, c->n_gas, c->n_halo, p, &g, dt, first && s == 0, c->rho, c->acc_sph,
                          c->acc_grav, c->ws, c->ws_bytes, st));
    if (n_steps == 0)
        SPHB_TRY(sph_evaluate(c->posm, c->vele, c->n_gas, c->n_halo, p, &g, c->rho, c->acc_sph, c->acc_grav, c->ws,
                              c->ws_bytes, st));
    SPHB_CUDA(cudaMemcpyAsync(posm, c->posm, (size_t)n * 16, cudaMemcpyDeviceToHost, st));
    SPHB_CUDA(cudaMemcpyAsync(vele, c->vele, (size_t)n * 16, cudaMemcpyDeviceToHost, st));
    if (rho && c->n_gas) SPHB_CUDA(cudaMemcpyAsync(rho, c->rho, (size_t)c->n_gas * 4, cudaMemcpyDeviceToHost, st));
    if (acc_sph && c->n_gas) SPHB_CUDA(cudaMemcpyAsync(acc_sph, c->acc_sph, (size_t)c->n_gas * 16, cudaMemcpyDeviceToHost, st));
    if (acc_grav) SPHB_CUDA(cudaMemcpyAsync(acc_grav, c->acc_grav, (size_t)n * 16, cudaMemcpyDeviceToHost, st));
    SPHB_CUDA(cudaStreamSynchronize(st));
    return SPH_OK;
}

int sph_step_host(float* posm, float* vele, int64_t n_gas, int64_t n_halo, const sph_params* p, float dt, int n_steps,
                  float* rho, float* acc_sph, float* acc_grav) {
    sph_host_ctx* c = nullptr;
    SPHB_TRY(sph_host_ctx_create(n_gas, n_halo, &c));
    int rc = sph_host_ctx_step(c, posm, vele, p, dt, n_steps, 1, rho, acc_sph, acc_grav);
    sph_host_ctx_destroy(c);
    return rc;
}

}  // extern "C"
