// step.cu — (a11) the System Update kernels (Eqs. 12-16), the workspace layout
// and the internal step / evaluate sequences (reading A11).
#include "common.cuh"

namespace sphb {

thread_local int g_last_cuda_error = 0;
std::atomic<long long> g_launch_count{0};

int num_sms() {   // of the CURRENT device (a process may drive several)
    static int n_dev[64] = {0};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    if (n_dev[dev] == 0) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        n_dev[dev] = n;
    }
    return n_dev[dev];
}

// ---------------------------------------------------------------- workspace
Workspace carve(void* base, int64_t n_gas, int64_t n_total, const sph_grid* g) {
    Workspace w;
    size_t off = 0;
    auto take = [&](size_t bytes) -> void* {
        void* p = base ? static_cast<char*>(base) + off : nullptr;
        off += round_up(bytes ? bytes : 1, 256);
        return p;
    };
    const int64_t M = (g && n_gas > 0) ? grid_cells(g) : 0;
    const size_t ng = (size_t)(n_gas > 0 ? n_gas : 0), nt = (size_t)(n_total > 0 ? n_total : 0);
    w.status = (unsigned int*)take(256);   // offset 0: the one block a caller zeroes in a new workspace
    w.bbox = (float*)take(8 * sizeof(float));
    w.key = (uint32_t*)take(ng * 4);
    w.rank_u = (uint32_t*)take(ng * 4);
    w.tmp = (uint32_t*)take(ng * 4);
    w.perm = (uint32_t*)take(ng * 4);
    w.cell_count = (uint32_t*)take((size_t)M * 4);
    w.tile_sums = (uint32_t*)take((size_t)(cdiv(M > 0 ? M : 1, 4096) + 1) * 4);   // right behind count[M]: one memset zeroes both (grid.cu)
    w.cell_start = (uint32_t*)take((size_t)(M + 1) * 4);
    w.posm_s = (float4*)take(ng * 16);
    w.velr_s = (float4*)take(ng * 16);
    w.pc_s = (float2*)take(ng * 8);
    w.h_s = (float*)take(ng * 4);
    w.dense.ctl = (unsigned int*)take(256);
    w.dense.items = (DenseItem*)take(dense_capacity((int64_t)ng) * sizeof(DenseItem));
    w.src_pk = (float4*)take((size_t)grav_padded(n_total) * 16);
    w.grav_part = (float4*)take((size_t)grav_splits(n_total) * nt * 16);
    w.grav_acc64_off = off;
    w.grav_acc64 = (long long*)take((size_t)grav_padded(n_total) * 3 * sizeof(long long));
    w.grav_flag = (unsigned int*)take(256);
    w.vele0 = (float4*)take(nt * 16);
    w.bytes = off;
    return w;
}

// ---------------------------------------------------------------- (a11) System Update
// Predictor, Eqs. 12-14:  v~ = v + dt Q ; e~ = e + dt E ; r(t+dt) = r + dt/2 (v~ + v).
// Q = a_sph + a_grav for gas, a_grav for halo (Eq. 10); E = de/dt (Eq. 11).  v(t), e(t) are saved.
__global__ void __launch_bounds__(256) k_update_pred(float4* __restrict__ posm, float4* __restrict__ vele,
                                                     float4* __restrict__ vele0, const float4* __restrict__ acc_sph,
                                                     const float4* __restrict__ acc_grav, int n_gas, int n, float dt_arg,
                                                     const float* __restrict__ dt_dev) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float dt = dt_dev ? *dt_dev : dt_arg;
    float4 r = posm[i];
    const float4 v = vele[i];
    float4 q = acc_grav[i];
    float e_rate = 0.f;
    if (i < n_gas) {
        const float4 a = acc_sph[i];
        q.x += a.x;
        q.y += a.y;
        q.z += a.z;
        e_rate = a.w;
    }
    float4 vt;
    vt.x = fmaf(dt, q.x, v.x);
    vt.y = fmaf(dt, q.y, v.y);
    vt.z = fmaf(dt, q.z, v.z);
    vt.w = fmaf(dt, e_rate, v.w);
    const float hdt = 0.5f * dt;
    r.x = fmaf(hdt, vt.x + v.x, r.x);
    r.y = fmaf(hdt, vt.y + v.y, r.y);
    r.z = fmaf(hdt, vt.z + v.z, r.z);
    vele0[i] = v;
    vele[i] = vt;
    posm[i] = r;
}

// Corrector, Eqs. 15-16:  v = (v(t) + v~)/2 + dt/2 Q~ ; e = (e(t) + e~)/2 + dt/2 E~.
__global__ void __launch_bounds__(256) k_update_corr(float4* __restrict__ vele, const float4* __restrict__ vele0,
                                                     const float4* __restrict__ acc_sph,
                                                     const float4* __restrict__ acc_grav, int n_gas, int n, float dt_arg,
                                                     const float* __restrict__ dt_dev) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float dt = dt_dev ? *dt_dev : dt_arg;
    const float4 vt = vele[i], v0 = vele0[i];
    float4 q = acc_grav[i];
    float e_rate = 0.f;
    if (i < n_gas) {
        const float4 a = acc_sph[i];
        q.x += a.x;
        q.y += a.y;
        q.z += a.z;
        e_rate = a.w;
    }
    const float hdt = 0.5f * dt;
    float4 o;
    o.x = fmaf(hdt, q.x, 0.5f * (v0.x + vt.x));
    o.y = fmaf(hdt, q.y, 0.5f * (v0.y + vt.y));
    o.z = fmaf(hdt, q.z, 0.5f * (v0.z + vt.z));
    o.w = fmaf(hdt, e_rate, 0.5f * (v0.w + vt.w));
    vele[i] = o;
}

int update_predictor(float4* posm, float4* vele, float4* vele0, const float4* acc_sph, const float4* acc_grav,
                     int64_t n_gas, int64_t n_total, float dt, const float* dt_dev, cudaStream_t st) {
    if (n_total <= 0) return SPH_OK;
    k_update_pred<<<(unsigned)cdiv(n_total, 256), 256, 0, st>>>(posm, vele, vele0, acc_sph, acc_grav, (int)n_gas,
                                                               (int)n_total, dt, dt_dev);
    SPHB_LAUNCHED();
    return SPH_OK;
}

int update_corrector(float4* vele, const float4* vele0, const float4* acc_sph, const float4* acc_grav, int64_t n_gas,
                     int64_t n_total, float dt, const float* dt_dev, cudaStream_t st) {
    if (n_total <= 0) return SPH_OK;
    k_update_corr<<<(unsigned)cdiv(n_total, 256), 256, 0, st>>>(vele, vele0, acc_sph, acc_grav, (int)n_gas, (int)n_total,
                                                               dt, dt_dev);
    SPHB_LAUNCHED();
    return SPH_OK;
}

}  // namespace sphb
