/*
 * sph_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU restatement of the hot path of Khrapov & Khoperskov,
 * "Smoothed-Particle Hydrodynamics Models: Implementation Features on GPUs"
 * (arXiv 1807.08116; the text is /root/reference/PAPER.md, cited below as "Lnn").
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.  It shares no code with the CUDA path (no headers, no
 * helpers, no tables); the struct below is this file's own declaration of the grid
 * descriptor of DESIGN.md reading A7.
 *
 * Every sum is the paper's definition written out (brute force over the stated index
 * set), in double.  Particle arrays are double[N][4] = (x,y,z,m) / (vx,vy,vz,e): the
 * Python wrapper widens the FP32 inputs exactly, and the oracle's own free-running
 * trajectories (pins P7/P8) stay in FP64.  The only FP32 arithmetic is
 * where the north star fixes it: the cell key (reading A7) and the cutoff predicate
 * (reading A8, "the cutoff test is done in FP32 on both sides").  OpenMP is used over
 * the *target* index only (each target's sum is still a plain sequential loop), so it
 * changes wall time, not results.
 *
 * Parity unpinned (specifications of this build, not fixed by the paper):
 *   - the softening form of Eq. 4 (reading A1: Plummer, (|dr|^2 + delta^2)^(3/2));
 *   - gamma (reading A6: a parameter, default 5/3);
 *   - the cell geometry / linearisation (reading A7);
 *   - in Eq. 17 (orc_cfl_terms): the value for a particle without neighbours (reading A22) and
 *     taking mu^max as the largest magnitude (reading A23).
 * Everything else is pinned by tests/test_oracle_pins.py.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (oracle/build.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    float origin[3];
    float cell;
    float inv_cell;
    int32_t dims[3];
} orc_grid;

typedef struct {
    double h, gamma, alpha, beta, eta;
} orc_sph_params;

static const double ORC_PI = 3.14159265358979323846264338327950288;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---------------------------------------------------------------- kernels ---- */

/* Eq. 8 (L79): cubic spline W(xi, h), xi = r/h, support 2h, prefactor 1/(pi h^3). */
double orc_W(double xi, double h) {
    double s = 1.0 / (ORC_PI * h * h * h);
    if (xi < 0.0) xi = -xi;
    if (xi <= 1.0) return s * (1.0 - 1.5 * xi * xi + 0.75 * xi * xi * xi);
    if (xi <= 2.0) {
        double t = 2.0 - xi;
        return s * 0.25 * t * t * t;
    }
    return 0.0;
}

/* Eq. 9 (L86): pressure kernel W_p(xi, h) = 15/(64 pi h^3) (2 - xi)^3 on [0,2]. */
double orc_Wp(double xi, double h) {
    if (xi < 0.0) xi = -xi;
    if (xi >= 2.0) return 0.0;
    double t = 2.0 - xi;
    return 15.0 / (64.0 * ORC_PI * h * h * h) * t * t * t;
}

/* d W_p / d xi from Eq. 9 (reading A3: Eq. 9 is authoritative, not the limit printed at L89):
 *   -45/(64 pi h^3) (2 - xi)^2  on [0,2), 0 beyond.                                   */
double orc_dWp_dxi(double xi, double h) {
    if (xi < 0.0) xi = -xi;
    if (xi >= 2.0) return 0.0;
    double t = 2.0 - xi;
    return -45.0 / (64.0 * ORC_PI * h * h * h) * t * t;
}

/* ---------------------------------------------------------------- gravity ---- */

/* Eq. 4 (L47) under reading A1:
 *   a_i = -G sum_{j=1..N} m_j (r_i - r_j) / (|r_i - r_j|^2 + delta^2)^(3/2)
 * j = i contributes exactly 0 (numerator 0) so it is not excluded; if delta == 0 a
 * zero separation is skipped (0/0).  posm[j] = (x,y,z,m).  targets == NULL
 * means targets 0..nt-1.  acc[t] = (ax, ay, az).                                        */
void orc_gravity(const double* posm, int64_t n, double G, double delta,
                 const int64_t* targets, int64_t nt, double* acc) {
    const double d2s = delta * delta;
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        double xi = posm[4 * i + 0], yi = posm[4 * i + 1], zi = posm[4 * i + 2];
        double ax = 0.0, ay = 0.0, az = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            double dx = xi - posm[4 * j + 0];
            double dy = yi - posm[4 * j + 1];
            double dz = zi - posm[4 * j + 2];
            double r2 = dx * dx + dy * dy + dz * dz + d2s;
            if (r2 == 0.0) continue;
            double w = posm[4 * j + 3] / (r2 * sqrt(r2));
            ax -= w * dx;
            ay -= w * dy;
            az -= w * dz;
        }
        acc[3 * t + 0] = G * ax;
        acc[3 * t + 1] = G * ay;
        acc[3 * t + 2] = G * az;
    }
}

/* Softened potential energy consistent with Eq. 4 / A1 (diagnostic for pin P7):
 *   U = -G/2 sum_i sum_{j != i} m_i m_j / sqrt(|r_ij|^2 + delta^2).                      */
double orc_potential_energy(const double* posm, int64_t n, double G, double delta) {
    const double d2s = delta * delta;
    double u = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : u)
    for (int64_t i = 0; i < n; ++i) {
        double xi = posm[4 * i + 0], yi = posm[4 * i + 1], zi = posm[4 * i + 2], mi = posm[4 * i + 3];
        double s = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double dx = xi - posm[4 * j + 0];
            double dy = yi - posm[4 * j + 1];
            double dz = zi - posm[4 * j + 2];
            s += posm[4 * j + 3] / sqrt(dx * dx + dy * dy + dz * dz + d2s);
        }
        u += mi * s;
    }
    return -0.5 * G * u;
}

/* ------------------------------------------------------------- grid (A7) ---- */

/* Reading A7: cell = fl(fl(2h) * (1 + 2^-9)), inv_cell = fl(1/cell), origin = min over gas,
 * M_x = (int)(fl(fl(max_x - origin_x) * inv_cell)) + 1.  All FP32, one rounding per op.
 * Returns 0, or -1 if a dimension exceeds 4096 or M >= 2^31, or n_gas <= 0.             */
int orc_grid_from_bbox(const double* posm, int64_t n_gas, float h, orc_grid* g) {
    if (n_gas <= 0 || !(h > 0.0f)) return -1;
    volatile float two_h = 2.0f * h;
    volatile float cell = two_h * 1.001953125f; /* 1 + 2^-9, exact in FP32 */
    volatile float inv = 1.0f / cell;
    float lo[3], hi[3];
    for (int a = 0; a < 3; ++a) lo[a] = hi[a] = (float)posm[a];
    for (int64_t i = 1; i < n_gas; ++i)
        for (int a = 0; a < 3; ++a) {
            float v = (float)posm[4 * i + a];
            if (v < lo[a]) lo[a] = v;
            if (v > hi[a]) hi[a] = v;
        }
    double m = 1.0;
    for (int a = 0; a < 3; ++a) {
        volatile float ext = hi[a] - lo[a];
        volatile float c = ext * inv;
        if (!(c < 4096.0f)) return -1;
        g->origin[a] = lo[a];
        g->dims[a] = (int32_t)c + 1;
        if (g->dims[a] > 4096) return -1;
        m *= g->dims[a];
    }
    if (m >= 2147483648.0) return -1;
    g->cell = cell;
    g->inv_cell = inv;
    return 0;
}

static inline int32_t orc_cell_coord(float x, float origin, float inv_cell, int32_t dim) {
    volatile float d = x - origin;       /* RN FP32 subtraction */
    volatile float c = d * inv_cell;     /* RN FP32 multiplication (separate op: no FMA) */
    float f = floorf(c);
    f = fmaxf(f, 0.0f);
    f = fminf(f, (float)(dim - 1));      /* clamp in float before the cast */
    return (int32_t)f;
}

/* (a1) k_i = ix + M_x (iy + M_y iz)  — "cell number k where the i-th particle is located", L161. */
void orc_cell_keys(const double* posm, int64_t n_gas, const orc_grid* g, uint32_t* key) {
    for (int64_t i = 0; i < n_gas; ++i) {
        int32_t ix = orc_cell_coord((float)posm[4 * i + 0], g->origin[0], g->inv_cell, g->dims[0]);
        int32_t iy = orc_cell_coord((float)posm[4 * i + 1], g->origin[1], g->inv_cell, g->dims[1]);
        int32_t iz = orc_cell_coord((float)posm[4 * i + 2], g->origin[2], g->inv_cell, g->dims[2]);
        key[i] = (uint32_t)ix + (uint32_t)g->dims[0] * ((uint32_t)iy + (uint32_t)g->dims[1] * (uint32_t)iz);
    }
}

/* (a2-a5) Sequential counting sort, the paper's arrays written out (L160-173):
 *   count[k]  = CellSPH[k].x ; incl[k] = CellSPH[k].y = incl[k-1] + count[k]  (L171) ;
 *   start[k]  = incl[k-1] (0 for k = 0), start[M] = n_gas   (reading A13) ;
 *   perm[start[k] + (number of i' < i in cell k)] = i         (stable: reading A16).
 * Visiting i in ascending order with a per-cell cursor gives exactly that rank.        */
int orc_counting_sort(const uint32_t* key, int64_t n_gas, int64_t M,
                      uint32_t* count, uint32_t* start, uint32_t* perm) {
    memset(count, 0, (size_t)M * sizeof(uint32_t));
    for (int64_t i = 0; i < n_gas; ++i) {
        if ((int64_t)key[i] >= M) return -1;
        count[key[i]] += 1;
    }
    uint32_t incl_prev = 0;
    for (int64_t k = 0; k < M; ++k) {
        start[k] = incl_prev;
        incl_prev = incl_prev + count[k];
    }
    start[M] = incl_prev;
    uint32_t* cursor = (uint32_t*)calloc((size_t)M, sizeof(uint32_t));
    if (!cursor) return -2;
    for (int64_t i = 0; i < n_gas; ++i) {
        uint32_t k = key[i];
        perm[start[k] + cursor[k]] = (uint32_t)i;
        cursor[k] += 1;
    }
    free(cursor);
    return 0;
}

/* --------------------------------------------------- neighbour predicate ---- */

/* Reading A8 / O2: FP32 separations, d2 = fma(dz,dz, fma(dy,dy, dx*dx)), neighbour iff d2 < rc2,
 * rc2 = fl(fl(2h) * fl(2h)).  Symmetric in (i,j).                                       */
static inline float orc_d2_f32(const double* pi, const double* pj) {
    /* positions rounded to FP32 first (exact when they came from FP32 arrays); the file is
     * built with -ffp-contract=off, so each line below is one RN FP32 operation.          */
    float dx = (float)pi[0] - (float)pj[0];
    float dy = (float)pi[1] - (float)pj[1];
    float dz = (float)pi[2] - (float)pj[2];
    float xx = dx * dx;
    float s = fmaf(dy, dy, xx);
    return fmaf(dz, dz, s);
}

float orc_rc2(float h) {
    volatile float two_h = 2.0f * h;
    volatile float rc2 = two_h * two_h;
    return rc2;
}

/* Per-particle smoothing lengths (L82: h_ij = (h_i + h_j)/2; reading A24): the pair (i,j) is a
 * neighbour pair iff d2 < rc2_ij with rc2_ij = fl(fl(h_i + h_j)^2) in FP32 (2 h_ij = h_i + h_j exactly).
 * hs == NULL: one global h, rc2 = orc_rc2(h).  With h_i = h_j = h both give the same number.        */
static inline float orc_rc2_pair(float rc2_global, const float* hs, int64_t i, int64_t j) {
    if (!hs) return rc2_global;
    volatile float sum = hs[i] + hs[j];
    volatile float rc2 = sum * sum;
    return rc2;
}

static int orc_cmp_u32(const void* a, const void* b) {
    uint32_t x = *(const uint32_t*)a, y = *(const uint32_t*)b;
    return (x > y) - (x < y);
}

/* N(i) = { j < n_gas : j != i, pred(i,j) } by brute force over all j (definition).
 * Two-call protocol: with nbr_index == NULL only nbr_count[t] is written.  Otherwise
 * nbr_offset[nt+1] (exclusive prefix of the counts) must be given and lists are written
 * ascending in j.                                                                        */
void orc_neighbours_brute(const double* posm, int64_t n_gas, float h, const float* hs /*[n_gas] or NULL*/,
                          const int64_t* targets, int64_t nt,
                          uint32_t* nbr_count, const int64_t* nbr_offset, uint32_t* nbr_index) {
    const float rc2 = orc_rc2(h);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        uint32_t c = 0;
        for (int64_t j = 0; j < n_gas; ++j) {
            if (j == i) continue;
            if (orc_d2_f32(posm + 4 * i, posm + 4 * j) < orc_rc2_pair(rc2, hs, i, j)) {
                if (nbr_index) nbr_index[nbr_offset[t] + c] = (uint32_t)j;
                ++c;
            }
        }
        if (!nbr_index) nbr_count[t] = c;
    }
}

/* Same sets through the oracle's own grid (3x3x3 stencil over the counting-sort ranges).
 * Proven equal to the brute-force sets by pin P1.                                       */
void orc_neighbours_grid(const double* posm, int64_t n_gas, float h, const float* hs /*[n_gas] or NULL; all <= h*/,
                         const orc_grid* g,
                         const uint32_t* key, const uint32_t* start, const uint32_t* perm,
                         const int64_t* targets, int64_t nt,
                         uint32_t* nbr_count, const int64_t* nbr_offset, uint32_t* nbr_index) {
    const float rc2 = orc_rc2(h);
    const int32_t Mx = g->dims[0], My = g->dims[1], Mz = g->dims[2];
    (void)n_gas;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        uint32_t k = key[i];
        int32_t ix = (int32_t)(k % (uint32_t)Mx);
        int32_t iy = (int32_t)((k / (uint32_t)Mx) % (uint32_t)My);
        int32_t iz = (int32_t)(k / ((uint32_t)Mx * (uint32_t)My));
        uint32_t c = 0;
        for (int32_t cz = iz - 1; cz <= iz + 1; ++cz) {
            if (cz < 0 || cz >= Mz) continue;
            for (int32_t cy = iy - 1; cy <= iy + 1; ++cy) {
                if (cy < 0 || cy >= My) continue;
                for (int32_t cx = ix - 1; cx <= ix + 1; ++cx) {
                    if (cx < 0 || cx >= Mx) continue;
                    int64_t cc = (int64_t)cx + (int64_t)Mx * ((int64_t)cy + (int64_t)My * cz);
                    for (uint32_t s = start[cc]; s < start[cc + 1]; ++s) {
                        int64_t j = perm[s];
                        if (j == i) continue;
                        if (orc_d2_f32(posm + 4 * i, posm + 4 * j) < orc_rc2_pair(rc2, hs, i, j)) {
                            if (nbr_index) nbr_index[nbr_offset[t] + c] = (uint32_t)j;
                            ++c;
                        }
                    }
                }
            }
        }
        if (nbr_index)
            qsort(nbr_index + nbr_offset[t], c, sizeof(uint32_t), orc_cmp_u32);
        else
            nbr_count[t] = c;
    }
}

/* ------------------------------------------------------------ SPH sums ---- */

/* Eq. 7 (L74) with the self term (reading A5):
 *   rho_i = m_i W(0,h_ii) + sum_{j in N(i)} m_j W(|r_i - r_j|/h_ij, h_ij)   (distances in FP64),
 * h_ij = (h_i + h_j)/2 (L82) when hs is given, else the global h.                                */
void orc_density(const double* posm, double h, const double* hs /*[n_gas] or NULL*/, const int64_t* targets, int64_t nt,
                 const int64_t* nbr_offset, const uint32_t* nbr_index, double* rho) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        double xi = posm[4 * i], yi = posm[4 * i + 1], zi = posm[4 * i + 2];
        double r = posm[4 * i + 3] * orc_W(0.0, hs ? hs[i] : h);
        for (int64_t q = nbr_offset[t]; q < nbr_offset[t + 1]; ++q) {
            int64_t j = nbr_index[q];
            double dx = xi - posm[4 * j], dy = yi - posm[4 * j + 1], dz = zi - posm[4 * j + 2];
            double d = sqrt(dx * dx + dy * dy + dz * dz);
            double hij = hs ? 0.5 * (hs[i] + hs[j]) : h;
            r += posm[4 * j + 3] * orc_W(d / hij, hij);
        }
        rho[t] = r;
    }
}

/* Eqs. 10-11 (L91-93), hydro part, with Pi_ij, nu^a_ij, mu_ij, rho_ij, c_ij of L95-99:
 *   grad W_p = dWp/dxi * dr/|dr| / h                (L95; dWp/dxi from Eq. 9, reading A3)
 *   mu_ij    = h dr.dv / (|dr|^2 + eta h^2) if dr.dv < 0 else 0               (L97)
 *   nu_ij    = mu_ij (beta mu_ij - alpha c_ij) / rho_ij                         (L97)
 *   Pi_ij    = p_i/rho_i^2 + p_j/rho_j^2 + nu_ij                (L95 with reading A2)
 *   a_i      = - sum_j m_j Pi_ij grad W_p                                   (Eq. 10)
 *   de_i/dt  = 1/2 sum_j m_j Pi_ij dv_ij . grad W_p                         (Eq. 11)
 *   p = (gamma-1) rho e (Eq. 5) ; c = sqrt(gamma p / rho) (L99).
 * rho_all[j] must hold the density of every j that appears (index by global gas index).
 * A pair at zero separation contributes nothing (reading A9).  out[t] = (ax, ay, az, de/dt).
 * gross (may be NULL): gross[t] = (sum_j |m_j Pi_ij grad W_p|, sum_j |1/2 m_j Pi_ij dv.grad W_p|), the
 * sums of the magnitudes of the same terms — a conditioning diagnostic for the parity tolerance
 * (reading A17), not part of the method.                                            */
void orc_forces(const double* posm, const double* vele, const double* rho_all, const orc_sph_params* p,
                const double* hs /*[n_gas] or NULL: h_ij = (h_i + h_j)/2 in grad W_p and mu_ij (L82, L95-97)*/,
                const int64_t* targets, int64_t nt,
                const int64_t* nbr_offset, const uint32_t* nbr_index, double* out, double* gross) {
    const double gm1 = p->gamma - 1.0;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        double xi = posm[4 * i], yi = posm[4 * i + 1], zi = posm[4 * i + 2];
        double vxi = vele[4 * i], vyi = vele[4 * i + 1], vzi = vele[4 * i + 2], ei = vele[4 * i + 3];
        double rhoi = rho_all[i];
        double pi_ = gm1 * rhoi * ei;
        double ci = sqrt(p->gamma * pi_ / rhoi);
        double ax = 0.0, ay = 0.0, az = 0.0, de = 0.0, ga = 0.0, ge = 0.0;
        for (int64_t q = nbr_offset[t]; q < nbr_offset[t + 1]; ++q) {
            int64_t j = nbr_index[q];
            double dx = xi - posm[4 * j], dy = yi - posm[4 * j + 1], dz = zi - posm[4 * j + 2];
            double r2 = dx * dx + dy * dy + dz * dz;
            if (r2 == 0.0) continue;
            double r = sqrt(r2);
            double h = hs ? 0.5 * (hs[i] + hs[j]) : p->h;
            double dwp = orc_dWp_dxi(r / h, h);
            double gx = dwp * dx / r / h, gy = dwp * dy / r / h, gz = dwp * dz / r / h;
            double dvx = vxi - vele[4 * j], dvy = vyi - vele[4 * j + 1], dvz = vzi - vele[4 * j + 2];
            double ej = vele[4 * j + 3], rhoj = rho_all[j], mj = posm[4 * j + 3];
            double pj = gm1 * rhoj * ej;
            double cj = sqrt(p->gamma * pj / rhoj);
            double rv = dx * dvx + dy * dvy + dz * dvz;
            double mu = (rv < 0.0) ? h * rv / (r2 + p->eta * h * h) : 0.0;
            double rhoij = 0.5 * (rhoi + rhoj), cij = 0.5 * (ci + cj);
            double nu = mu * (p->beta * mu - p->alpha * cij) / rhoij;
            double Pi = pi_ / (rhoi * rhoi) + pj / (rhoj * rhoj) + nu;
            ax -= mj * Pi * gx;
            ay -= mj * Pi * gy;
            az -= mj * Pi * gz;
            de += 0.5 * mj * Pi * (dvx * gx + dvy * gy + dvz * gz);
            ga += fabs(mj * Pi) * sqrt(gx * gx + gy * gy + gz * gz);
            ge += fabs(0.5 * mj * Pi * (dvx * gx + dvy * gy + dvz * gz));
        }
        if (gross) {
            gross[2 * t + 0] = ga;
            gross[2 * t + 1] = ge;
        }
        out[4 * t + 0] = ax;
        out[4 * t + 1] = ay;
        out[4 * t + 2] = az;
        out[4 * t + 3] = de;
    }
}

/* Modified CFL condition, Eq. 17 (L125-129), per target particle i over its neighbour list:
 *   s_i = min_j |r_i - r_j|,  c_i^max = max_j c_ij,  mu_i^max = max_j |mu_ij|
 * with c_ij = (c_i + c_j)/2, c = sqrt(gamma p / rho) (L99) and mu_ij of L97.  Readings:
 * A23 mu^max is the largest MAGNITUDE (mu_ij <= 0 by its definition, so "max" as printed would always
 * be 0); A9 pairs at zero separation are skipped; A22 a particle with no neighbour gets s = 2h,
 * c^max = c_i, mu^max = 0.  out[t] = (s_i, c_i^max, mu_i^max).                                     */
void orc_cfl_terms(const double* posm, const double* vele, const double* rho_all, const orc_sph_params* p,
                   const double* hs /*[n_gas] or NULL: h_ij = (h_i + h_j)/2 in mu_ij (L82, L97); no neighbour: s = 2 h_i*/,
                   const int64_t* targets, int64_t nt,
                   const int64_t* nbr_offset, const uint32_t* nbr_index, double* out) {
    const double gm1 = p->gamma - 1.0;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        double ci = sqrt(p->gamma * (gm1 * rho_all[i] * vele[4 * i + 3]) / rho_all[i]);
        double smin = -1.0, cmax = ci, mumax = 0.0;
        for (int64_t q = nbr_offset[t]; q < nbr_offset[t + 1]; ++q) {
            int64_t j = nbr_index[q];
            double dx = posm[4 * i] - posm[4 * j], dy = posm[4 * i + 1] - posm[4 * j + 1], dz = posm[4 * i + 2] - posm[4 * j + 2];
            double r2 = dx * dx + dy * dy + dz * dz;
            if (r2 == 0.0) continue;
            double r = sqrt(r2);
            double rv = dx * (vele[4 * i] - vele[4 * j]) + dy * (vele[4 * i + 1] - vele[4 * j + 1]) +
                        dz * (vele[4 * i + 2] - vele[4 * j + 2]);
            double h = hs ? 0.5 * (hs[i] + hs[j]) : p->h;
            double mu = (rv < 0.0) ? h * rv / (r2 + p->eta * h * h) : 0.0;
            double cj = sqrt(p->gamma * (gm1 * rho_all[j] * vele[4 * j + 3]) / rho_all[j]);
            double cij = 0.5 * (ci + cj);
            if (smin < 0.0 || r < smin) smin = r;
            if (cij > cmax) cmax = cij;
            if (fabs(mu) > mumax) mumax = fabs(mu);
        }
        out[3 * t + 0] = smin < 0.0 ? 2.0 * (hs ? hs[i] : p->h) : smin;
        out[3 * t + 1] = cmax;
        out[3 * t + 2] = mumax;
    }
}
