/*
 * tnlm_oracle.c -- CPU ORACLE for the TNLM enhancement hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code, header, table or helper with the
 * CUDA path under paper_1201_2450_b200/ and must never be reachable from the product path.
 *
 * What it computes (arxiv/paper_1201_2450, Jia et al., "4D-CBCT reconstruction and
 * enhancement using a temporal non-local means method"), written as the plain definition:
 * six nested loops, fp64 arithmetic, no blocking, no separable sums, no reuse tricks.
 *
 *   weights      w(x,y) = (1/Z) exp(-||p_i(x) - p_j(y)||_2^2 / (2 h^2))        PAPER.md:103 Eq. 3,
 *                estimated from the latest images                            PAPER.md:185 Eq. 9,
 *                y restricted to a (2M+1)^3 search window centred at x       PAPER.md:223,
 *                p = (2d+1)^3 cube centred at the voxel, plain l2
 *   sweep        f_i^{l+1}(x) = mu/(2+mu) g_i(x)
 *                   + 1/(2+mu) [ sum_y f_{i+1}^l(y) w_{i,i+1}(x,y)
 *                              + sum_y f_{i-1}^l(y) w_{i,i-1}(x,y) ]          PAPER.md:176 Eq. 8
 *   enhancement  f^0 = g; repeat { weights from f^k ; one sweep }
 *   phases       cyclic, f_{Np+1} = f_1
 *
 * Readings where the paper is silent or ambiguous:
 *   P1  Z normalises over the candidates y of ONE updated voxel x and ONE neighbour phase
 *       (forced by the coefficients mu/(2+mu), 1/(2+mu) of Eq. 7).
 *   P2  plain sum over the cube, exponent exactly -D/(2 h^2).
 *   P3  exp is evaluated as exp(-(D - D_min(x))/(2h^2)); identical to Eq. 3 because Z
 *       cancels any common factor, and the only form that does not underflow to 0/0.
 *   P4  clamp-to-edge on every read: ref~(v) = ref(clamp(v)), f~(v) = f(clamp(v)), every
 *       voxel keeps its full (2M+1)^3 window.
 *   P5  the zero offset y = x is a candidate (it is a different phase).
 *   P6  phase indices mod P in both directions, P >= 2 (no intra-phase term).
 *   P8  pure Jacobi: every phase reads only the old iterate.
 *   P12 fp64 arithmetic on fp32 inputs; the iterate is rounded to fp32 after every sweep
 *       (that is what crosses the C ABI on the GPU side).
 *
 * Parity pins: tests/test_oracle_pins.py (brute force over all voxel pairs, M=0 closed
 * form, h->inf == scipy uniform_filter, constant fixed point, convex bounds, frozen-weight
 * fixed point == dense linear solve, DFT closed form, Eq. 6 per-voxel stationarity,
 * symmetric-weight energy descent, mutual-weight symmetry).  Nothing here is "parity
 * unpinned" except the paper's own images/tables, whose data is not available.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t n_phase, nz, ny, nx;  /* stack [n_phase][nz][ny][nx], x fastest */
    int32_t patch_radius;         /* d */
    int32_t search_radius;        /* M */
    double h;                     /* Eq. 3 */
    double mu;                    /* Eq. 4 */
} tnlm_ref_params;

enum { REF_OK = 0, REF_NULL = -1, REF_BAD_DIMS = -2, REF_BAD_PARAM = -3, REF_NOMEM = -8 };

static int check(const tnlm_ref_params *p)
{
    if (!p) return REF_NULL;
    if (p->n_phase < 2 || p->nz < 1 || p->ny < 1 || p->nx < 1) return REF_BAD_DIMS;
    if (p->patch_radius < 0 || p->search_radius < 0) return REF_BAD_PARAM;
    if (!(p->h > 0.0) || !isfinite(p->h) || !(p->mu > 0.0) || !isfinite(p->mu)) return REF_BAD_PARAM;
    return REF_OK;
}

static inline int clampi(int v, int n) { return v < 0 ? 0 : (v >= n ? n - 1 : v); }

/* value of one phase volume at a (possibly out-of-volume) coordinate: reading P4 */
static inline double at(const double *vol, const tnlm_ref_params *p, int z, int y, int x)
{
    return vol[((size_t)clampi(z, p->nz) * p->ny + clampi(y, p->ny)) * p->nx + clampi(x, p->nx)];
}

/* D_t(x) = sum over the (2d+1)^3 cube of (ref_i(x+delta) - ref_j(x+t+delta))^2   Eq. 3 / Eq. 9 */
static double patch_distance(const double *ri, const double *rj, const tnlm_ref_params *p,
                             int z, int y, int x, int tz, int ty, int tx)
{
    const int d = p->patch_radius;
    double D = 0.0;
    for (int dz = -d; dz <= d; ++dz)
        for (int dy = -d; dy <= d; ++dy)
            for (int dx = -d; dx <= d; ++dx) {
                double a = at(ri, p, z + dz, y + dy, x + dx);
                double b = at(rj, p, z + tz + dz, y + ty + dy, x + tx + dx);
                D += (a - b) * (a - b);
            }
    return D;
}

/*
 * Normalised weights of voxel (z,y,x) of phase i towards phase j, w[k], k over the window in
 * (tz,ty,tx) raster order; returns nothing else.  scratch holds n_t doubles.
 */
static void voxel_weights(const double *ri, const double *rj, const tnlm_ref_params *p,
                          int z, int y, int x, double *w)
{
    const int M = p->search_radius;
    const double inv2h2 = 1.0 / (2.0 * p->h * p->h);
    int k = 0;
    double Dmin = INFINITY;
    for (int tz = -M; tz <= M; ++tz)
        for (int ty = -M; ty <= M; ++ty)
            for (int tx = -M; tx <= M; ++tx) {
                w[k] = patch_distance(ri, rj, p, z, y, x, tz, ty, tx);
                if (w[k] < Dmin) Dmin = w[k];
                ++k;
            }
    double Z = 0.0;
    for (int q = 0; q < k; ++q) {
        w[q] = exp(-(w[q] - Dmin) * inv2h2); /* reading P3 */
        Z += w[q];
    }
    for (int q = 0; q < k; ++q) w[q] /= Z;
}

/* NLM_s(x) = sum_t w_t f_j(x+t): the bracket of Eq. 8 for one neighbour phase */
static double voxel_nlm(const double *fj, const tnlm_ref_params *p, int z, int y, int x, const double *w)
{
    const int M = p->search_radius;
    int k = 0;
    double acc = 0.0;
    for (int tz = -M; tz <= M; ++tz)
        for (int ty = -M; ty <= M; ++ty)
            for (int tx = -M; tx <= M; ++tx)
                acc += w[k++] * at(fj, p, z + tz, y + ty, x + tx);
    return acc;
}

static size_t n_offsets(const tnlm_ref_params *p)
{
    size_t e = (size_t)(2 * p->search_radius + 1);
    return e * e * e;
}

static inline int phase_mod(int i, int P) { return ((i % P) + P) % P; }

/* ------------------------------------------------------------------ fp64 entry points */

/* w_out[p][s][k][z][y][x], s=0 => phase p-1, s=1 => phase p+1 (cyclic) */
int tnlm_ref_weights_f64(const tnlm_ref_params *p, const double *ref, double *w_out)
{
    int rc = check(p);
    if (rc) return rc;
    if (!ref || !w_out) return REF_NULL;
    const size_t V = (size_t)p->nz * p->ny * p->nx, nt = n_offsets(p);
    int fail = 0;
#pragma omp parallel
    {
        double *w = (double *)malloc(nt * sizeof(double));
        if (!w) {
#pragma omp atomic write
            fail = 1;
        }
        {
#pragma omp for collapse(2) schedule(dynamic, 1)
            for (int ph = 0; ph < p->n_phase; ++ph)
                for (int z = 0; z < p->nz; ++z)
                    for (int s = 0; s < 2; ++s) {
                        const int j = phase_mod(ph + (s ? 1 : -1), p->n_phase);
                        for (int y = 0; y < p->ny; ++y)
                            for (int x = 0; x < p->nx && w; ++x) {
                                voxel_weights(ref + ph * V, ref + j * V, p, z, y, x, w);
                                size_t vox = ((size_t)z * p->ny + y) * p->nx + x;
                                for (size_t k = 0; k < nt; ++k)
                                    w_out[(((size_t)ph * 2 + s) * nt + k) * V + vox] = w[k];
                            }
                    }
            free(w);
        }
    }
    return fail ? REF_NOMEM : REF_OK;
}

/* out[p][z][y][x] = NLM_s for direction dir (+1 or -1): the bracket term of Eq. 8 */
int tnlm_ref_nlm_f64(const tnlm_ref_params *p, const double *f, const double *ref, int dir, double *out)
{
    int rc = check(p);
    if (rc) return rc;
    if (!f || !ref || !out) return REF_NULL;
    if (dir != 1 && dir != -1) return REF_BAD_PARAM;
    const size_t V = (size_t)p->nz * p->ny * p->nx, nt = n_offsets(p);
    int fail = 0;
#pragma omp parallel
    {
        double *w = (double *)malloc(nt * sizeof(double));
        if (!w) {
#pragma omp atomic write
            fail = 1;
        }
        {
#pragma omp for collapse(2) schedule(dynamic, 1)
            for (int ph = 0; ph < p->n_phase; ++ph)
                for (int z = 0; z < p->nz; ++z) {
                    const int j = phase_mod(ph + dir, p->n_phase);
                    for (int y = 0; y < p->ny; ++y)
                        for (int x = 0; x < p->nx && w; ++x) {
                            voxel_weights(ref + ph * V, ref + j * V, p, z, y, x, w);
                            out[ph * V + ((size_t)z * p->ny + y) * p->nx + x] =
                                voxel_nlm(f + j * V, p, z, y, x, w);
                        }
                }
            free(w);
        }
    }
    return fail ? REF_NOMEM : REF_OK;
}

/* one voxel of Eq. 8 */
static double voxel_update(const tnlm_ref_params *p, const double *f, const double *g, const double *ref,
                           int ph, int z, int y, int x, double *w)
{
    const size_t V = (size_t)p->nz * p->ny * p->nx;
    const int jm = phase_mod(ph - 1, p->n_phase), jp = phase_mod(ph + 1, p->n_phase);
    voxel_weights(ref + ph * V, ref + jp * V, p, z, y, x, w);
    const double nlm_p = voxel_nlm(f + jp * V, p, z, y, x, w);
    voxel_weights(ref + ph * V, ref + jm * V, p, z, y, x, w);
    const double nlm_m = voxel_nlm(f + jm * V, p, z, y, x, w);
    const double gi = g[ph * V + ((size_t)z * p->ny + y) * p->nx + x];
    return p->mu / (2.0 + p->mu) * gi + 1.0 / (2.0 + p->mu) * (nlm_p + nlm_m);
}

/* one Gauss-Jacobi sweep, everything fp64 (for the pins; no rounding anywhere) */
int tnlm_ref_jacobi_step_f64(const tnlm_ref_params *p, const double *f, const double *g, const double *ref,
                             double *f_out)
{
    int rc = check(p);
    if (rc) return rc;
    if (!f || !g || !f_out) return REF_NULL;
    if (!ref) ref = f;
    const size_t V = (size_t)p->nz * p->ny * p->nx, nt = n_offsets(p);
    int fail = 0;
#pragma omp parallel
    {
        double *w = (double *)malloc(nt * sizeof(double));
        if (!w) {
#pragma omp atomic write
            fail = 1;
        }
        {
#pragma omp for collapse(2) schedule(dynamic, 1)
            for (int ph = 0; ph < p->n_phase; ++ph)
                for (int z = 0; z < p->nz; ++z)
                    for (int y = 0; y < p->ny; ++y)
                        for (int x = 0; x < p->nx && w; ++x)
                            f_out[ph * V + ((size_t)z * p->ny + y) * p->nx + x] =
                                voxel_update(p, f, g, ref, ph, z, y, x, w);
            free(w);
        }
    }
    return fail ? REF_NOMEM : REF_OK;
}

/*
 * Eq. 8 applied with GIVEN weights (layout of tnlm_ref_weights_f64): f_out_i(x) =
 * mu/(2+mu) g_i(x) + 1/(2+mu) sum_s sum_k w[i][s][k](x) f_{i+s}(x + t_k).  PAPER.md:176.
 * Used by the pins that need weights the paper's Eq. 6 is exact for (symmetric, balanced),
 * and to cross-check tnlm_ref_jacobi_step_f64 against weights() followed by this.
 */
int tnlm_ref_sweep_with_weights_f64(const tnlm_ref_params *p, const double *f, const double *g,
                                    const double *w, double *f_out)
{
    int rc = check(p);
    if (rc) return rc;
    if (!f || !g || !w || !f_out) return REF_NULL;
    const size_t V = (size_t)p->nz * p->ny * p->nx, nt = n_offsets(p);
    const int M = p->search_radius;
    for (int ph = 0; ph < p->n_phase; ++ph)
        for (int z = 0; z < p->nz; ++z)
            for (int y = 0; y < p->ny; ++y)
                for (int x = 0; x < p->nx; ++x) {
                    const size_t vox = ((size_t)z * p->ny + y) * p->nx + x;
                    double bracket = 0.0;
                    for (int s = 0; s < 2; ++s) {
                        const double *fj = f + (size_t)phase_mod(ph + (s ? 1 : -1), p->n_phase) * V;
                        size_t k = 0;
                        for (int tz = -M; tz <= M; ++tz)
                            for (int ty = -M; ty <= M; ++ty)
                                for (int tx = -M; tx <= M; ++tx, ++k)
                                    bracket += w[(((size_t)ph * 2 + s) * nt + k) * V + vox] *
                                               at(fj, p, z + tz, y + ty, x + tx);
                    }
                    f_out[ph * V + vox] = p->mu / (2.0 + p->mu) * g[ph * V + vox] + bracket / (2.0 + p->mu);
                }
    return REF_OK;
}

/* ------------------------------------------------------------------ fp32-boundary entry points
 * Same arithmetic; inputs are fp32 (widened exactly), the result is rounded to fp32 once. */

static double *widen(const float *src, size_t n)
{
    double *dst = (double *)malloc(n * sizeof(double));
    if (dst)
        for (size_t i = 0; i < n; ++i) dst[i] = (double)src[i];
    return dst;
}

int tnlm_ref_jacobi_step(const tnlm_ref_params *p, const float *f, const float *g, const float *ref,
                         float *f_out)
{
    int rc = check(p);
    if (rc) return rc;
    if (!f || !g || !f_out) return REF_NULL;
    const size_t n = (size_t)p->n_phase * p->nz * p->ny * p->nx;
    double *fd = widen(f, n), *gd = widen(g, n), *rd = ref ? widen(ref, n) : NULL;
    double *od = (double *)malloc(n * sizeof(double));
    rc = REF_NOMEM;
    if (fd && gd && od && (rd || !ref)) {
        rc = tnlm_ref_jacobi_step_f64(p, fd, gd, rd, od);
        if (rc == REF_OK)
            for (size_t i = 0; i < n; ++i) f_out[i] = (float)od[i];
    }
    free(fd); free(gd); free(rd); free(od);
    return rc;
}

/* Eq. 8 at a list of output voxels (flat indices into [P][Z][Y][X]); for full-size sampled parity */
int tnlm_ref_jacobi_step_at(const tnlm_ref_params *p, const float *f, const float *g, const float *ref,
                            int64_t n_idx, const int64_t *idx, float *out)
{
    int rc = check(p);
    if (rc) return rc;
    if (!f || !g || !idx || !out) return REF_NULL;
    if (!ref) ref = f;
    const size_t V = (size_t)p->nz * p->ny * p->nx, nt = n_offsets(p);
    const int M = p->search_radius, d = p->patch_radius, R = M + d;
    int fail = 0;
#pragma omp parallel
    {
        /* local fp64 copies of the (2R+1)^3 neighbourhoods would be an optimisation; instead
         * widen on the fly through small per-voxel boxes so the arithmetic stays the plain
         * definition: build three widened sub-volumes (clamped reads) and run voxel_update. */
        const int E = 2 * R + 1;
        tnlm_ref_params q = *p;
        q.n_phase = 3; q.nz = E; q.ny = E; q.nx = E;
        const size_t BV = (size_t)E * E * E;
        double *fb = (double *)malloc(3 * BV * sizeof(double));
        double *rb = (double *)malloc(3 * BV * sizeof(double));
        double *gb = (double *)malloc(3 * BV * sizeof(double));
        double *w = (double *)malloc(nt * sizeof(double));
        if (!fb || !rb || !gb || !w) {
#pragma omp atomic write
            fail = 1;
            free(w);
            w = NULL;
        }
        {
#pragma omp for schedule(dynamic, 16)
            for (int64_t n = 0; n < n_idx; ++n) {
                if (!w) continue;
                int64_t id = idx[n];
                const int ph = (int)(id / (int64_t)V);
                int64_t r = id % (int64_t)V;
                const int z = (int)(r / ((int64_t)p->ny * p->nx));
                r %= (int64_t)p->ny * p->nx;
                const int y = (int)(r / p->nx), x = (int)(r % p->nx);
                /* box phase 0 = ph-1, 1 = ph, 2 = ph+1; box voxel (bz,by,bx) = volume voxel
                 * clamp(z-R+bz, ...): every read voxel_update makes (offsets within R of the
                 * centre) lands inside the box, so the box's own clamp never triggers. */
                for (int b = 0; b < 3; ++b) {
                    const int src = phase_mod(ph - 1 + b, p->n_phase);
                    for (int bz = 0; bz < E; ++bz)
                        for (int by = 0; by < E; ++by)
                            for (int bx = 0; bx < E; ++bx) {
                                size_t o = (size_t)src * V +
                                           ((size_t)clampi(z - R + bz, p->nz) * p->ny + clampi(y - R + by, p->ny)) * p->nx +
                                           clampi(x - R + bx, p->nx);
                                size_t bo = (size_t)b * BV + ((size_t)bz * E + by) * E + bx;
                                fb[bo] = (double)f[o];
                                rb[bo] = (double)ref[o];
                                gb[bo] = (double)g[o];
                            }
                }
                out[n] = (float)voxel_update(&q, fb, gb, rb, 1, R, R, R, w);
            }
        }
        free(fb); free(rb); free(gb); free(w);
    }
    return fail ? REF_NOMEM : REF_OK;
}

/* normalised weights as fp32 inputs -> fp64 weights (same layout as tnlm_ref_weights_f64) */
int tnlm_ref_weights(const tnlm_ref_params *p, const float *ref, double *w_out)
{
    int rc = check(p);
    if (rc) return rc;
    if (!ref || !w_out) return REF_NULL;
    const size_t n = (size_t)p->n_phase * p->nz * p->ny * p->nx;
    double *rd = widen(ref, n);
    if (!rd) return REF_NOMEM;
    rc = tnlm_ref_weights_f64(p, rd, w_out);
    free(rd);
    return rc;
}

/* TNLM-E: f^0 = f_init or g; n_iter x { weights from f^k; one sweep };
 * the iterate is rounded to fp32 after every sweep (reading P12). */
int tnlm_ref_enhance(const tnlm_ref_params *p, const float *g, const float *f_init, float *f_out, int32_t n_iter)
{
    int rc = check(p);
    if (rc) return rc;
    if (!g || !f_out) return REF_NULL;
    if (n_iter < 0) return REF_BAD_PARAM;
    const size_t n = (size_t)p->n_phase * p->nz * p->ny * p->nx;
    float *cur = (float *)malloc(n * sizeof(float));
    if (!cur) return REF_NOMEM;
    memcpy(cur, f_init ? f_init : g, n * sizeof(float));
    for (int k = 0; k < n_iter && rc == REF_OK; ++k) {
        rc = tnlm_ref_jacobi_step(p, cur, g, NULL, f_out);
        memcpy(cur, f_out, n * sizeof(float));
    }
    if (rc == REF_OK) memcpy(f_out, cur, n * sizeof(float));
    free(cur);
    return rc;
}

int tnlm_ref_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}
