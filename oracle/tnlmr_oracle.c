/*
 * CPU oracle of the TNLM-R data-fidelity step (arxiv/paper_1201_2450): the cone-beam projection operator P_i, its
 * transpose, and CGLS on ||P g - y||^2.  TEST INFRASTRUCTURE ONLY: used by tests/, __graft_entry__.smoke() and
 * bench.py's CPU legs; shares no code with paper_1201_2450_b200/.  Plain C, fp64, written as the definitions.
 *
 * What the paper fixes: P_i "maps the image f_i into a set of projections corresponding to various projection
 * angles"; (P1) = argmin sum_i ||P_i g_i - y_i||^2 (Eq. 5), solved "phase by phase" with
 * the "conjugate gradient least square (CGLS) method" started from f^(k-1);
 * projections of the phantom study are "numerically generated using Siddon's ray-tracing algorithm"
 * in a circular cone-beam geometry (source-to-isocenter and source-to-detector distances, flat detector).
 * Readings where it is silent:
 *   R2  P is Siddon's exact radiological path: entry (ray, voxel) of P = length of the ray's intersection with the
 *       voxel; one ray per detector pixel, from the point source to the pixel centre.
 *   R3  geometry: source at (sid cos t, sid sin t, 0), rotation about z; detector centre at the source minus
 *       sdd (cos t, sin t, 0); detector axes u = (-sin t, cos t, 0), v = (0, 0, 1); pixel (iu, iv) centre at
 *       u = (iu - (nu-1)/2) du, v = (iv - (nv-1)/2) dv.  Volume [nz][ny][nx] of cubic voxels centred on the isocentre.
 *   R4  the back-projector is the exact transpose of P (CGLS needs the adjoint).
 *   R5  CGLS is Bjorck's recurrence with a fixed number of iterations.
 *
 * siddon() follows Siddon (1985) literally: the parametric values alpha at which the ray S + alpha (D - S) crosses
 * the x-, y- and z-planes of the voxel grid are collected, merged and sorted; every pair of consecutive values gives
 * one voxel (found from the segment's midpoint) and one intersection length.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t n_view, nu, nv;      /* views of this phase, detector pixels along u and v */
    int32_t nz, ny, nx;          /* volume */
    double du, dv;               /* detector pixel pitch */
    double sid, sdd;             /* source-isocentre, source-detector distance */
    double voxel;                /* voxel edge */
} tnlmr_ref_geom;

static int cmp_double(const void *a, const void *b)
{
    const double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* reading R3 */
static void ray_endpoints(const tnlmr_ref_geom *g, double theta, int iu, int iv, double S[3], double D[3])
{
    const double c = cos(theta), s = sin(theta);
    const double u = (iu - 0.5 * (g->nu - 1)) * g->du, v = (iv - 0.5 * (g->nv - 1)) * g->dv;
    S[0] = g->sid * c; S[1] = g->sid * s; S[2] = 0.0;
    D[0] = (g->sid - g->sdd) * c - u * s;
    D[1] = (g->sid - g->sdd) * s + u * c;
    D[2] = v;
}

/* Siddon's radiological path (reading R2).  Writes up to nx+ny+nz+3 (voxel index, length) pairs; returns their number. */
static int siddon(const tnlmr_ref_geom *g, const double S[3], const double D[3], int64_t *vox, double *len, double *alpha)
{
    const int n[3] = {g->nx, g->ny, g->nz};
    double lo[3], d[3];
    double amin = 0.0, amax = 1.0;
    for (int k = 0; k < 3; ++k) {
        lo[k] = -0.5 * n[k] * g->voxel;               /* first plane of axis k */
        d[k] = D[k] - S[k];
        if (d[k] != 0.0) {
            const double a0 = (lo[k] - S[k]) / d[k], a1 = (lo[k] + n[k] * g->voxel - S[k]) / d[k];
            amin = fmax(amin, fmin(a0, a1));
            amax = fmin(amax, fmax(a0, a1));
        } else if (S[k] <= lo[k] || S[k] >= lo[k] + n[k] * g->voxel) {
            return 0;                                  /* parallel to the slab and outside it */
        }
    }
    if (!(amax > amin)) return 0;
    int m = 0;
    alpha[m++] = amin;
    alpha[m++] = amax;
    for (int k = 0; k < 3; ++k) {
        if (d[k] == 0.0) continue;
        for (int i = 0; i <= n[k]; ++i) {
            const double a = (lo[k] + i * g->voxel - S[k]) / d[k];
            if (a > amin && a < amax) alpha[m++] = a;
        }
    }
    qsort(alpha, (size_t)m, sizeof(double), cmp_double);
    const double L = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    int cnt = 0;
    for (int j = 0; j + 1 < m; ++j) {
        const double seg = alpha[j + 1] - alpha[j];
        if (!(seg > 0.0)) continue;
        const double mid = 0.5 * (alpha[j] + alpha[j + 1]);
        int idx[3];
        int inside = 1;
        for (int k = 0; k < 3; ++k) {
            idx[k] = (int)floor((S[k] + mid * d[k] - lo[k]) / g->voxel);
            if (idx[k] < 0 || idx[k] >= n[k]) inside = 0;
        }
        if (!inside) continue;
        vox[cnt] = ((int64_t)idx[2] * g->ny + idx[1]) * g->nx + idx[0];
        len[cnt] = seg * L;
        ++cnt;
    }
    return cnt;
}

static int ray_capacity(const tnlmr_ref_geom *g) { return g->nx + g->ny + g->nz + 8; }

/* y[view][iv][iu] = sum over voxels of (intersection length) * f[voxel]        (y = P f) */
int tnlmr_ref_project(const tnlmr_ref_geom *g, const double *angles, const double *f, double *y)
{
    const int64_t nray = (int64_t)g->n_view * g->nv * g->nu;
    const int cap = ray_capacity(g);
    int fail = 0;
#pragma omp parallel
    {
        int64_t *vox = (int64_t *)malloc(sizeof(int64_t) * (size_t)cap);
        double *len = (double *)malloc(sizeof(double) * (size_t)cap);
        double *alpha = (double *)malloc(sizeof(double) * (size_t)cap);
        if (!vox || !len || !alpha) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 256)
            for (int64_t r = 0; r < nray; ++r) {
                const int iu = (int)(r % g->nu), iv = (int)((r / g->nu) % g->nv), view = (int)(r / ((int64_t)g->nu * g->nv));
                double S[3], D[3];
                ray_endpoints(g, angles[view], iu, iv, S, D);
                const int cnt = siddon(g, S, D, vox, len, alpha);
                double acc = 0.0;
                for (int j = 0; j < cnt; ++j) acc += len[j] * f[vox[j]];
                y[r] = acc;
            }
        }
        free(vox); free(len); free(alpha);
    }
    return fail ? -1 : 0;
}

/* f[voxel] = sum over rays of (intersection length) * y[ray]                   (f = P^T y, reading R4) */
int tnlmr_ref_backproject(const tnlmr_ref_geom *g, const double *angles, const double *y, double *f)
{
    const int64_t nray = (int64_t)g->n_view * g->nv * g->nu;
    const int64_t nvox = (int64_t)g->nz * g->ny * g->nx;
    const int cap = ray_capacity(g);
    int fail = 0;
    memset(f, 0, sizeof(double) * (size_t)nvox);
#pragma omp parallel
    {
        int64_t *vox = (int64_t *)malloc(sizeof(int64_t) * (size_t)cap);
        double *len = (double *)malloc(sizeof(double) * (size_t)cap);
        double *alpha = (double *)malloc(sizeof(double) * (size_t)cap);
        if (!vox || !len || !alpha) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 256)
            for (int64_t r = 0; r < nray; ++r) {
                const int iu = (int)(r % g->nu), iv = (int)((r / g->nu) % g->nv), view = (int)(r / ((int64_t)g->nu * g->nv));
                double S[3], D[3];
                ray_endpoints(g, angles[view], iu, iv, S, D);
                const int cnt = siddon(g, S, D, vox, len, alpha);
                for (int j = 0; j < cnt; ++j) {
                    const double add = len[j] * y[r];
#pragma omp atomic
                    f[vox[j]] += add;
                }
            }
        }
        free(vox); free(len); free(alpha);
    }
    return fail ? -1 : 0;
}

static double dot(const double *a, const double *b, int64_t n)
{
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i) s += a[i] * b[i];
    return s;
}

/*
 * CGLS for min ||P x - y||^2 from the start x (in/out), n_iter iterations (reading R5; Bjorck 1996):
 *   r = y - P x;  s = P^T r;  p = s;  gamma = ||s||^2
 *   repeat:  q = P p;  alpha = gamma / ||q||^2;  x += alpha p;  r -= alpha q;  s = P^T r;
 *            gamma' = ||s||^2;  beta = gamma' / gamma;  p = s + beta p;  gamma = gamma'
 * An iteration with gamma = 0 or ||q|| = 0 (already a least-squares solution) leaves x unchanged and stops.
 * res_out (may be NULL): ||P^T (y - P x)|| after every iteration, n_iter + 1 numbers starting with the initial one.
 */
int tnlmr_ref_cgls(const tnlmr_ref_geom *g, const double *angles, const double *y, double *x, int32_t n_iter, double *res_out)
{
    const int64_t nray = (int64_t)g->n_view * g->nv * g->nu, nvox = (int64_t)g->nz * g->ny * g->nx;
    double *r = (double *)malloc(sizeof(double) * (size_t)nray), *q = (double *)malloc(sizeof(double) * (size_t)nray);
    double *s = (double *)malloc(sizeof(double) * (size_t)nvox), *p = (double *)malloc(sizeof(double) * (size_t)nvox);
    int rc = -1;
    if (r && q && s && p) {
        rc = tnlmr_ref_project(g, angles, x, r);
        for (int64_t i = 0; i < nray; ++i) r[i] = y[i] - r[i];
        if (!rc) rc = tnlmr_ref_backproject(g, angles, r, s);
        memcpy(p, s, sizeof(double) * (size_t)nvox);
        double gamma = dot(s, s, nvox);
        if (res_out) res_out[0] = sqrt(gamma);
        for (int it = 0; it < n_iter && !rc; ++it) {
            if (res_out) res_out[it + 1] = sqrt(gamma);      /* stays if the iteration is a no-op */
            if (!(gamma > 0.0)) continue;
            rc = tnlmr_ref_project(g, angles, p, q);
            const double qq = dot(q, q, nray);
            if (!(qq > 0.0)) continue;
            const double alpha = gamma / qq;
            for (int64_t i = 0; i < nvox; ++i) x[i] += alpha * p[i];
            for (int64_t i = 0; i < nray; ++i) r[i] -= alpha * q[i];
            if (!rc) rc = tnlmr_ref_backproject(g, angles, r, s);
            const double gnew = dot(s, s, nvox);
            const double beta = gnew / gamma;
            for (int64_t i = 0; i < nvox; ++i) p[i] = s[i] + beta * p[i];
            gamma = gnew;
            if (res_out) res_out[it + 1] = sqrt(gamma);
        }
    }
    free(r); free(q); free(s); free(p);
    return rc;
}

/* One ray's (voxel, length) list, for the hand-checked pins.  Returns the count (<= cap). */
int tnlmr_ref_ray(const tnlmr_ref_geom *g, const double *S, const double *D, int64_t *vox, double *len, int32_t cap)
{
    const int need = ray_capacity(g);
    int64_t *v = (int64_t *)malloc(sizeof(int64_t) * (size_t)need);
    double *l = (double *)malloc(sizeof(double) * (size_t)need), *a = (double *)malloc(sizeof(double) * (size_t)need);
    int cnt = -1;
    if (v && l && a) {
        cnt = siddon(g, S, D, v, l, a);
        for (int j = 0; j < cnt && j < cap; ++j) { vox[j] = v[j]; len[j] = l[j]; }
    }
    free(v); free(l); free(a);
    return cnt;
}

/* Source and pixel-centre positions of one ray of the geometry (reading R3). */
void tnlmr_ref_ray_endpoints(const tnlmr_ref_geom *g, double theta, int32_t iu, int32_t iv, double *S, double *D)
{
    ray_endpoints(g, theta, iu, iv, S, D);
}
