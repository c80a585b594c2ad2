/*
 * tnlmr.h -- C ABI of the TNLM reconstruction path (TNLM-R) in libtnlm.so.
 *
 * TNLM-R (arxiv/paper_1201_2450) alternates, for k = 1, 2, ...:
 *   1. (P1) g^(k) = CGLS on sum_i ||P_i g_i - y_i||^2 started from f^(k-1), phase by phase   (PAPER.md:145 Eq. 5, :147-149, :197)
 *   2. weights from g^(k)                                                                   (PAPER.md:185 Eq. 9, :198)
 *   3. f^(k) = one Gauss-Jacobi sweep of Eq. 8 with g = g^(k)
 *   4. f^(k) = max(f^(k), 0)
 * Steps 2-3 are tnlm_jacobi_step of tnlm.h; this header adds the cone-beam projection operator P_i, its transpose,
 * CGLS and the loop.  Readings of the silent points are DESIGN.md section 12 (R1-R5): P is Siddon's radiological path
 * (one ray per detector pixel, source -> pixel centre; PAPER.md:245 names Siddon's algorithm), the back-projector is its
 * exact transpose, CGLS is Bjorck's recurrence with a fixed iteration count, the single sweep of step 3 starts from g^(k).
 *
 * Geometry (reading R3): circular orbit about z; at gantry angle t the source is at (sid cos t, sid sin t, 0), the flat
 * detector's centre at the source minus sdd (cos t, sin t, 0), its axes u = (-sin t, cos t, 0) and v = (0, 0, 1); pixel
 * (iu, iv) has its centre at u = (iu - (nu-1)/2) du, v = (iv - (nv-1)/2) dv.  The volume [nz][ny][nx] of cubic voxels
 * of edge `voxel` is centred on the isocentre.
 *
 * Layout: volumes are [phase][z][y][x] fp32 stacks (as in tnlm.h), projections [phase][view][v][u] fp32; both DEVICE
 * pointers, 16-byte aligned, owned by the caller.  `angles` is a HOST pointer to n_phase * n_view doubles (radians,
 * [phase][view]); it is read before the call returns.  Every phase has n_view views.  Every call first uploads the
 * (cos, sin) table of the angles and waits for that copy on `cuda_stream` (one stream synchronisation, so work queued
 * earlier on the stream has finished too); the kernels are then enqueued and the call returns.  Argument errors are
 * synchronous negative tnlm_status codes (tnlm.h).
 * The back-projector and the dot products of CGLS accumulate with atomic adds, so results are reproducible to
 * rounding, not bit for bit.
 */
#ifndef TNLMR_H
#define TNLMR_H

#include <stddef.h>
#include <stdint.h>

#include "tnlm.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int32_t n_phase, nz, ny, nx;   /* volume stack */
    int32_t n_view, nv, nu;        /* views per phase, detector rows (v) and columns (u) */
    float voxel;                   /* voxel edge */
    float du, dv;                  /* detector pixel pitch */
    float sid, sdd;                /* source-isocentre and source-detector distance, same unit as voxel */
} tnlmr_geometry;

enum { TNLMR_START_G = 0, TNLMR_START_PREVIOUS = 1 };   /* the sweep of step 3 averages g^(k) (reading R1) or f^(k-1) */

/* Device workspace tnlmr_cgls / tnlmr_reconstruct need (0 if the geometry or the parameters are invalid).  `p` may be
 * NULL for tnlmr_cgls alone. */
size_t tnlmr_workspace_bytes(const tnlmr_geometry *g, const tnlm_params *p);

/* y = P f for every phase: y[phase][view][iv][iu] = sum over voxels of (length of the ray inside the voxel) * f. */
int tnlmr_project(const tnlmr_geometry *g, const double *angles, const float *f, float *y, void *ws, size_t ws_bytes,
                  void *cuda_stream);

/* f = P^T y for every phase (overwrites f). */
int tnlmr_backproject(const tnlmr_geometry *g, const double *angles, const float *y, float *f, void *ws, size_t ws_bytes,
                      void *cuda_stream);

/* n_iter iterations of CGLS on ||P_i x_i - y_i||^2 for every phase independently, x in/out. */
int tnlmr_cgls(const tnlmr_geometry *g, const double *angles, const float *y, float *x, int32_t n_iter, void *ws,
               size_t ws_bytes, void *cuda_stream);

/*
 * TNLM-R: n_outer iterations of steps 1-4 from f_init (a stack; the paper uses FDK, any start works), n_cgls CGLS
 * iterations in step 1, TNLM parameters `p` (its n_phase, nz, ny, nx must equal the geometry's).  f_out receives
 * f^(n_outer); it must not overlap f_init, y or the workspace.  n_outer = 0 copies f_init.
 */
int tnlmr_reconstruct(const tnlmr_geometry *g, const tnlm_params *p, const double *angles, const float *y,
                      const float *f_init, float *f_out, int32_t n_outer, int32_t n_cgls, int32_t inner_start, void *ws,
                      size_t ws_bytes, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
