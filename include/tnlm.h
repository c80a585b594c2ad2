/*
 * tnlm.h -- C ABI of libtnlm.so: the temporal non-local means (TNLM) enhancement hot path of
 * arxiv/paper_1201_2450 (Jia, Tian, Lou, Sonke, Jiang) as hand-written sm_100a CUDA kernels.
 *
 * Citations are lines of the paper text with the equation they fall in.
 *
 * Data model: a 4D image stack {f_i}, i = 1..N_p respiratory phases,
 * cyclic in i (f_{N_p+1} = f_1), stored as ONE contiguous fp32 array [n_phase][nz][ny][nx],
 * x fastest.  All stack pointers below are DEVICE pointers on the current CUDA device unless a
 * function name ends in _host.  They are allocated and freed by the caller, must be 16-byte
 * aligned, and are only read or written by work enqueued on `cuda_stream` (a cudaStream_t passed
 * as void*; NULL = the legacy default stream).  Calls enqueue and return; results are valid
 * once the stream has been synchronised.  The library allocates no device memory and keeps no
 * global state (except the text of the last CUDA error of the calling thread); calls on different
 * streams with distinct workspaces may run concurrently.
 *
 * Boundary handling (the paper is silent; reading P4): every read of a stack at a
 * coordinate outside the volume returns the nearest in-volume voxel (clamp-to-edge), so every
 * voxel has its full (2M+1)^3 search window.  Phases are taken mod n_phase.
 *
 * Errors: every int-returning function returns TNLM_OK (0) or a negative tnlm_status.  Argument
 * errors are detected synchronously, before anything is enqueued; on error no output is written.
 * NaN/Inf in the inputs are not scanned for (they propagate).  No C++ exception crosses the ABI.
 *
 * Input range: the packed sweep kernels accumulate sum_y u(x,y) f(y) with weights u held below 2^107 relative to a
 * per-voxel reference, so intensities must satisfy |f| < 2^20 (about 1e6) for the sums to
 * stay finite; CT numbers in any usual unit are far inside.  Rescale (f, g, h by one factor: Eq. 3 / Eq. 8 are
 * covariant) if a stack exceeds it.
 */
#ifndef TNLM_H_
#define TNLM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int32_t n_phase, nz, ny, nx; /* stack [n_phase][nz][ny][nx], fp32, contiguous; n_phase >= 2   */
    int32_t patch_radius;        /* d >= 0: patch = (2d+1)^3 cube centred at the voxel */
    int32_t search_radius;       /* M >= 0: search window (2M+1)^3 centred at x       */
    float h;                     /* > 0, finite: similarity scale of Eq. 3, PAPER.md:103 (h < 1e-18 is refused:
                                    1/(2h^2) must be representable in fp32)                          */
    float mu;                    /* > 0, finite: fidelity weight of Eq. 4             */
} tnlm_params;

typedef enum {
    TNLM_OK = 0,
    TNLM_ERR_NULL_POINTER = -1, /* a required pointer is NULL                                      */
    TNLM_ERR_BAD_DIMS = -2,     /* an extent < 1, n_phase < 2 (a phase is never compared with
                                   itself), or the stack exceeds 2^31-1 voxels       */
    TNLM_ERR_BAD_PARAM = -3,    /* h or mu not finite or <= 0; h < 1e-18; negative radius; n_iter < 0 */
    TNLM_ERR_UNSUPPORTED = -4,  /* radius outside the compiled set (d <= 3, M <= 6), bad variant   */
    TNLM_ERR_ALIAS = -5,        /* f_out overlaps an input (Jacobi reads only the old iterate,
                                   PAPER.md:176) or the workspace                                  */
    TNLM_ERR_WORKSPACE = -6,    /* workspace NULL, too small or not 16-byte aligned                */
    TNLM_ERR_CUDA = -7,         /* a CUDA call failed; tnlm_strerror(TNLM_ERR_CUDA) has the text   */
    TNLM_ERR_TOO_LARGE = -8     /* larger than the fixed scratch of a *_static entry point         */
} tnlm_status;

/* Kernel variants, for tests and benchmarks.  AUTO picks the fastest one compiled for (d, M):
 *   GENERIC  any d <= 3, M <= 6, any ref: one thread per voxel, loops as the definition
 *   TILED    d = 1, 1 <= M <= 4, ref == f: scalar FP32 tiles (first optimised kernel, kept for cross-checks)
 *   PAIRED   d = 1 or 2, 1 <= M <= 4, any ref: row-pair packed FP32 (FADD2 / FFMA2) -- what AUTO selects there
 *            (with ref != f the kernel keeps a second neighbour tile for the candidate values: smaller tiles, slower)
 *   PAIRED_TMEM  d = 1 or 2, 2 <= M <= 4, ref == f: the PAIRED arithmetic with the thread-private operands (the -ref_i
 *            windows, Z, N and the reference exponents) in Blackwell tensor memory, and (d = 1: M >= 3; d = 2: all) a
 *            rolling window of ref_j planes in shared memory (three / two CTAs per SM instead of one or two) -- what
 *            AUTO selects there
 * A separate ref with TILED or PAIRED_TMEM is refused (TNLM_ERR_UNSUPPORTED). */
enum { TNLM_VARIANT_AUTO = 0, TNLM_VARIANT_GENERIC = 1, TNLM_VARIANT_TILED = 2, TNLM_VARIANT_PAIRED = 3,
       TNLM_VARIANT_PAIRED_TMEM = 4 };

/*
 * Bytes of caller-owned device workspace that tnlm_jacobi_step / tnlm_enhance / tnlm_weights need
 * for these parameters (the second iterate buffer of the Jacobi double buffering plus kernel
 * scratch).  Returns 0 if the parameters are invalid.
 */
size_t tnlm_workspace_bytes(const tnlm_params *p);

/* Bytes of the w_out array of tnlm_weights: n_phase*2*(2M+1)^3*nz*ny*nx*4; 0 if invalid or overflow. */
size_t tnlm_weights_bytes(const tnlm_params *p);

/*
 * Normalised TNLM weights of Eq. 3 estimated from `ref` as in Eq. 9:
 *   w_out[p][s][k][z][y][x] = exp(-D_k(x)/2h^2) / sum_k' exp(-D_k'(x)/2h^2),
 *   D_k(x) = sum_{delta in [-d,d]^3} (ref_p(x+delta) - ref_q(x+t_k+delta))^2   (plain l2),
 *   q = p-1 for s = 0, q = p+1 for s = 1 (cyclic); t_k = (tz,ty,tx) in [-M,M]^3 with
 *   k = ((tz+M)(2M+1) + (ty+M))(2M+1) + (tx+M); the candidate voxel is y = x + t_k.
 * The normaliser runs over the candidates of ONE voxel x and ONE neighbour phase (PAPER.md:105 with
 * the coefficients of Eq. 7), so sum_k w = 1 for every (p, s, x).  The exponentials
 * are evaluated relative to the smallest D of the window (identical to Eq. 3, never 0/0).
 * For inspection and tests: config 3 of BASELINE.json would need 84 GB.  ws may be NULL.
 */
int tnlm_weights(const tnlm_params *p, const float *ref, float *w_out, void *ws, size_t ws_bytes,
                 void *cuda_stream);

/*
 * One Gauss-Jacobi sweep of Eq. 8 for all phases, weights of Eq. 9 computed on the
 * fly from `ref` (never stored):
 *   f_out_i(x) = mu/(2+mu) g_i(x) + 1/(2+mu) [ sum_y f_{i+1}(y) w_{i,i+1}(x,y) + sum_y f_{i-1}(y) w_{i,i-1}(x,y) ].
 * ref == NULL means ref = f (TNLM-E); TNLM-R passes ref = g^(k).
 * All phases read only `f` (pure Jacobi): f_out must not overlap f, g, ref or ws.
 * n_phase == 2 is legal: phases i+1 and i-1 coincide and are counted twice, as Eq. 8 reads.
 */
int tnlm_jacobi_step(const tnlm_params *p, const float *f, const float *g, const float *ref, float *f_out,
                     void *ws, size_t ws_bytes, void *cuda_stream);

/* Same, with an explicit kernel variant (TNLM_VARIANT_*); TNLM_ERR_UNSUPPORTED if that variant is
 * not compiled for (d, M). */
int tnlm_jacobi_step_variant(const tnlm_params *p, const float *f, const float *g, const float *ref,
                             float *f_out, void *ws, size_t ws_bytes, void *cuda_stream, int variant);

/*
 * TNLM enhancement, TNLM-E: f^0 = f_init (NULL => g); n_iter times
 * { weights from f^k (Eq. 9); one sweep of Eq. 8 }.  A fixed iteration count replaces "until
 * convergence" (the paper ran 10).  No positivity clamp (that is TNLM-R step 4 only,
 * PAPER.md:200).  n_iter == 0 copies f^0 to f_out.  f_out must not overlap g, f_init or ws.
 * To resume, pass the earlier result as f_init together with the ORIGINAL g.
 */
int tnlm_enhance(const tnlm_params *p, const float *g, const float *f_init, float *f_out, int32_t n_iter,
                 void *ws, size_t ws_bytes, void *cuda_stream);

int tnlm_enhance_variant(const tnlm_params *p, const float *g, const float *f_init, float *f_out,
                         int32_t n_iter, void *ws, size_t ws_bytes, void *cuda_stream, int variant);

/*
 * End-to-end form of tnlm_enhance for HOST buffers: g_host / f_init_host (may be NULL) / f_out_host
 * are host pointers (pinned memory makes the copies asynchronous).  The call copies the inputs to the
 * device, runs tnlm_enhance and copies the result back, all on `cuda_stream`, then synchronises the
 * stream before returning.  For f_init_host == NULL, n_iter >= 1 and nz >= 32 the copies are pipelined: the
 * stack travels in z-slabs of 8, 16, 32, ... planes on a copy stream that the call creates and destroys, the first
 * sweep starts on the slabs that have arrived (with the M + d planes of halo beyond them) and the last sweep returns
 * its slabs, largest first, as they finish (same bits as the plain path: slab sweeps reproduce the whole-volume
 * sweep exactly).  dev_ws is a caller-owned DEVICE workspace of at least
 * tnlm_host_workspace_bytes(p) bytes (it holds the device stacks as well as the kernel workspace).
 */
size_t tnlm_host_workspace_bytes(const tnlm_params *p);
int tnlm_enhance_host(const tnlm_params *p, const float *g_host, const float *f_init_host, float *f_out_host,
                      int32_t n_iter, void *dev_ws, size_t dev_ws_bytes, void *cuda_stream);

/*
 * tnlm_enhance_host with a caller-owned copy stream for the pipelined copies (a cudaStream_t other than
 * `cuda_stream`, on the same device; NULL = the call creates and destroys one, as tnlm_enhance_host does).  The copy
 * stream is ordered after the work already queued on `cuda_stream`, and both streams are synchronised before the
 * call returns.  A caller that enhances many stacks saves the stream creation per call.
 */
int tnlm_enhance_host_streams(const tnlm_params *p, const float *g_host, const float *f_init_host, float *f_out_host,
                              int32_t n_iter, void *dev_ws, size_t dev_ws_bytes, void *cuda_stream, void *copy_stream);

/*
 * Z-slab form of one sweep for data-parallel sharding: computes only the
 * output planes z in [z_begin, z_end) of every phase.  f, g, ref and f_out are FULL stacks (the rank
 * needs planes within M+d of its slab to be valid in f / ref); planes outside the slab are untouched.
 */
int tnlm_jacobi_step_slab(const tnlm_params *p, const float *f, const float *g, const float *ref, float *f_out,
                          int32_t z_begin, int32_t z_end, void *ws, size_t ws_bytes, void *cuda_stream);

int tnlm_jacobi_step_slab_variant(const tnlm_params *p, const float *f, const float *g, const float *ref,
                                  float *f_out, int32_t z_begin, int32_t z_end, void *ws, size_t ws_bytes,
                                  void *cuda_stream, int variant);

/*
 * Image-quality metrics of the paper (evaluation, not on the TNLM-E hot path).
 *
 * tnlm_tv_diff: tv_out[p] = TV(a_p - b_p) for every phase p, TV(h) = int dx |grad h(x)| (the
 *   seminorm of Eq. 10).  b == NULL means TV(a_p).  Discretisation (the paper gives none; M3): forward
 *   differences at unit voxel spacing, a difference that would reach outside the volume is 0,
 *   |grad h| = sqrt(hx^2 + hy^2 + hz^2) per voxel in fp32, plain sum over the voxels of the phase in fp64.
 * tnlm_srr: srr_out[p] = [TV(f_fdk_p - f_star_p) - TV(f_enh_p - f_star_p)] / TV(f_fdk_p - f_star_p)  (Eq. 10).
 *   ws: device scratch of at least 2 * n_phase * 8 bytes, 8-byte aligned.
 * tnlm_cnr: out5 = { S, sigma, S_b, sigma_b, CNR } with CNR = 2 |S - S_b| / (sigma + sigma_b) for
 *   the voxels of `phase` inside the half-open boxes roi / roi_bg = { z0, z1, y0, y1, x0, x1 } (HOST arrays of
 *   6 int32, read before the call returns); sigma = population standard deviation.
 * tv_out, srr_out (n_phase doubles) and out5 (5 doubles) are DEVICE pointers, 8-byte aligned.  The stack
 * arguments follow the rules at the top of this file; patch_radius, search_radius, h, mu of `p` are ignored
 * but must be valid.  Errors: TNLM_ERR_NULL_POINTER, TNLM_ERR_BAD_DIMS (phase or a box outside the volume,
 * empty box), TNLM_ERR_WORKSPACE (misaligned pointer, ws too small), TNLM_ERR_CUDA.
 */
int tnlm_tv_diff(const tnlm_params *p, const float *a, const float *b, double *tv_out, void *cuda_stream);
int tnlm_srr(const tnlm_params *p, const float *f_fdk, const float *f_enh, const float *f_star, double *srr_out,
             void *ws, size_t ws_bytes, void *cuda_stream);
int tnlm_cnr(const tnlm_params *p, const float *stack, int32_t phase, const int32_t *roi, const int32_t *roi_bg,
             double *out5, void *cuda_stream);

/*
 * tnlm_srr for callers that must not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same result as tnlm_srr (Eq. 10), no `ws` argument.  The two
 * per-phase TV sums live in a static device array inside the library of 2 * TNLM_SRR_STATIC_MAX_PHASES doubles
 * (1 KB, held by every GPU that loads the library until the process exits); the call itself allocates nothing (no
 * cudaMalloc / cudaFree, no allocating library routine; the first call on a device looks the array's address up once).
 * n_phase > TNLM_SRR_STATIC_MAX_PHASES is refused with TNLM_ERR_TOO_LARGE: use tnlm_srr with a caller workspace.
 * Inputs and srr_out (n_phase doubles, DEVICE, 8-byte aligned) are the caller's, as in tnlm_srr.  Every call on a
 * device shares the one array: the call clears the sums it uses on `cuda_stream` before accumulating, so calls
 * queued on ONE stream are safe back to back, but two calls that can overlap on the GPU (different streams, or
 * different host threads on different streams) RACE on it and give wrong ratios -- serialise them, or use tnlm_srr.
 * Other errors as tnlm_srr.
 */
#define TNLM_SRR_STATIC_MAX_PHASES 64
int tnlm_srr_static(const tnlm_params *p, const float *f_fdk, const float *f_enh, const float *f_star,
                    double *srr_out, void *cuda_stream);

/* Message for a status code; for TNLM_ERR_CUDA includes the calling thread's last CUDA error text. */
const char *tnlm_strerror(int code);

/* Name of the kernel that TNLM_VARIANT_AUTO selects for these parameters (static string). */
const char *tnlm_kernel_name(const tnlm_params *p);

/* Number of kernel launches one tnlm_jacobi_step enqueues for these parameters (>= 1), 0 if invalid. */
int32_t tnlm_launches_per_sweep(const tnlm_params *p);

/*
 * z-tile period of the sweep kernels TNLM_VARIANT_AUTO may select for (d, M) (ref == f or not), 1 for the generic
 * kernel, 0 if the parameters are invalid.  The tiled kernels cut z into tiles that start at multiples of their tile
 * depth, and a voxel's result depends (in the last bits) on its position inside the tile.  tnlm_jacobi_step_slab
 * therefore reproduces a whole-volume sweep bit for bit for any [z_begin, z_end).  A rank of the z-slab partition
 * that stores only its slab plus M+d halo planes gets the same guarantee by
 * placing its local plane 0 at a global plane that is a multiple of this period, filling the halo planes beyond the
 * ends of the global volume with copies of the end planes (= the clamp-to-edge reading of the boundary along z), and
 * calling tnlm_jacobi_step_slab on the local arrays (nz = local plane count, [z_begin, z_end) = its slab in local
 * indices): paper_1201_2450_b200/dist.py does exactly that.
 */
int32_t tnlm_z_tile(const tnlm_params *p);

/*
 * Measurement aid for the FP32 roofline: enqueues a register-resident FFMA
 * loop on every SM; it executes exactly tnlm_probe_fp32_ffma_count(n_iter) FFMA lane-operations.
 * sink is a device buffer of at least 4 bytes.  Time it with CUDA events on `cuda_stream`.
 */
int tnlm_probe_fp32(int32_t n_iter, float *sink, void *cuda_stream);
double tnlm_probe_fp32_ffma_count(int32_t n_iter);

#ifdef __cplusplus
}
#endif
#endif /* TNLM_H_ */
