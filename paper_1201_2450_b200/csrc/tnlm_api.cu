// C-ABI entry points of libtnlm.so (include/tnlm.h): argument validation, workspace carving,
// kernel selection and launch.  Every step of the hot path runs in the kernels of this library.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <vector>

#include "tnlm_common.cuh"
#include "tnlm_generic.cuh"
#include "tnlm_tiled.cuh"
#include "tnlm_pair.cuh"
#include "tnlm_pair5.cuh"
#include "tnlm_pair5_tm.cuh"
#include "tnlm_metrics.cuh"

namespace {

using namespace tnlm;

thread_local char g_cuda_err[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char *where)
{
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", where, cudaGetErrorString(e));
    return TNLM_ERR_CUDA;
}
}  // namespace

// the other translation units of the library (tnlmr_api.cu) record their CUDA errors in the same thread-local text
namespace tnlm {
int record_cuda_error(cudaError_t e, const char *where) { return cuda_fail(e, where); }
}

namespace {

constexpr int kMaxPatchRadius = 3;
constexpr int kMaxSearchRadius = 6;

int check_params(const tnlm_params *p)
{
    if (!p) return TNLM_ERR_NULL_POINTER;
    if (p->n_phase < 2 || p->nz < 1 || p->ny < 1 || p->nx < 1) return TNLM_ERR_BAD_DIMS;
    const double n = (double)p->n_phase * p->nz * p->ny * p->nx;
    if (n > 2147483647.0) return TNLM_ERR_BAD_DIMS;
    if (p->patch_radius < 0 || p->search_radius < 0) return TNLM_ERR_BAD_PARAM;
    if (!(p->h > 0.f) || !std::isfinite(p->h) || !(p->mu > 0.f) || !std::isfinite(p->mu)) return TNLM_ERR_BAD_PARAM;
    // the kernels scale distances by c2 = log2(e)/(2h^2) in fp32 (flush-to-zero): an h so small that c2 overflows
    // would turn every exponent into 0*inf; h -> infinity is fine (c2 -> 0: uniform weights)
    const double c2 = 1.4426950408889634 / (2.0 * (double)p->h * (double)p->h);
    if (!(c2 < 1.0e37)) return TNLM_ERR_BAD_PARAM;
    if (p->patch_radius > kMaxPatchRadius || p->search_radius > kMaxSearchRadius) return TNLM_ERR_UNSUPPORTED;
    return TNLM_OK;
}

size_t stack_bytes(const tnlm_params *p) { return (size_t)p->n_phase * p->nz * p->ny * p->nx * sizeof(float); }

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    if (!a || !b || na == 0 || nb == 0) return false;
    const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    return x < y + nb && y < x + na;
}

bool misaligned(const void *p) { return ((uintptr_t)p & 15u) != 0; }

int sm_count()
{
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 148;
    return n;
}

// ref_is_f: the sweep takes its weights from the stack it averages (TNLM-E); the TMEM kernel covers only that
int pick_variant(const tnlm_params *p, int variant, bool ref_is_f = true)
{
    if (variant == TNLM_VARIANT_GENERIC) return TNLM_VARIANT_GENERIC;
    if (variant == TNLM_VARIANT_PAIRED_TMEM) return (pair_tm_supported(*p) && ref_is_f) ? TNLM_VARIANT_PAIRED_TMEM : -1;
    if (variant == TNLM_VARIANT_AUTO && pair_tm_supported(*p) && ref_is_f) return TNLM_VARIANT_PAIRED_TMEM;
    if (variant == TNLM_VARIANT_TILED) return tiled_supported(*p) ? TNLM_VARIANT_TILED : -1;
    if (variant == TNLM_VARIANT_PAIRED) return (pair_supported(*p) || pair5_supported(*p)) ? TNLM_VARIANT_PAIRED : -1;
    if (variant == TNLM_VARIANT_AUTO) return (pair_supported(*p) || pair5_supported(*p)) ? TNLM_VARIANT_PAIRED : TNLM_VARIANT_GENERIC;
    return -1;
}

// One sweep over the slab [z0, z1); all pointers already validated.
int launch_sweep(const tnlm_params *p, const float *f, const float *g, const float *ref, float *f_out, int z0, int z1,
                 void *kernel_ws, size_t kernel_ws_bytes, cudaStream_t st, int variant)
{
    if (z1 <= z0) return TNLM_OK;
    const Dims dm = make_dims(*p, z0, z1);
    if (variant == TNLM_VARIANT_PAIRED_TMEM) {
        if (ref != f) return TNLM_ERR_UNSUPPORTED;
        cudaError_t e = launch_pair_tm(*p, dm, f, g, f_out, st);
        return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "paired (TMEM) sweep launch");
    }
    if (variant == TNLM_VARIANT_PAIRED) {
        cudaError_t e = p->patch_radius == 2 ? launch_pair5(*p, dm, f, g, ref, f_out, st) : launch_pair(*p, dm, f, g, ref, f_out, st);
        return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "paired sweep launch");
    }
    if (variant == TNLM_VARIANT_TILED) {
        cudaError_t e = launch_tiled(*p, dm, f, g, ref, f_out, kernel_ws, kernel_ws_bytes, st);
        return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "tiled sweep launch");
    }
    const size_t total = (size_t)p->n_phase * (z1 - z0) * p->ny * p->nx;
    size_t blocks = (total + 255) / 256;
    const size_t cap = (size_t)sm_count() * 64;
    if (blocks > cap) blocks = cap;
    jacobi_generic_kernel<<<(unsigned)blocks, 256, 0, st>>>(f, g, ref, f_out, dm);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "generic sweep launch");
}

int check_ws(const tnlm_params *p, const void *ws, size_t ws_bytes)
{
    if (!ws) return TNLM_ERR_WORKSPACE;
    if (misaligned(ws) || ws_bytes < tnlm_workspace_bytes(p)) return TNLM_ERR_WORKSPACE;
    return TNLM_OK;
}

}  // namespace

extern "C" {

size_t tnlm_workspace_bytes(const tnlm_params *p)
{
    if (check_params(p) != TNLM_OK) return 0;
    // [second iterate buffer][kernel scratch]
    return align_up(stack_bytes(p), 256) + align_up(tiled_scratch_bytes(*p), 256);
}

size_t tnlm_weights_bytes(const tnlm_params *p)
{
    if (check_params(p) != TNLM_OK) return 0;
    const double e = 2.0 * p->search_radius + 1.0;
    const double n = (double)p->n_phase * 2.0 * e * e * e * p->nz * p->ny * p->nx * 4.0;
    if (n > 1.8e19) return 0;
    return (size_t)n;
}

size_t tnlm_host_workspace_bytes(const tnlm_params *p)
{
    if (check_params(p) != TNLM_OK) return 0;
    // [g][f_init][f_out][tnlm_enhance workspace]
    return 3 * align_up(stack_bytes(p), 256) + tnlm_workspace_bytes(p);
}

int tnlm_weights(const tnlm_params *p, const float *ref, float *w_out, void *ws, size_t ws_bytes, void *cuda_stream)
{
    (void)ws; (void)ws_bytes;
    int rc = check_params(p);
    if (rc) return rc;
    if (!ref || !w_out) return TNLM_ERR_NULL_POINTER;
    const size_t wb = tnlm_weights_bytes(p);
    if (wb == 0) return TNLM_ERR_BAD_DIMS;
    if (misaligned(ref) || misaligned(w_out)) return TNLM_ERR_WORKSPACE;
    if (overlaps(w_out, wb, ref, stack_bytes(p))) return TNLM_ERR_ALIAS;
    const Dims dm = make_dims(*p, 0, p->nz);
    const size_t total = (size_t)p->n_phase * 2 * p->nz * p->ny * p->nx;
    size_t blocks = (total + 255) / 256;
    const size_t cap = (size_t)sm_count() * 64;
    if (blocks > cap) blocks = cap;
    weights_generic_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(ref, w_out, dm);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "weights launch");
}

int tnlm_jacobi_step_slab_variant(const tnlm_params *p, const float *f, const float *g, const float *ref, float *f_out,
                                  int32_t z_begin, int32_t z_end, void *ws, size_t ws_bytes, void *cuda_stream,
                                  int variant)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!f || !g || !f_out) return TNLM_ERR_NULL_POINTER;
    if (z_begin < 0 || z_end > p->nz || z_begin > z_end) return TNLM_ERR_BAD_DIMS;
    if (!ref) ref = f;
    int v = pick_variant(p, variant, ref == f);
    if (v < 0) return TNLM_ERR_UNSUPPORTED;
    if (v == TNLM_VARIANT_TILED && ref != f) {   // the scalar tiled kernel covers TNLM-E (ref = f) only
        if (variant != TNLM_VARIANT_AUTO) return TNLM_ERR_UNSUPPORTED;
        v = TNLM_VARIANT_GENERIC;
    }
    const size_t sb = stack_bytes(p);
    if (misaligned(f) || misaligned(g) || misaligned(ref) || misaligned(f_out)) return TNLM_ERR_WORKSPACE;
    if (overlaps(f_out, sb, f, sb) || overlaps(f_out, sb, g, sb) || overlaps(f_out, sb, ref, sb)) return TNLM_ERR_ALIAS;
    rc = check_ws(p, ws, ws_bytes);
    if (rc) return rc;
    if (overlaps(ws, ws_bytes, f_out, sb) || overlaps(ws, ws_bytes, f, sb) || overlaps(ws, ws_bytes, g, sb) ||
        overlaps(ws, ws_bytes, ref, sb))
        return TNLM_ERR_ALIAS;
    char *kws = (char *)ws + align_up(sb, 256);
    return launch_sweep(p, f, g, ref, f_out, z_begin, z_end, kws, ws_bytes - align_up(sb, 256),
                        (cudaStream_t)cuda_stream, v);
}

int tnlm_jacobi_step_slab(const tnlm_params *p, const float *f, const float *g, const float *ref, float *f_out,
                          int32_t z_begin, int32_t z_end, void *ws, size_t ws_bytes, void *cuda_stream)
{
    return tnlm_jacobi_step_slab_variant(p, f, g, ref, f_out, z_begin, z_end, ws, ws_bytes, cuda_stream,
                                         TNLM_VARIANT_AUTO);
}

int tnlm_jacobi_step_variant(const tnlm_params *p, const float *f, const float *g, const float *ref, float *f_out,
                             void *ws, size_t ws_bytes, void *cuda_stream, int variant)
{
    if (!p) return TNLM_ERR_NULL_POINTER;
    return tnlm_jacobi_step_slab_variant(p, f, g, ref, f_out, 0, p->nz, ws, ws_bytes, cuda_stream, variant);
}

int tnlm_jacobi_step(const tnlm_params *p, const float *f, const float *g, const float *ref, float *f_out, void *ws,
                     size_t ws_bytes, void *cuda_stream)
{
    return tnlm_jacobi_step_variant(p, f, g, ref, f_out, ws, ws_bytes, cuda_stream, TNLM_VARIANT_AUTO);
}

int tnlm_enhance_variant(const tnlm_params *p, const float *g, const float *f_init, float *f_out, int32_t n_iter,
                         void *ws, size_t ws_bytes, void *cuda_stream, int variant)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!g || !f_out) return TNLM_ERR_NULL_POINTER;
    if (n_iter < 0) return TNLM_ERR_BAD_PARAM;
    const int v = pick_variant(p, variant);
    if (v < 0) return TNLM_ERR_UNSUPPORTED;
    const size_t sb = stack_bytes(p);
    if (misaligned(g) || misaligned(f_init) || misaligned(f_out)) return TNLM_ERR_WORKSPACE;
    if (overlaps(f_out, sb, g, sb) || overlaps(f_out, sb, f_init, sb)) return TNLM_ERR_ALIAS;
    rc = check_ws(p, ws, ws_bytes);
    if (rc) return rc;
    if (overlaps(ws, ws_bytes, f_out, sb) || overlaps(ws, ws_bytes, g, sb) || overlaps(ws, ws_bytes, f_init, sb))
        return TNLM_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const float *cur = f_init ? f_init : g;   // f^0
    if (n_iter == 0) {
        cudaError_t e = cudaMemcpyAsync(f_out, cur, sb, cudaMemcpyDeviceToDevice, st);
        return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "enhance copy");
    }
    float *buf_ws = (float *)ws;
    char *kws = (char *)ws + align_up(sb, 256);
    const size_t kws_bytes = ws_bytes - align_up(sb, 256);
    // ping-pong between f_out and the workspace buffer so that the last sweep lands in f_out
    float *dst = (n_iter % 2 == 1) ? f_out : buf_ws;
    for (int k = 0; k < n_iter; ++k) {
        // weights from the latest iterate f^k (ref = f^k), one sweep of Eq. 8
        rc = launch_sweep(p, cur, g, cur, dst, 0, p->nz, kws, kws_bytes, st, v);
        if (rc) return rc;
        cur = dst;
        dst = (dst == f_out) ? buf_ws : f_out;
    }
    return TNLM_OK;
}

int tnlm_enhance(const tnlm_params *p, const float *g, const float *f_init, float *f_out, int32_t n_iter, void *ws,
                 size_t ws_bytes, void *cuda_stream)
{
    return tnlm_enhance_variant(p, g, f_init, f_out, n_iter, ws, ws_bytes, cuda_stream, TNLM_VARIANT_AUTO);
}

// Slab bounds of the pipelined host path.  A slab of the first sweep can start once its planes and `look` planes
// beyond them are on the device, and the copy runs about twice as fast as the 5^3-window sweep, so the slabs double:
// [0, 8) [8, 24) [24, 56) [56, 120) ... keep the kernel one slab behind the copy after a start-up of 8 + look planes.
// The last sweep mirrors the bounds (... 32, 16, 8 planes): each slab's way back overlaps the sweeps of the smaller
// slabs after it and only the last 8 planes are exposed.  A single sweep (first and last at once) takes 16-plane slabs.
static std::vector<int> slab_bounds(const int nz, const bool grow, const bool shrink)
{
    std::vector<int> zb{0};
    if (grow && shrink) {
        const int step = std::max(16, (nz + 11) / 12 / 8 * 8);
        for (int z = step; z < nz; z += step) zb.push_back(z);
    } else {
        std::vector<int> cut;
        for (int z = 8; z < nz; z = 2 * z + 8) cut.push_back(z);
        if (grow) {
            zb.insert(zb.end(), cut.begin(), cut.end());
        } else {
            for (auto it = cut.rbegin(); it != cut.rend(); ++it) {
                const int z = (nz - *it) / 8 * 8;
                if (z > zb.back()) zb.push_back(z);
            }
        }
    }
    zb.push_back(nz);
    return zb;
}

// Pipelined form of tnlm_enhance_host (f_init == g, n_iter >= 1, nz >= 32): the stack goes to the device in z-chunks
// on an internal copy stream while the first sweep already runs on the slabs whose planes (and the planes their last
// z-tile and the M+d halo reach into) have arrived, and the last sweep hands its slabs back the same way.  Slab sweeps
// are bit-identical to whole-volume sweeps (z-tiles are aligned to absolute plane indices), so the result equals
// tnlm_enhance's bit for bit.
static int enhance_host_pipelined(const tnlm_params *p, const float *g_host, float *f_out_host, int32_t n_iter,
                                  float *g_dev, float *fo_dev, void *ws, size_t ws_bytes, cudaStream_t st, int variant,
                                  cudaStream_t caller_cs)
{
    // planes past its end that a slab's sweep reads: the halo, and the rest of a z-tile that straddles the bound
    // (bounds are multiples of 8; the deepest tile of any sweep kernel is 8 planes)
    const int zt = tnlm_z_tile(p);
    const int look = p->search_radius + p->patch_radius + ((zt > 0 && 8 % zt == 0) ? 0 : 7);
    const size_t plane = (size_t)p->ny * p->nx, pitch = plane * p->nz * sizeof(float), sb = stack_bytes(p);
    const std::vector<int> zin = slab_bounds(p->nz, true, n_iter == 1);
    const std::vector<int> zout = n_iter == 1 ? zin : slab_bounds(p->nz, false, true);
    const int n_in = (int)zin.size() - 1, n_out = (int)zout.size() - 1;
    cudaStream_t cs = caller_cs;
    std::vector<cudaEvent_t> ev_in(n_in, nullptr), ev_out(n_out, nullptr);
    cudaEvent_t ev_start = nullptr;
    if (!caller_cs) {
        cudaError_t e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
        if (e != cudaSuccess) return cuda_fail(e, "copy stream");
    }
    int rc = TNLM_OK;
    auto fail = [&](cudaError_t err, const char *what) { rc = cuda_fail(err, what); };
    auto ck = [&](cudaError_t err, const char *what) { if (err != cudaSuccess && rc == TNLM_OK) fail(err, what); return err == cudaSuccess; };
    ck(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming), "event");
    for (int s = 0; s < n_in && rc == TNLM_OK; ++s) ck(cudaEventCreateWithFlags(&ev_in[s], cudaEventDisableTiming), "event");
    for (int s = 0; s < n_out && rc == TNLM_OK; ++s) ck(cudaEventCreateWithFlags(&ev_out[s], cudaEventDisableTiming), "event");
    if (rc == TNLM_OK) {
        // the copy stream starts after whatever the caller queued on its stream before this call; chunk s ends where
        // slab s of the first sweep stops reading, so ev_in[s] is all that slab waits for
        ck(cudaEventRecord(ev_start, st), "event record");
        ck(cudaStreamWaitEvent(cs, ev_start, 0), "stream wait");
        int z0 = 0;
        for (int s = 0; s < n_in && rc == TNLM_OK; ++s) {
            const int z1 = s == n_in - 1 ? p->nz : std::min(p->nz, zin[s + 1] + look);
            if (z1 > z0) {
                const size_t off = (size_t)z0 * plane;
                ck(cudaMemcpy2DAsync(g_dev + off, pitch, g_host + off, pitch, (size_t)(z1 - z0) * plane * sizeof(float),
                                     (size_t)p->n_phase, cudaMemcpyHostToDevice, cs), "H2D chunk");
                z0 = z1;
            }
            ck(cudaEventRecord(ev_in[s], cs), "event record");
        }
    }
    float *buf_ws = (float *)ws;
    char *kws = (char *)ws + align_up(sb, 256);
    const size_t kws_bytes = ws_bytes - align_up(sb, 256);
    const float *cur = g_dev;
    float *dst = (n_iter % 2 == 1) ? fo_dev : buf_ws;
    for (int k = 0; k < n_iter && rc == TNLM_OK; ++k) {
        const bool first = k == 0, last = k == n_iter - 1;
        if (!first && !last) {
            rc = launch_sweep(p, cur, g_dev, cur, dst, 0, p->nz, kws, kws_bytes, st, variant);
        } else {
            const std::vector<int> &zb = first ? zin : zout;
            const int ns = (int)zb.size() - 1;
            for (int s = 0; s < ns && rc == TNLM_OK; ++s) {
                if (first) ck(cudaStreamWaitEvent(st, ev_in[s], 0), "stream wait");
                if (rc == TNLM_OK) rc = launch_sweep(p, cur, g_dev, cur, dst, zb[s], zb[s + 1], kws, kws_bytes, st, variant);
                if (last && rc == TNLM_OK) {
                    const size_t off = (size_t)zb[s] * plane;
                    ck(cudaEventRecord(ev_out[s], st), "event record");
                    ck(cudaStreamWaitEvent(cs, ev_out[s], 0), "stream wait");
                    ck(cudaMemcpy2DAsync(f_out_host + off, pitch, dst + off, pitch,
                                         (size_t)(zb[s + 1] - zb[s]) * plane * sizeof(float), (size_t)p->n_phase,
                                         cudaMemcpyDeviceToHost, cs), "D2H slab");
                }
            }
        }
        cur = dst;
        dst = (dst == fo_dev) ? buf_ws : fo_dev;
    }
    // drain both streams whatever happened, then release the internal objects
    cudaError_t e1 = cudaStreamSynchronize(st), e2 = cudaStreamSynchronize(cs);
    if (rc == TNLM_OK) { ck(e1, "enhance_host sync"); ck(e2, "enhance_host copy sync"); }
    for (cudaEvent_t ev : ev_in) if (ev) cudaEventDestroy(ev);
    for (cudaEvent_t ev : ev_out) if (ev) cudaEventDestroy(ev);
    if (ev_start) cudaEventDestroy(ev_start);
    if (!caller_cs) cudaStreamDestroy(cs);
    return rc;
}

int tnlm_enhance_host(const tnlm_params *p, const float *g_host, const float *f_init_host, float *f_out_host,
                      int32_t n_iter, void *dev_ws, size_t dev_ws_bytes, void *cuda_stream)
{
    return tnlm_enhance_host_streams(p, g_host, f_init_host, f_out_host, n_iter, dev_ws, dev_ws_bytes, cuda_stream, nullptr);
}

int tnlm_enhance_host_streams(const tnlm_params *p, const float *g_host, const float *f_init_host, float *f_out_host,
                              int32_t n_iter, void *dev_ws, size_t dev_ws_bytes, void *cuda_stream, void *copy_stream)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!g_host || !f_out_host) return TNLM_ERR_NULL_POINTER;
    if (n_iter < 0) return TNLM_ERR_BAD_PARAM;
    if (!dev_ws || misaligned(dev_ws) || dev_ws_bytes < tnlm_host_workspace_bytes(p)) return TNLM_ERR_WORKSPACE;
    const size_t sb = stack_bytes(p), sba = align_up(sb, 256);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    float *g_dev = (float *)dev_ws;
    float *fi_dev = (float *)((char *)dev_ws + sba);
    float *fo_dev = (float *)((char *)dev_ws + 2 * sba);
    void *ws = (char *)dev_ws + 3 * sba;
    if (!f_init_host && n_iter >= 1 && p->nz >= 32)
        return enhance_host_pipelined(p, g_host, f_out_host, n_iter, g_dev, fo_dev, ws, dev_ws_bytes - 3 * sba, st,
                                      pick_variant(p, TNLM_VARIANT_AUTO), (cudaStream_t)copy_stream);
    cudaError_t e = cudaMemcpyAsync(g_dev, g_host, sb, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e, "H2D g");
    if (f_init_host) {
        e = cudaMemcpyAsync(fi_dev, f_init_host, sb, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return cuda_fail(e, "H2D f_init");
    }
    rc = tnlm_enhance(p, g_dev, f_init_host ? fi_dev : nullptr, fo_dev, n_iter, ws, dev_ws_bytes - 3 * sba, st);
    if (rc) return rc;
    e = cudaMemcpyAsync(f_out_host, fo_dev, sb, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return cuda_fail(e, "D2H f_out");
    e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "enhance_host sync");
}

int tnlm_tv_diff(const tnlm_params *p, const float *a, const float *b, double *tv_out, void *cuda_stream)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!a || !tv_out) return TNLM_ERR_NULL_POINTER;
    if (misaligned(a) || misaligned(b) || ((uintptr_t)tv_out & 7u)) return TNLM_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMemsetAsync(tv_out, 0, sizeof(double) * p->n_phase, st);
    if (e != cudaSuccess) return cuda_fail(e, "tv memset");
    const int xq = (p->nx + 3) / 4;
    const int XQ = xq > 32 ? 64 : xq > 16 ? 32 : 16;                 // x-quads per CTA row
    const int tiles_xq = (xq + XQ - 1) / XQ, tiles_y = (p->ny + kMetricThreads / XQ - 1) / (kMetricThreads / XQ);
    const long long blocks = (long long)tiles_xq * tiles_y * ((p->nz + kTvZChunk - 1) / kTvZChunk);
    if (blocks > 2147483647LL) return TNLM_ERR_BAD_DIMS;
    const dim3 grid((unsigned)blocks, (unsigned)p->n_phase);
    if (XQ == 64) tv_diff_kernel<64><<<grid, kMetricThreads, 0, st>>>(a, b, tv_out, p->nz, p->ny, p->nx, tiles_xq, tiles_y);
    else if (XQ == 32) tv_diff_kernel<32><<<grid, kMetricThreads, 0, st>>>(a, b, tv_out, p->nz, p->ny, p->nx, tiles_xq, tiles_y);
    else tv_diff_kernel<16><<<grid, kMetricThreads, 0, st>>>(a, b, tv_out, p->nz, p->ny, p->nx, tiles_xq, tiles_y);
    e = cudaGetLastError();
    return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "tv launch");
}

int tnlm_srr(const tnlm_params *p, const float *f_fdk, const float *f_enh, const float *f_star, double *srr_out,
             void *ws, size_t ws_bytes, void *cuda_stream)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!f_fdk || !f_enh || !f_star || !srr_out) return TNLM_ERR_NULL_POINTER;
    if (!ws || ((uintptr_t)ws & 7u) || ((uintptr_t)srr_out & 7u) || ws_bytes < 2 * sizeof(double) * (size_t)p->n_phase)
        return TNLM_ERR_WORKSPACE;
    double *t = (double *)ws;
    rc = tnlm_tv_diff(p, f_fdk, f_star, t, cuda_stream);
    if (rc) return rc;
    rc = tnlm_tv_diff(p, f_enh, f_star, t + p->n_phase, cuda_stream);
    if (rc) return rc;
    srr_finish_kernel<<<(p->n_phase + 63) / 64, 64, 0, (cudaStream_t)cuda_stream>>>(t, srr_out, p->n_phase);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "srr launch");
}

// ---- tnlm_srr for callers that cannot allocate (tnlm.h: tnlm_srr_static) -----------------------------------------
// The two per-phase TV sums that tnlm_srr keeps in the caller's `ws` live in a file-scope device array: 2 x
// TNLM_SRR_STATIC_MAX_PHASES doubles (1 KB) that every GPU which loads the library holds until the process exits.
// In host code `g_srr_scratch` is only a stand-in for the symbol, not a device address; the address of the current
// device's copy comes from cudaGetSymbolAddress, looked up once per device and cached.
}  // extern "C"

namespace {

static __device__ __align__(256) double g_srr_scratch[2 * TNLM_SRR_STATIC_MAX_PHASES];

constexpr int kSrrMaxDevices = 64;
std::atomic<double *> g_srr_scratch_addr[kSrrMaxDevices];   // per device ordinal, nullptr until looked up

// Device address of the current device's g_srr_scratch.  Two threads that race on the first call of a device both
// look the address up and store the same value.
int srr_scratch_ptr(double **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "srr_static: cudaGetDevice");
    if (dev < 0 || dev >= kSrrMaxDevices) return cuda_fail(cudaErrorInvalidDevice, "srr_static: device ordinal beyond the address table");
    double *ptr = g_srr_scratch_addr[dev].load(std::memory_order_acquire);
    if (!ptr) {
        e = cudaGetSymbolAddress((void **)&ptr, g_srr_scratch);
        if (e != cudaSuccess) return cuda_fail(e, "srr_static: cudaGetSymbolAddress");
        if (!ptr) return cuda_fail(cudaErrorInvalidSymbol, "srr_static: cudaGetSymbolAddress returned NULL");
        g_srr_scratch_addr[dev].store(ptr, std::memory_order_release);
    }
    *out = ptr;
    return TNLM_OK;
}

}  // namespace

extern "C" {

int tnlm_srr_static(const tnlm_params *p, const float *f_fdk, const float *f_enh, const float *f_star, double *srr_out,
                    void *cuda_stream)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!f_fdk || !f_enh || !f_star || !srr_out) return TNLM_ERR_NULL_POINTER;
    if (p->n_phase > TNLM_SRR_STATIC_MAX_PHASES) return TNLM_ERR_TOO_LARGE;
    if ((uintptr_t)srr_out & 7u) return TNLM_ERR_WORKSPACE;
    double *t = nullptr;
    rc = srr_scratch_ptr(&t);
    if (rc) return rc;
    // the array keeps the previous call's sums: tnlm_tv_diff clears its n_phase outputs on the stream before it
    // accumulates into them, so each half starts at zero
    rc = tnlm_tv_diff(p, f_fdk, f_star, t, cuda_stream);
    if (rc) return rc;
    rc = tnlm_tv_diff(p, f_enh, f_star, t + p->n_phase, cuda_stream);
    if (rc) return rc;
    srr_finish_kernel<<<(p->n_phase + 63) / 64, 64, 0, (cudaStream_t)cuda_stream>>>(t, srr_out, p->n_phase);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "srr_static launch");
}

int tnlm_cnr(const tnlm_params *p, const float *stack, int32_t phase, const int32_t *roi, const int32_t *roi_bg,
             double *out5, void *cuda_stream)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!stack || !roi || !roi_bg || !out5) return TNLM_ERR_NULL_POINTER;
    if (misaligned(stack) || ((uintptr_t)out5 & 7u)) return TNLM_ERR_WORKSPACE;
    if (phase < 0 || phase >= p->n_phase) return TNLM_ERR_BAD_DIMS;
    Box bx[2];
    const int32_t *src[2] = {roi, roi_bg};
    double n[2];
    for (int r = 0; r < 2; ++r) {
        const int32_t *q = src[r];
        if (q[0] < 0 || q[1] > p->nz || q[0] >= q[1] || q[2] < 0 || q[3] > p->ny || q[2] >= q[3] || q[4] < 0 ||
            q[5] > p->nx || q[4] >= q[5])
            return TNLM_ERR_BAD_DIMS;
        bx[r] = Box{q[0], q[1], q[2], q[3], q[4], q[5]};
        n[r] = (double)(q[1] - q[0]) * (q[3] - q[2]) * (q[5] - q[4]);
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMemsetAsync(out5, 0, 5 * sizeof(double), st);
    if (e != cudaSuccess) return cuda_fail(e, "cnr memset");
    const double nmax = n[0] > n[1] ? n[0] : n[1];
    size_t blocks = (size_t)((nmax + kMetricThreads - 1) / kMetricThreads);
    const size_t cap = (size_t)sm_count() * 4;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    const float *vol = stack + (size_t)phase * p->nz * p->ny * p->nx;
    roi_sums_kernel<<<dim3((unsigned)blocks, 2), kMetricThreads, 0, st>>>(vol, p->ny, p->nx, bx[0], bx[1], 0.f, out5);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "cnr sums launch");
    cnr_finish_kernel<<<1, 32, 0, st>>>(out5, n[0], n[1], 0.f, out5);
    e = cudaGetLastError();
    return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "cnr finish launch");
}

const char *tnlm_strerror(int code)
{
    switch (code) {
        case TNLM_OK: return "ok";
        case TNLM_ERR_NULL_POINTER: return "a required pointer is NULL";
        case TNLM_ERR_BAD_DIMS: return "bad dimensions (extent < 1, n_phase < 2, slab out of range or stack too large)";
        case TNLM_ERR_BAD_PARAM: return "bad parameter (h, mu not finite or <= 0; h below 1e-18; negative radius; n_iter < 0)";
        case TNLM_ERR_UNSUPPORTED: return "radius or kernel variant not compiled in";
        case TNLM_ERR_ALIAS: return "output overlaps an input or the workspace";
        case TNLM_ERR_WORKSPACE: return "workspace or stack pointer NULL, too small or not 16-byte aligned";
        case TNLM_ERR_CUDA: return g_cuda_err;
        case TNLM_ERR_TOO_LARGE: return "problem larger than the fixed scratch of a *_static entry point (tnlm_srr_static: n_phase > TNLM_SRR_STATIC_MAX_PHASES)";
        default: return "unknown tnlm status";
    }
}

const char *tnlm_kernel_name(const tnlm_params *p)
{
    if (check_params(p) != TNLM_OK) return "invalid";
    if (pair_tm_supported(*p)) return pair_tm_name(*p);
    if (pair5_supported(*p)) return pair5_name(*p);
    return pair_supported(*p) ? pair_name(*p) : "jacobi_generic_kernel";
}

int32_t tnlm_launches_per_sweep(const tnlm_params *p)
{
    if (check_params(p) != TNLM_OK) return 0;
    return 1;
}

int32_t tnlm_z_tile(const tnlm_params *p)
{
    if (check_params(p) != TNLM_OK) return 0;
    // least common multiple of the tile depths in launch_pair / launch_pair5 / launch_pair_tm (ref == f and separate ref)
    if (pair_supported(*p)) return p->search_radius >= 3 ? 12 : 4;    // <1,4> <2,4> <3,6> <4,4>; TMEM: 4, 6, 6; SEP: 4, 4, 2, 2
    if (pair5_supported(*p)) return p->search_radius <= 3 ? 12 : 4;   // 6|4, 4|2, 4|2, 2|2 (ref == f | SEP); TMEM: 6, 6, 4
    return 1;
}

int tnlm_probe_fp32(int32_t n_iter, float *sink, void *cuda_stream)
{
    if (!sink) return TNLM_ERR_NULL_POINTER;
    if (n_iter < 0) return TNLM_ERR_BAD_PARAM;
    fp32_probe_kernel<<<sm_count() * kProbeBlocksPerSM, kProbeThreads, 0, (cudaStream_t)cuda_stream>>>(
        n_iter, sink, 0.999f, 0.001f);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? TNLM_OK : cuda_fail(e, "fp32 probe launch");
}

double tnlm_probe_fp32_ffma_count(int32_t n_iter)
{
    return (double)sm_count() * kProbeBlocksPerSM * kProbeThreads * (double)kProbeChains * (double)n_iter;
}

}  // extern "C"
