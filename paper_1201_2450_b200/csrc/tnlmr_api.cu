// TNLM-R in libtnlm.so (include/tnlmr.h): Siddon projector pair, CGLS, the outer loop.  The TNLM sweep of steps 2-3
// is tnlm_jacobi_step (tnlm_api.cu).  Not the north-star hot path: written for correctness against oracle/tnlmr_oracle.c
// (one thread per ray, voxel crossings walked incrementally, transpose by atomic adds).
#include <cmath>
#include <cstdio>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/tnlmr.h"

namespace tnlm {
int record_cuda_error(cudaError_t e, const char *where);   // tnlm_api.cu
}

namespace {

struct RGeom {
    int P, Z, Y, X, NV, V, U;
    float inv_voxel, voxel, du, dv, sid, sdd;
};

__device__ __forceinline__ double block_sum(double v, double *sh)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) sh[w] = v;
    __syncthreads();
    v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
    if (w == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;
}

// One thread per ray (phase = blockIdx.y).  BACK = false: y[ray] = sum len * vol[voxel]; BACK = true: vol[voxel] += len * y[ray].
// The ray S + alpha (D - S), alpha in [0, 1], is clipped against the volume and walked from crossing to crossing
// (the radiological path of Siddon 1985 in its incremental form); coordinates are in voxel units from the volume's corner.
template <bool BACK>
__global__ void __launch_bounds__(128) siddon_kernel(const RGeom g, const double2 *__restrict__ trig, const float *__restrict__ vol_in,
                                                     float *__restrict__ vol_out, const float *__restrict__ y_in, float *__restrict__ y_out)
{
    const int ph = blockIdx.y;
    const long long nray = (long long)g.NV * g.V * g.U;
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nray) return;
    const int iu = (int)(r % g.U), iv = (int)((r / g.U) % g.V), view = (int)(r / ((long long)g.U * g.V));
    // The crossing parameters are kept in fp64: a segment is the difference of two parameters ~0.6 whose spacing is
    // ~1e-3, so fp32 parameters would leave 5e-5 of relative error on every intersection length (it cancels along a
    // ray in P f but not in P^T y).  Lengths and data are fp32.
    const double2 cs = trig[ph * g.NV + view];
    const double u = (iu - 0.5 * (g.U - 1)) * (double)g.du, v = (iv - 0.5 * (g.V - 1)) * (double)g.dv;
    const double Sx = g.sid * cs.x, Sy = g.sid * cs.y;
    const double Dx = ((double)g.sid - g.sdd) * cs.x - u * cs.y, Dy = ((double)g.sid - g.sdd) * cs.y + u * cs.x, Dz = v;
    const double L = sqrt((Dx - Sx) * (Dx - Sx) + (Dy - Sy) * (Dy - Sy) + Dz * Dz);
    // voxel units, origin at the volume's low corner
    const double iv_ = 1.0 / (double)g.voxel;
    const double s[3] = {Sx * iv_ + 0.5 * g.X, Sy * iv_ + 0.5 * g.Y, 0.5 * g.Z};
    const double d[3] = {(Dx - Sx) * iv_, (Dy - Sy) * iv_, Dz * iv_};
    const int n[3] = {g.X, g.Y, g.Z};
    double amin = 0.0, amax = 1.0;
    bool hit = true;
    int entry = -1;                                             // axis whose face the ray enters through
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        if (d[k] != 0.0) {
            const double a0 = (0.0 - s[k]) / d[k], a1 = ((double)n[k] - s[k]) / d[k];
            const double lo = fmin(a0, a1);
            if (lo > amin) { amin = lo; entry = k; }
            amax = fmin(amax, fmax(a0, a1));
        } else if (s[k] <= 0.0 || s[k] >= (double)n[k]) {
            hit = false;
        }
    }
    const size_t vbase = (size_t)ph * g.Z * g.Y * g.X;
    const size_t ybase = (size_t)ph * nray + r;
    float acc = 0.f;
    if (hit && amax > amin) {
        int ix, iy, iz, sx, sy, sz;
        double ax, ay, az, dx, dy, dz;
        // first voxel: on the entry axis the one behind the entry face, elsewhere the one that holds the entry point
        auto setup = [&](const int k, int &i, int &st, double &an, double &ad) {
            i = k == entry ? (d[k] > 0.0 ? 0 : n[k] - 1) : (int)floor(s[k] + amin * d[k]);
            i = min(max(i, 0), n[k] - 1);
            if (d[k] > 0.0) { st = 1; an = ((double)(i + 1) - s[k]) / d[k]; ad = 1.0 / d[k]; }
            else if (d[k] < 0.0) { st = -1; an = ((double)i - s[k]) / d[k]; ad = -1.0 / d[k]; }
            else { st = 0; an = 2.0; ad = 0.0; }
        };
        setup(0, ix, sx, ax, dx);
        setup(1, iy, sy, ay, dy);
        setup(2, iz, sz, az, dz);
        const float yr = BACK ? y_in[ybase] : 0.f;
        double ac = amin;
        size_t vi = vbase + ((size_t)iz * g.Y + iy) * g.X + ix;
        const ptrdiff_t stx = sx, sty = (ptrdiff_t)sy * g.X, stz = (ptrdiff_t)sz * g.Y * g.X;
        // one segment per iteration: the nearest crossing ends it (a crossing that rounding put before the entry must
        // not move the walk back; the exit parameter ends the last one); branches instead of 64-bit selects
        for (int it = g.X + g.Y + g.Z + 4; it > 0; --it) {
            double an;
            int axis;
            if (ax <= ay && ax <= az) { an = ax; axis = 0; }
            else if (ay <= az) { an = ay; axis = 1; }
            else { an = az; axis = 2; }
            const bool last = !(an < amax);
            if (last) an = amax;
            if (an > ac) {
                const float len = (float)((an - ac) * L);
                if (BACK) atomicAdd(vol_out + vi, len * yr);
                else acc = fmaf(len, __ldg(vol_in + vi), acc);
                ac = an;
            }
            if (last) break;
            if (axis == 0) { ix += sx; ax += dx; vi += stx; if ((unsigned)ix >= (unsigned)g.X) break; }
            else if (axis == 1) { iy += sy; ay += dy; vi += sty; if ((unsigned)iy >= (unsigned)g.Y) break; }
            else { iz += sz; az += dz; vi += stz; if ((unsigned)iz >= (unsigned)g.Z) break; }
        }
    }
    if (!BACK) y_out[ybase] = acc;
}

__global__ void sub_from_kernel(const float *__restrict__ y, float *__restrict__ r, size_t n)   // r = y - r
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) r[i] = y[i] - r[i];
}

// out[phase] += sum a*b over the phase's n elements (fp64 accumulation, one atomic per block)
__global__ void __launch_bounds__(256) dot_kernel(const float *__restrict__ a, const float *__restrict__ b, size_t n, double *out)
{
    __shared__ double sh[8];
    const int ph = blockIdx.y;
    const float *pa = a + (size_t)ph * n, *pb = b + (size_t)ph * n;
    double s = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        s += (double)pa[i] * (double)pb[i];
    s = block_sum(s, sh);
    if (threadIdx.x == 0) atomicAdd(out + ph, s);
}

// v[phase] += sign * (num[phase] / den[phase]) * w[phase]; a phase whose num or den is not positive is left alone
__global__ void axpy_ratio_kernel(float *__restrict__ v, const float *__restrict__ w, size_t n, const double *num, const double *den,
                                  float sign)
{
    const int ph = blockIdx.y;
    const double nu = num[ph], de = den[ph];
    if (!(nu > 0.0) || !(de > 0.0)) return;
    const float a = sign * (float)(nu / de);
    float *pv = v + (size_t)ph * n;
    const float *pw = w + (size_t)ph * n;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) pv[i] = fmaf(a, pw[i], pv[i]);
}

// p[phase] = s[phase] + (gnew/gold) p[phase]   (beta = 0 where gold is not positive)
__global__ void update_dir_kernel(float *__restrict__ p, const float *__restrict__ s, size_t n, const double *gnew, const double *gold)
{
    const int ph = blockIdx.y;
    const double go = gold[ph];
    const float beta = go > 0.0 ? (float)(gnew[ph] / go) : 0.f;
    float *pp = p + (size_t)ph * n;
    const float *ps = s + (size_t)ph * n;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) pp[i] = fmaf(beta, pp[i], ps[i]);
}

__global__ void clamp_kernel(float *__restrict__ f, size_t n)   // step 4: f = max(f, 0)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) f[i] = fmaxf(f[i], 0.f);
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
bool misaligned(const void *p) { return ((uintptr_t)p & 15u) != 0; }
bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    if (!a || !b || na == 0 || nb == 0) return false;
    const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    return x < y + nb && y < x + na;
}

int check_geom(const tnlmr_geometry *g)
{
    if (!g) return TNLM_ERR_NULL_POINTER;
    if (g->n_phase < 1 || g->nz < 1 || g->ny < 1 || g->nx < 1 || g->n_view < 1 || g->nv < 1 || g->nu < 1) return TNLM_ERR_BAD_DIMS;
    if ((double)g->n_phase * g->nz * g->ny * g->nx > 2147483647.0) return TNLM_ERR_BAD_DIMS;
    if ((double)g->n_phase * g->n_view * g->nv * g->nu > 2147483647.0) return TNLM_ERR_BAD_DIMS;
    const float vals[5] = {g->voxel, g->du, g->dv, g->sid, g->sdd};
    for (float v : vals)
        if (!(v > 0.f) || !std::isfinite(v)) return TNLM_ERR_BAD_PARAM;
    // the source must lie outside the volume's circumscribed cylinder and the detector behind the isocentre
    const double rad = 0.5 * g->voxel * std::sqrt((double)g->nx * g->nx + (double)g->ny * g->ny);
    if (!(g->sid > rad) || !(g->sdd > g->sid)) return TNLM_ERR_BAD_PARAM;
    return TNLM_OK;
}

size_t vol_bytes(const tnlmr_geometry *g) { return (size_t)g->n_phase * g->nz * g->ny * g->nx * sizeof(float); }
size_t proj_bytes(const tnlmr_geometry *g) { return (size_t)g->n_phase * g->n_view * g->nv * g->nu * sizeof(float); }
size_t trig_bytes(const tnlmr_geometry *g) { return align_up((size_t)g->n_phase * g->n_view * sizeof(double2), 256); }
size_t scalar_bytes(const tnlmr_geometry *g) { return align_up(3 * (size_t)g->n_phase * sizeof(double), 256); }

// workspace: [trig][scalars][r][q][s][p]  (+ [g^(k)][tnlm workspace] for tnlmr_reconstruct)
struct Carve {
    double2 *trig; double *gamma, *qq, *gnew; float *r, *q, *s, *p; char *rest; size_t rest_bytes;
};
size_t cgls_bytes(const tnlmr_geometry *g)
{
    return trig_bytes(g) + scalar_bytes(g) + 2 * align_up(proj_bytes(g), 256) + 2 * align_up(vol_bytes(g), 256);
}
Carve carve(const tnlmr_geometry *g, void *ws, size_t ws_bytes)
{
    Carve c;
    char *b = (char *)ws;
    c.trig = (double2 *)b; b += trig_bytes(g);
    c.gamma = (double *)b; c.qq = c.gamma + g->n_phase; c.gnew = c.qq + g->n_phase; b += scalar_bytes(g);
    c.r = (float *)b; b += align_up(proj_bytes(g), 256);
    c.q = (float *)b; b += align_up(proj_bytes(g), 256);
    c.s = (float *)b; b += align_up(vol_bytes(g), 256);
    c.p = (float *)b; b += align_up(vol_bytes(g), 256);
    c.rest = b;
    c.rest_bytes = ws_bytes - (size_t)(b - (char *)ws);
    return c;
}

RGeom make_rgeom(const tnlmr_geometry *g)
{
    RGeom r;
    r.P = g->n_phase; r.Z = g->nz; r.Y = g->ny; r.X = g->nx; r.NV = g->n_view; r.V = g->nv; r.U = g->nu;
    r.voxel = g->voxel; r.inv_voxel = 1.0f / g->voxel; r.du = g->du; r.dv = g->dv; r.sid = g->sid; r.sdd = g->sdd;
    return r;
}

int cuda_fail(cudaError_t e, const char *where) { return tnlm::record_cuda_error(e, where); }   // text for tnlm_strerror
#define CU(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, where); } while (0)

int upload_trig(const tnlmr_geometry *g, const double *angles, double2 *trig, cudaStream_t st)
{
    const size_t n = (size_t)g->n_phase * g->n_view;
    std::vector<double2> h(n);
    for (size_t i = 0; i < n; ++i) h[i] = make_double2(std::cos(angles[i]), std::sin(angles[i]));
    // pageable source: the copy is staged before the call returns, so the vector may go out of scope
    CU(cudaMemcpyAsync(trig, h.data(), n * sizeof(double2), cudaMemcpyHostToDevice, st), "angle table upload");
    CU(cudaStreamSynchronize(st), "angle table upload");
    return TNLM_OK;
}

unsigned blocks_for(size_t n, unsigned threads, unsigned cap) { size_t b = (n + threads - 1) / threads; return (unsigned)(b < 1 ? 1 : (b > cap ? cap : b)); }

int launch_project(const tnlmr_geometry *g, const double2 *trig, const float *f, float *y, cudaStream_t st)
{
    const long long nray = (long long)g->n_view * g->nv * g->nu;
    const dim3 grid((unsigned)((nray + 127) / 128), (unsigned)g->n_phase);
    siddon_kernel<false><<<grid, 128, 0, st>>>(make_rgeom(g), trig, f, nullptr, nullptr, y);
    CU(cudaGetLastError(), "project launch");
    return TNLM_OK;
}

int launch_backproject(const tnlmr_geometry *g, const double2 *trig, const float *y, float *f, cudaStream_t st)
{
    CU(cudaMemsetAsync(f, 0, vol_bytes(g), st), "backproject clear");
    const long long nray = (long long)g->n_view * g->nv * g->nu;
    const dim3 grid((unsigned)((nray + 127) / 128), (unsigned)g->n_phase);
    siddon_kernel<true><<<grid, 128, 0, st>>>(make_rgeom(g), trig, nullptr, f, y, nullptr);
    CU(cudaGetLastError(), "backproject launch");
    return TNLM_OK;
}

int launch_dot(const tnlmr_geometry *g, const float *a, const float *b, size_t n_per_phase, double *out, cudaStream_t st)
{
    CU(cudaMemsetAsync(out, 0, sizeof(double) * g->n_phase, st), "dot clear");
    const dim3 grid(blocks_for(n_per_phase, 256, 1184), (unsigned)g->n_phase);
    dot_kernel<<<grid, 256, 0, st>>>(a, b, n_per_phase, out);
    CU(cudaGetLastError(), "dot launch");
    return TNLM_OK;
}

// CGLS on all phases at once, scalars per phase (reading R5; oracle/tnlmr_oracle.c: tnlmr_ref_cgls)
int run_cgls(const tnlmr_geometry *g, const Carve &c, const float *y, float *x, int n_iter, cudaStream_t st)
{
    const size_t nv = (size_t)g->nz * g->ny * g->nx, np = (size_t)g->n_view * g->nv * g->nu;
    const dim3 gv(blocks_for(nv, 256, 2368), (unsigned)g->n_phase), gp(blocks_for(np, 256, 2368), (unsigned)g->n_phase);
    int rc;
    if ((rc = launch_project(g, c.trig, x, c.r, st))) return rc;
    sub_from_kernel<<<blocks_for(np * g->n_phase, 256, 4736), 256, 0, st>>>(y, c.r, np * g->n_phase);   // r = y - P x
    if ((rc = launch_backproject(g, c.trig, c.r, c.s, st))) return rc;                                     // s = P^T r
    CU(cudaMemcpyAsync(c.p, c.s, vol_bytes(g), cudaMemcpyDeviceToDevice, st), "cgls p = s");
    if ((rc = launch_dot(g, c.s, c.s, nv, c.gamma, st))) return rc;
    for (int it = 0; it < n_iter; ++it) {
        if ((rc = launch_project(g, c.trig, c.p, c.q, st))) return rc;                                     // q = P p
        if ((rc = launch_dot(g, c.q, c.q, np, c.qq, st))) return rc;
        axpy_ratio_kernel<<<gv, 256, 0, st>>>(x, c.p, nv, c.gamma, c.qq, 1.f);                             // x += alpha p
        axpy_ratio_kernel<<<gp, 256, 0, st>>>(c.r, c.q, np, c.gamma, c.qq, -1.f);                          // r -= alpha q
        if ((rc = launch_backproject(g, c.trig, c.r, c.s, st))) return rc;                                 // s = P^T r
        if ((rc = launch_dot(g, c.s, c.s, nv, c.gnew, st))) return rc;
        update_dir_kernel<<<gv, 256, 0, st>>>(c.p, c.s, nv, c.gnew, c.gamma);                              // p = s + beta p
        CU(cudaMemcpyAsync(c.gamma, c.gnew, sizeof(double) * g->n_phase, cudaMemcpyDeviceToDevice, st), "cgls gamma");
        CU(cudaGetLastError(), "cgls iteration");
    }
    return TNLM_OK;
}

}  // namespace

extern "C" {

size_t tnlmr_workspace_bytes(const tnlmr_geometry *g, const tnlm_params *p)
{
    if (check_geom(g) != TNLM_OK) return 0;
    size_t n = cgls_bytes(g);
    if (p) {
        if (p->n_phase != g->n_phase || p->nz != g->nz || p->ny != g->ny || p->nx != g->nx) return 0;
        const size_t t = tnlm_workspace_bytes(p);
        if (t == 0) return 0;
        n += align_up(vol_bytes(g), 256) + t;
    }
    return n;
}

int tnlmr_project(const tnlmr_geometry *g, const double *angles, const float *f, float *y, void *ws, size_t ws_bytes, void *cuda_stream)
{
    int rc = check_geom(g);
    if (rc) return rc;
    if (!angles || !f || !y) return TNLM_ERR_NULL_POINTER;
    if (!ws || misaligned(ws) || ws_bytes < trig_bytes(g) || misaligned(f) || misaligned(y)) return TNLM_ERR_WORKSPACE;
    if (overlaps(y, proj_bytes(g), f, vol_bytes(g))) return TNLM_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = upload_trig(g, angles, (double2 *)ws, st))) return rc;
    return launch_project(g, (const double2 *)ws, f, y, st);
}

int tnlmr_backproject(const tnlmr_geometry *g, const double *angles, const float *y, float *f, void *ws, size_t ws_bytes, void *cuda_stream)
{
    int rc = check_geom(g);
    if (rc) return rc;
    if (!angles || !f || !y) return TNLM_ERR_NULL_POINTER;
    if (!ws || misaligned(ws) || ws_bytes < trig_bytes(g) || misaligned(f) || misaligned(y)) return TNLM_ERR_WORKSPACE;
    if (overlaps(y, proj_bytes(g), f, vol_bytes(g))) return TNLM_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = upload_trig(g, angles, (double2 *)ws, st))) return rc;
    return launch_backproject(g, (const double2 *)ws, y, f, st);
}

int tnlmr_cgls(const tnlmr_geometry *g, const double *angles, const float *y, float *x, int32_t n_iter, void *ws, size_t ws_bytes,
               void *cuda_stream)
{
    int rc = check_geom(g);
    if (rc) return rc;
    if (!angles || !x || !y) return TNLM_ERR_NULL_POINTER;
    if (n_iter < 0) return TNLM_ERR_BAD_PARAM;
    if (!ws || misaligned(ws) || ws_bytes < cgls_bytes(g) || misaligned(x) || misaligned(y)) return TNLM_ERR_WORKSPACE;
    if (overlaps(y, proj_bytes(g), x, vol_bytes(g)) || overlaps(ws, ws_bytes, x, vol_bytes(g)) || overlaps(ws, ws_bytes, y, proj_bytes(g)))
        return TNLM_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Carve c = carve(g, ws, ws_bytes);
    if ((rc = upload_trig(g, angles, c.trig, st))) return rc;
    return run_cgls(g, c, y, x, n_iter, st);
}

int tnlmr_reconstruct(const tnlmr_geometry *g, const tnlm_params *p, const double *angles, const float *y, const float *f_init,
                      float *f_out, int32_t n_outer, int32_t n_cgls, int32_t inner_start, void *ws, size_t ws_bytes, void *cuda_stream)
{
    int rc = check_geom(g);
    if (rc) return rc;
    if (!p || !angles || !y || !f_init || !f_out) return TNLM_ERR_NULL_POINTER;
    if (p->n_phase != g->n_phase || p->nz != g->nz || p->ny != g->ny || p->nx != g->nx) return TNLM_ERR_BAD_DIMS;
    if (n_outer < 0 || n_cgls < 0 || (inner_start != TNLMR_START_G && inner_start != TNLMR_START_PREVIOUS)) return TNLM_ERR_BAD_PARAM;
    const size_t need = tnlmr_workspace_bytes(g, p);
    if (need == 0) return TNLM_ERR_BAD_PARAM;
    if (!ws || misaligned(ws) || ws_bytes < need || misaligned(y) || misaligned(f_init) || misaligned(f_out)) return TNLM_ERR_WORKSPACE;
    const size_t vb = vol_bytes(g), pb = proj_bytes(g);
    if (overlaps(f_out, vb, f_init, vb) || overlaps(f_out, vb, y, pb) || overlaps(ws, ws_bytes, f_out, vb) ||
        overlaps(ws, ws_bytes, f_init, vb) || overlaps(ws, ws_bytes, y, pb))
        return TNLM_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Carve c = carve(g, ws, ws_bytes);
    float *gk = (float *)c.rest;
    void *tws = c.rest + align_up(vb, 256);
    const size_t tws_bytes = c.rest_bytes - align_up(vb, 256);
    if ((rc = upload_trig(g, angles, c.trig, st))) return rc;
    if (n_outer == 0) {
        CU(cudaMemcpyAsync(f_out, f_init, vb, cudaMemcpyDeviceToDevice, st), "reconstruct copy");
        return TNLM_OK;
    }
    const size_t nel = vb / sizeof(float);
    const float *prev = f_init;                                    // f^(k-1)
    for (int k = 0; k < n_outer; ++k) {
        // step 1: g^(k) = CGLS from f^(k-1)
        CU(cudaMemcpyAsync(gk, prev, vb, cudaMemcpyDeviceToDevice, st), "reconstruct start");
        if ((rc = run_cgls(g, c, y, gk, n_cgls, st))) return rc;
        // steps 2-3: weights from g^(k), one sweep of Eq. 8 with g = g^(k)
        if (inner_start == TNLMR_START_G) {
            rc = tnlm_jacobi_step(p, gk, gk, nullptr, f_out, tws, tws_bytes, cuda_stream);
        } else {
            // f^(k-1) is f_out itself from the second iteration on: keep a copy in the CGLS direction buffer
            const float *start = prev;
            if (prev == f_out) {
                CU(cudaMemcpyAsync(c.p, f_out, vb, cudaMemcpyDeviceToDevice, st), "reconstruct keep f^(k-1)");
                start = c.p;
            }
            rc = tnlm_jacobi_step(p, start, gk, gk, f_out, tws, tws_bytes, cuda_stream);
        }
        if (rc) return rc;
        clamp_kernel<<<blocks_for(nel, 256, 4736), 256, 0, st>>>(f_out, nel);                              // step 4
        CU(cudaGetLastError(), "clamp launch");
        prev = f_out;
    }
    return TNLM_OK;
}

}  // extern "C"
