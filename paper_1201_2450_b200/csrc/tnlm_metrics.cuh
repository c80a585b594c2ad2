// Evaluation metrics of the paper as CUDA kernels: TV seminorm of a difference stack (Eq. 10,
// PAPER.md:269-272), streak-reduction ratio, ROI statistics and CNR.  HBM-bound
// reductions: every voxel of the operands is read once from DRAM (the +1 neighbours of the forward
// differences hit L1/L2), fp64 accumulation, warp shuffles, one atomicAdd(double) per CTA.
#pragma once
#include "tnlm_common.cuh"

namespace tnlm {

constexpr int kMetricThreads = 256;

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// CTA-wide sum of NV running values; thread 0 adds the totals to dst[0..NV) with atomicAdd.
template <int NV>
__device__ __forceinline__ void block_accumulate(double (&v)[NV], double *dst)
{
    __shared__ double part[NV][kMetricThreads / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const double s = warp_sum(v[k]);
        if (lane == 0) part[k][warp] = s;
    }
    __syncthreads();
    if (threadIdx.x < NV) {
        double s = 0.0;
        for (int w = 0; w < kMetricThreads / 32; ++w) s += part[threadIdx.x][w];
        atomicAdd(dst + threadIdx.x, s);
    }
}

// Four consecutive values h = a - b of a row (fp32); vec: the quad is 16-byte aligned.
__device__ __forceinline__ void load_h4(const float *__restrict__ ap, const float *__restrict__ bp, const size_t idx,
                                        const int n, const bool vec, float (&c)[4])
{
    if (vec) {
        const float4 av = __ldg(reinterpret_cast<const float4 *>(ap + idx));
        float4 bv = make_float4(0.f, 0.f, 0.f, 0.f);
        if (bp) bv = __ldg(reinterpret_cast<const float4 *>(bp + idx));
        c[0] = av.x - bv.x; c[1] = av.y - bv.y; c[2] = av.z - bv.z; c[3] = av.w - bv.w;
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) c[k] = k < n ? __ldg(ap + idx + k) - (bp ? __ldg(bp + idx + k) : 0.f) : 0.f;
    }
}

// tv[p] += sum over the voxels of phase p of |grad (a - b)| (forward differences, 0 across the boundary).
// A CTA is a tile of kTvXQ x-quads x 256/kTvXQ rows that marches kTvZChunk planes: a thread handles 4 consecutive x of one row
// and keeps the next plane's quad in registers, so the plane-down difference costs no second read; the row-down quad
// and the scalar right of the quad are re-reads inside the CTA's own tile (L1) except at its last row.  Every voxel
// thus crosses L2 about 1.3 times (the first, grid-stride form read every operand three times from L2 and was bound
// by it at 0.4 of the HBM roofline).  Per-voxel arithmetic in fp32 (each |grad h| is good to ~3 ulp = 2e-7 relative,
// and the terms are non-negative, so the sum inherits that bound: DESIGN.md M4), accumulation in fp64.
constexpr int kTvZChunk = 16;

template <int kTvXQ>   // x-quads per CTA row: 64, or fewer for narrow volumes so that no thread idles
__global__ void __launch_bounds__(kMetricThreads)
tv_diff_kernel(const float *__restrict__ a, const float *__restrict__ b, double *__restrict__ tv, const int Z,
               const int Y, const int X, const int tiles_xq, const int tiles_y)
{
    constexpr int kTvRows = kMetricThreads / kTvXQ;
    const int ph = blockIdx.y;
    const size_t V = (size_t)Z * Y * X;
    const float *ap = a + ph * V;
    const float *bp = b ? b + ph * V : nullptr;
    int t = blockIdx.x;
    const int bxq = t % tiles_xq; t /= tiles_xq;
    const int by = t % tiles_y; t /= tiles_y;
    const int z0 = t * kTvZChunk, z1 = min(z0 + kTvZChunk, Z);
    const int xg = bxq * kTvXQ + (threadIdx.x % kTvXQ), y = by * kTvRows + threadIdx.x / kTvXQ;
    const bool vec = (X % 4) == 0;
    double acc[1] = {0.0};
    if (4 * xg < X && y < Y) {
        const int n = min(4, X - 4 * xg);
        const bool has_y = y + 1 < Y, has_next = 4 * xg + n < X;
        const size_t plane = (size_t)Y * X;
        size_t base = ((size_t)z0 * Y + y) * X + 4 * xg;
        float c[4], cz[4];
        load_h4(ap, bp, base, n, vec, c);
        for (int z = z0; z < z1; ++z, base += plane) {
            const bool has_z = z + 1 < Z;
            float cy[4];
            if (has_z) load_h4(ap, bp, base + plane, n, vec, cz);
            if (has_y) load_h4(ap, bp, base + X, n, vec, cy);
            float cnext = 0.f;                         // h at x + n (first voxel of the next quad), if inside the row
            if (has_next) cnext = __ldg(ap + base + n) - (bp ? __ldg(bp + base + n) : 0.f);
            float quad = 0.f;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (k < n) {
                    const bool last_x = (4 * xg + k == X - 1);
                    const float nx = (k + 1 < n) ? c[(k + 1) & 3] : cnext;
                    const float gx = last_x ? 0.f : nx - c[k];
                    const float gy = has_y ? cy[k] - c[k] : 0.f;
                    const float gz = has_z ? cz[k] - c[k] : 0.f;
                    quad += sqrtf(fmaf(gx, gx, fmaf(gy, gy, gz * gz)));
                }
            }
            acc[0] += (double)quad;
#pragma unroll
            for (int k = 0; k < 4; ++k) c[k] = cz[k];
        }
    }
    block_accumulate<1>(acc, tv + ph);
}

// srr[p] = (t0[p] - t1[p]) / t0[p]
__global__ void srr_finish_kernel(const double *__restrict__ t, double *__restrict__ srr, const int P)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < P) srr[p] = (t[p] - t[P + p]) / t[p];
}

struct Box { int z0, z1, y0, y1, x0, x1; };

// sums[2*r + {0,1}] += (sum, sum of squares about `shift`) over box r (r = blockIdx.y) of one phase volume
__global__ void __launch_bounds__(kMetricThreads)
roi_sums_kernel(const float *__restrict__ vol, const int Y, const int X, const Box b0, const Box b1,
                const float shift, double *__restrict__ sums)
{
    const Box bx = blockIdx.y ? b1 : b0;
    const int nx = bx.x1 - bx.x0, ny = bx.y1 - bx.y0, nz = bx.z1 - bx.z0;
    const size_t n = (size_t)nx * ny * nz;
    double acc[2] = {0.0, 0.0};
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int x = bx.x0 + (int)(i % nx);
        const int y = bx.y0 + (int)((i / nx) % ny);
        const int z = bx.z0 + (int)(i / ((size_t)nx * ny));
        const double v = (double)__ldg(vol + ((size_t)z * Y + y) * X + x) - (double)shift;
        acc[0] += v;
        acc[1] += v * v;
    }
    block_accumulate<2>(acc, sums + 2 * blockIdx.y);
}

// out5 = { S, sigma, S_b, sigma_b, 2 |S - S_b| / (sigma + sigma_b) }
__global__ void cnr_finish_kernel(const double *sums, const double n0, const double n1, const float shift, double *out5)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        const double a0 = sums[0], a1 = sums[1], a2 = sums[2], a3 = sums[3];   // sums and out5 may be the same buffer
        const double m0 = a0 / n0, m1 = a2 / n1;
        const double s0 = sqrt(fmax(a1 / n0 - m0 * m0, 0.0)), s1 = sqrt(fmax(a3 / n1 - m1 * m1, 0.0));
        const double S = m0 + (double)shift, Sb = m1 + (double)shift;
        out5[0] = S; out5[1] = s0; out5[2] = Sb; out5[3] = s1;
        out5[4] = 2.0 * fabs(S - Sb) / (s0 + s1);
    }
}

}  // namespace tnlm
