// Generic (any d, M) TNLM kernels: one thread per output voxel, loops written as the definition.
// These are the correctness baseline of the CUDA path and the fallback for (d, M) pairs the tiled
// kernel is not compiled for; tnlm_weights (inspection only) also lives here.
#pragma once
#include "tnlm_common.cuh"

namespace tnlm {

// D_t(x) of Eq. 3 / Eq. 9 with clamp-to-edge reads (reading P4).
__device__ __forceinline__ float patch_distance(const float *__restrict__ ri, const float *__restrict__ rj,
                                                const Dims &dm, int z, int y, int x, int tz, int ty, int tx)
{
    float D = 0.f;
    for (int dz = -dm.d; dz <= dm.d; ++dz) {
        const int za = clampi(z + dz, dm.Z), zb = clampi(z + tz + dz, dm.Z);
        for (int dy = -dm.d; dy <= dm.d; ++dy) {
            const int ya = clampi(y + dy, dm.Y), yb = clampi(y + ty + dy, dm.Y);
            const float *ra = ri + ((size_t)za * dm.Y + ya) * dm.X;
            const float *rb = rj + ((size_t)zb * dm.Y + yb) * dm.X;
            for (int dx = -dm.d; dx <= dm.d; ++dx) {
                const float diff = __ldg(ra + clampi(x + dx, dm.X)) - __ldg(rb + clampi(x + tx + dx, dm.X));
                D = fmaf(diff, diff, D);
            }
        }
    }
    return D;
}

// NLM_s(x) = sum_t w_t f_j(x+t), bracket of Eq. 8, with a running reference exponent
// (online form of the softmax-shifted weights, reading P3).
__device__ __forceinline__ float nlm_one_direction(const float *__restrict__ ri, const float *__restrict__ rj,
                                                   const float *__restrict__ fj, const Dims &dm, int z, int y, int x)
{
    float Dm = INFINITY, Zs = 0.f, Ns = 0.f;
    for (int tz = -dm.M; tz <= dm.M; ++tz)
        for (int ty = -dm.M; ty <= dm.M; ++ty)
            for (int tx = -dm.M; tx <= dm.M; ++tx) {
                const float D = patch_distance(ri, rj, dm, z, y, x, tz, ty, tx);
                if (D < Dm) {  // new best candidate: rescale what was accumulated so far
                    const float sc = ex2((D - Dm) * dm.c2);   // Dm = inf -> ex2(-inf) = 0
                    Zs *= sc;
                    Ns *= sc;
                    Dm = D;
                }
                const float u = ex2((Dm - D) * dm.c2);
                const float v = __ldg(fj + ((size_t)clampi(z + tz, dm.Z) * dm.Y + clampi(y + ty, dm.Y)) * dm.X +
                                      clampi(x + tx, dm.X));
                Zs += u;
                Ns = fmaf(u, v, Ns);
            }
    return Ns / Zs;
}

__global__ void __launch_bounds__(256)
jacobi_generic_kernel(const float *__restrict__ f, const float *__restrict__ g, const float *__restrict__ ref,
                      float *__restrict__ f_out, Dims dm)
{
    const size_t V = (size_t)dm.Z * dm.Y * dm.X;
    const size_t slabV = (size_t)(dm.z_end - dm.z_begin) * dm.Y * dm.X;
    const size_t total = slabV * dm.P;
    for (size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x; id < total; id += (size_t)gridDim.x * blockDim.x) {
        const int ph = (int)(id / slabV);
        size_t r = id % slabV;
        const int z = dm.z_begin + (int)(r / ((size_t)dm.Y * dm.X));
        r %= (size_t)dm.Y * dm.X;
        const int y = (int)(r / dm.X), x = (int)(r % dm.X);
        const int jp = (ph + 1) % dm.P, jm = (ph + dm.P - 1) % dm.P;
        const float nlm_p = nlm_one_direction(ref + ph * V, ref + jp * V, f + jp * V, dm, z, y, x);
        const float nlm_m = nlm_one_direction(ref + ph * V, ref + jm * V, f + jm * V, dm, z, y, x);
        const size_t o = ph * V + ((size_t)z * dm.Y + y) * dm.X + x;
        f_out[o] = fmaf(dm.a_g, __ldg(g + o), dm.a_n * (nlm_p + nlm_m));   // Eq. 8
    }
}

// w_out[p][s][k][z][y][x].  Every patch distance is computed once: pass 1 parks D_k in w_out[k] (the thread's own
// column of the output) and finds the smallest one, pass 2 turns the parked distances into exp2((Dmin - D_k) c2)
// (the shifted form, reading P3) and sums the normaliser, pass 3 scales.  w_out must not alias ref (checked by
// the caller), so the __ldg reads of ref stay valid while w_out is written.
__global__ void __launch_bounds__(256)
weights_generic_kernel(const float *__restrict__ ref, float *w_out, Dims dm)
{
    const size_t V = (size_t)dm.Z * dm.Y * dm.X;
    const size_t total = V * dm.P * 2;
    const int e = 2 * dm.M + 1;
    const size_t nt = (size_t)e * e * e;
    for (size_t id = (size_t)blockIdx.x * blockDim.x + threadIdx.x; id < total; id += (size_t)gridDim.x * blockDim.x) {
        const size_t vox = id % V;
        const int s = (int)((id / V) % 2);
        const int ph = (int)(id / (2 * V));
        const int z = (int)(vox / ((size_t)dm.Y * dm.X));
        const int y = (int)((vox / dm.X) % dm.Y), x = (int)(vox % dm.X);
        const int j = (ph + (s ? 1 : dm.P - 1)) % dm.P;
        const float *ri = ref + ph * V, *rj = ref + j * V;
        float *w = w_out + ((size_t)ph * 2 + s) * nt * V + vox;   // w[k * V], k = 0 .. nt-1
        float Dm = INFINITY;
        size_t k = 0;
        for (int tz = -dm.M; tz <= dm.M; ++tz)
            for (int ty = -dm.M; ty <= dm.M; ++ty)
                for (int tx = -dm.M; tx <= dm.M; ++tx, ++k) {
                    const float D = patch_distance(ri, rj, dm, z, y, x, tz, ty, tx);
                    w[k * V] = D;
                    Dm = fminf(Dm, D);
                }
        float Zs = 0.f;
        for (k = 0; k < nt; ++k) {
            const float u = ex2((Dm - w[k * V]) * dm.c2);
            w[k * V] = u;
            Zs += u;
        }
        const float inv = 1.0f / Zs;
        for (k = 0; k < nt; ++k) w[k * V] *= inv;
    }
}

// Register-resident FFMA loop for the measured FP32 peak.
constexpr int kProbeChains = 16;
constexpr int kProbeThreads = 256;
constexpr int kProbeBlocksPerSM = 8;

__global__ void __launch_bounds__(kProbeThreads)
fp32_probe_kernel(int n_iter, float *sink, float a, float b)
{
    float acc[kProbeChains];
#pragma unroll
    for (int i = 0; i < kProbeChains; ++i) acc[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < n_iter; ++it) {
#pragma unroll
        for (int i = 0; i < kProbeChains; ++i) acc[i] = fmaf(acc[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kProbeChains; ++i) s += acc[i];
    if (s == 12345.678f) *sink = s;   // never true in practice; keeps the loop alive
}

}  // namespace tnlm
