// Shared device helpers of libtnlm (CUDA path only; nothing here is used by the CPU oracle).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tnlm.h"

namespace tnlm {

// exp(-D/(2h^2)) = exp2(-c2 * D) with c2 = log2(e)/(2h^2)        (Eq. 3)
__host__ __device__ inline float exp2_scale(float h) { return 1.4426950408889634f / (2.0f * h * h); }

__device__ __forceinline__ int clampi(int v, int n) { return min(max(v, 0), n - 1); }

__device__ __forceinline__ float ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

struct Dims {
    int P, Z, Y, X;
    int d, M;
    float c2;       // log2(e)/(2h^2)
    float a_g;      // mu/(2+mu)
    float a_n;      // 1/(2+mu)
    int z_begin, z_end;   // output slab
};

inline Dims make_dims(const tnlm_params &p, int z_begin, int z_end)
{
    Dims D;
    D.P = p.n_phase; D.Z = p.nz; D.Y = p.ny; D.X = p.nx;
    D.d = p.patch_radius; D.M = p.search_radius;
    D.c2 = exp2_scale(p.h);
    D.a_g = p.mu / (2.0f + p.mu);
    D.a_n = 1.0f / (2.0f + p.mu);
    D.z_begin = z_begin; D.z_end = z_end;
    return D;
}

}  // namespace tnlm
