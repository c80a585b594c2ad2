// Shared device helpers of libtnlm (CUDA path only; nothing here is used by the CPU oracle).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

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

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the (kernel, device) pair: set it once per device the
// process launches on (bit d of `done`; devices >= 64 set it on every launch).  Safe from concurrent host threads:
// the call is idempotent and the bit is only set after it succeeded.
template <typename Kernel>
inline cudaError_t ensure_dynamic_smem(Kernel kernel, size_t bytes, std::atomic<uint64_t> &done)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const uint64_t bit = dev < 64 ? (1ull << dev) : 0ull;
    if (bit && (done.load(std::memory_order_acquire) & bit)) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess && bit) done.fetch_or(bit, std::memory_order_release);
    return e;
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
