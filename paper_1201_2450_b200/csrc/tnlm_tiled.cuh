// Tiled sm_100a TNLM sweep kernel for 3^3 patches (d = 1), search radius M in {1,2,3,4}.
//
// One CTA = one (phase i, x-tile, y-group, z-slab) and both neighbour phases j = i-1, i+1
// (Eq. 8).  The CTA stages a halo tile of ref_i (halo d) and of ref_j = f_j (halo
// d+M, clamp-to-edge applied while staging: reading P4) in shared memory once, then every warp
// runs without any further block-level synchronisation:
//
//   lane        = one y-row (32 rows per warp, rows 0 and 31 are the d-halo: 30 outputs)
//   thread      = an x-run of 4 voxels x 1 row x a column of RZ output planes
//   registers   = the accumulators (Z, N, reference exponent) of its 4*RZ outputs, for the whole
//                 search window; nothing per-offset ever leaves the register file
//   per (ty,tz) = a "pass": march the RZ+2 planes; per plane
//       a1  diffs (ref_i - ref_j(+t)) for the 2M+1 (or a chunk of) tx at once from one float4 row window
//       a2x 3-tap x-sum of squares, in registers, two outputs share the middle pair
//       a2y 3-tap y-sum through two warp shuffles (lanes are rows)
//       a2z 3-tap z-sum from a two-plane register ring
//       a3  u = ex2(bias - c2*D)    (one FFMA + one MUFU; bias = lazily updated reference exponent)
//       a4  Z += u, N += u * f_j(x+t)   (candidate value = centre of the row window already in registers)
//   epilogue    = a5: f_out = mu/(2+mu) g + (N-/Z- + N+/Z+)/(2+mu)
//
// The reference exponent (reading P3: weights relative to the best candidate) is handled lazily:
// a pass adds its terms optimistically and checks the partial normaliser; only if a term overflowed
// the 2^60 guard band is that output re-based (rare, cold path).  The result equals the shifted
// softmax up to rounding.
#pragma once
#include <cstdlib>

#include "tnlm_common.cuh"

namespace tnlm {

constexpr int kTiledWarps = 8;                 // warps per CTA, one x-run each: TX = 32
constexpr int kTiledTX = 4 * kTiledWarps;
constexpr int kTiledRowsOut = 30;              // valid output rows per warp (32 lanes - 2 halo rows)
constexpr float kGuard = 1.152921504606847e18f;   // 2^60

template <int M> struct TiledGeom {
    static constexpr int HXB = (M + 1 <= 4) ? 4 : 8;                    // x halo of the B tile, multiple of 4
    static constexpr int PA = kTiledTX + 4;                             // A pitch: 36 = 4 * odd -> conflict-free LDS.128
    static constexpr int WB = ((HXB + 5 + M) + 3) / 4 * 4;              // B row window words per thread
    static constexpr int PB_MIN = kTiledTX - 4 + WB;
    static constexpr int PB = (PB_MIN % 8 == 4) ? PB_MIN : PB_MIN + 4;  // 4 * odd
    static constexpr int RA = 32;                                       // A rows
    static constexpr int RB = 32 + 2 * M;                               // B rows
};

template <int M, int RZ> struct TiledSmem {
    using G = TiledGeom<M>;
    static constexpr int NA = RZ + 2, NB = RZ + 2 + 2 * M;
    static constexpr int A_WORDS = NA * G::RA * G::PA;
    static constexpr int B_WORDS = NB * G::RB * G::PB;
    static constexpr size_t BYTES = (size_t)(A_WORDS + B_WORDS) * sizeof(float);
};

struct Acc4 { float z[4], n[4], b[4]; };   // normaliser, weighted sum, reference exponent (log2 units) of an x-run

// Cold path: re-base one output on the best candidate of this pass, then add the pass's terms.
template <int W>
__device__ __noinline__ float3 rebase_and_add(float Z, float N, float bias, float c2,
                                              float D0, float D1, float D2, float D3, float D4,
                                              float v0, float v1, float v2, float v3, float v4)
{
    float Dmin = D0;
    if (W > 1) Dmin = fminf(Dmin, D1);
    if (W > 2) Dmin = fminf(Dmin, D2);
    if (W > 3) Dmin = fminf(Dmin, D3);
    if (W > 4) Dmin = fminf(Dmin, D4);
    const float nb = c2 * Dmin;
    if (nb < bias) {                         // a better candidate than any seen so far
        const float sc = ex2(nb - bias);     // bias = +inf on first use -> ex2(-inf) = 0, and Z = N = 0
        Z *= sc;
        N *= sc;
        bias = nb;
    }
    float u;
    u = ex2(fmaf(-c2, D0, bias)); Z += u; N = fmaf(u, v0, N);
    if (W > 1) { u = ex2(fmaf(-c2, D1, bias)); Z += u; N = fmaf(u, v1, N); }
    if (W > 2) { u = ex2(fmaf(-c2, D2, bias)); Z += u; N = fmaf(u, v2, N); }
    if (W > 3) { u = ex2(fmaf(-c2, D3, bias)); Z += u; N = fmaf(u, v3, N); }
    if (W > 4) { u = ex2(fmaf(-c2, D4, bias)); Z += u; N = fmaf(u, v4, N); }
    return make_float3(Z, N, bias);
}

// One pass: W consecutive x-offsets (tx = txs .. txs+W-1) at fixed (ty, tz), marching RZ+2 planes.
//   aRow: &A[plane 0][row lane][x0]          (word k  <-> x = x0 - 1 + k)
//   bRow: &B[plane 0 + tz][row lane + ty][x0 + BOFF]   (word k' <-> x = x0 - 1 + txs + k' - QOFF ... see QOFF)
// QOFF: index of the word that pairs with a[0] for the first offset of the chunk.
template <int RZ, int W, int QOFF, int NB4, int A_PLANE, int B_PLANE>
__device__ __forceinline__ void tiled_pass(const float *__restrict__ aRow, const float *__restrict__ bRow,
                                           const float c2, Acc4 (&acc)[RZ])
{
    float ring0[W][4], ring1[W][4];
    float bprev[4 * NB4];
#pragma unroll
    for (int p = 0; p < RZ + 2; ++p) {
        float a[8], b[4 * NB4];
        {
            const float4 a0 = *reinterpret_cast<const float4 *>(aRow + p * A_PLANE);
            const float4 a1 = *reinterpret_cast<const float4 *>(aRow + p * A_PLANE + 4);
            a[0] = a0.x; a[1] = a0.y; a[2] = a0.z; a[3] = a0.w; a[4] = a1.x; a[5] = a1.y; a[6] = a1.z; a[7] = a1.w;
#pragma unroll
            for (int v = 0; v < NB4; ++v) {
                const float4 bv = *reinterpret_cast<const float4 *>(bRow + p * B_PLANE + 4 * v);
                b[4 * v] = bv.x; b[4 * v + 1] = bv.y; b[4 * v + 2] = bv.z; b[4 * v + 3] = bv.w;
            }
        }
        float Y[W][4];
#pragma unroll
        for (int q = 0; q < W; ++q) {
            // a1 + a2x: squared differences, 3-tap x-sum; outputs (0,1) share d1^2+d2^2, (2,3) share d3^2+d4^2
            const float d0 = a[0] - b[0 + q + QOFF], d1 = a[1] - b[1 + q + QOFF], d2 = a[2] - b[2 + q + QOFF];
            const float d3 = a[3] - b[3 + q + QOFF], d4 = a[4] - b[4 + q + QOFF], d5 = a[5] - b[5 + q + QOFF];
            const float c12 = fmaf(d2, d2, d1 * d1);
            const float c34 = fmaf(d4, d4, d3 * d3);
            float X[4];
            X[0] = fmaf(d0, d0, c12);
            X[1] = fmaf(d3, d3, c12);
            X[2] = fmaf(d2, d2, c34);
            X[3] = fmaf(d5, d5, c34);
            // a2y: rows are lanes
#pragma unroll
            for (int i = 0; i < 4; ++i)
                Y[q][i] = X[i] + __shfl_up_sync(0xffffffffu, X[i], 1) + __shfl_down_sync(0xffffffffu, X[i], 1);
        }
        if (p >= 2) {
            Acc4 &ac = acc[p - 2];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                float D[W], zp = 0.f, np = 0.f;
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    D[q] = ring0[q][i] + ring1[q][i] + Y[q][i];                    // a2z
                    const float u = ex2(fmaf(-c2, D[q], ac.b[i]));                 // a3
                    zp += u;                                                       // a4
                    np = fmaf(u, bprev[i + q + QOFF + 1], np);
                }
                if (zp <= kGuard) {
                    ac.z[i] += zp;
                    ac.n[i] += np;
                } else {   // a term left the guard band (or first use, bias = +inf): cold path
                    const float3 r = rebase_and_add<W>(
                        ac.z[i], ac.n[i], ac.b[i], c2, D[0], D[W > 1 ? 1 : 0], D[W > 2 ? 2 : 0], D[W > 3 ? 3 : 0],
                        D[W > 4 ? 4 : 0], bprev[i + 0 + QOFF + 1], bprev[i + (W > 1 ? 1 : 0) + QOFF + 1],
                        bprev[i + (W > 2 ? 2 : 0) + QOFF + 1], bprev[i + (W > 3 ? 3 : 0) + QOFF + 1],
                        bprev[i + (W > 4 ? 4 : 0) + QOFF + 1]);
                    ac.z[i] = r.x; ac.n[i] = r.y; ac.b[i] = r.z;
                }
            }
        }
#pragma unroll
        for (int q = 0; q < W; ++q)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                ring0[q][i] = ring1[q][i];
                ring1[q][i] = Y[q][i];
            }
#pragma unroll
        for (int k = 0; k < 4 * NB4; ++k) bprev[k] = b[k];
    }
}

// All x-offsets of one (ty, tz): split into aligned chunks of at most 5 offsets.
template <int M, int RZ>
__device__ __forceinline__ void tiled_row_of_offsets(const float *aRow, const float *bRow, float c2, Acc4 (&acc)[RZ])
{
    using G = TiledGeom<M>;
    using S = TiledSmem<M, RZ>;
    constexpr int AP = G::RA * G::PA, BP = G::RB * G::PB;
    (void)sizeof(S);
    // word 0 of bRow <-> x = x0 - HXB; a[0] <-> x = x0 - 1; offset tx pairs a[k] with x0 - 1 + k + tx
    if constexpr (M == 1) {          // tx -1..1 : b index = k + tx + 3 = k + q + 2
        tiled_pass<RZ, 3, 2, 3, AP, BP>(aRow, bRow, c2, acc);
    } else if constexpr (M == 2) {   // tx -2..2 : k + q + 1
        tiled_pass<RZ, 5, 1, 3, AP, BP>(aRow, bRow, c2, acc);
    } else if constexpr (M == 3) {   // tx -3..0 : k + q + 0 (12 words) ; tx 1..3 from word 4: k + q + 0 (8 words)
        tiled_pass<RZ, 4, 0, 3, AP, BP>(aRow, bRow, c2, acc);
        tiled_pass<RZ, 3, 0, 2, AP, BP>(aRow, bRow + 4, c2, acc);
    } else {                         // M == 4, HXB = 8: tx -4..-1 : k + q + 3 (12 words) ; tx 0..4 from word 4: k + q + 3 (16 words)
        tiled_pass<RZ, 4, 3, 3, AP, BP>(aRow, bRow, c2, acc);
        tiled_pass<RZ, 5, 3, 4, AP, BP>(aRow, bRow + 4, c2, acc);
    }
}

template <int M, int RZ>
__global__ void __launch_bounds__(32 * kTiledWarps, 1)
tnlm_tiled_kernel(const float *__restrict__ f, const float *__restrict__ g, float *__restrict__ f_out, const Dims dm,
                  const int tiles_x, const int tiles_y, const int tiles_z)
{
    using G = TiledGeom<M>;
    using S = TiledSmem<M, RZ>;
    extern __shared__ __align__(16) float smem[];
    float *sA = smem;
    float *sB = smem + S::A_WORDS;

    int t = blockIdx.x;
    const int bx = t % tiles_x; t /= tiles_x;
    const int by = t % tiles_y; t /= tiles_y;
    const int bz = t % tiles_z; t /= tiles_z;
    const int ph = t;
    const int X0 = bx * kTiledTX, Y0 = by * kTiledRowsOut, Z0 = dm.z_begin + bz * RZ;
    const size_t V = (size_t)dm.Z * dm.Y * dm.X;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int x0 = 4 * warp;

    // ---- stage the ref_i tile (halo 1): A[pz][r][c] <-> (Z0-1+pz, Y0-1+r, X0-1+c), clamped
    {
        const float *src = f + (size_t)ph * V;
        for (int idx = tid; idx < S::A_WORDS; idx += 32 * kTiledWarps) {
            const int c = idx % G::PA, r = (idx / G::PA) % G::RA, pz = idx / (G::PA * G::RA);
            const int z = clampi(Z0 - 1 + pz, dm.Z), y = clampi(Y0 - 1 + r, dm.Y), x = clampi(X0 - 1 + c, dm.X);
            sA[idx] = __ldg(src + ((size_t)z * dm.Y + y) * dm.X + x);
        }
    }

#pragma unroll 1
    for (int s = 0; s < 2; ++s) {
        const int j = (ph + (s ? 1 : dm.P - 1)) % dm.P;
        __syncthreads();   // everyone is done with the previous B tile
        // ---- stage the f_j tile (halo 1+M): B[pz][r][c] <-> (Z0-1-M+pz, Y0-1-M+r, X0-HXB+c), clamped
        {
            const float *src = f + (size_t)j * V;
            for (int idx = tid; idx < S::B_WORDS; idx += 32 * kTiledWarps) {
                const int c = idx % G::PB, r = (idx / G::PB) % G::RB, pz = idx / (G::PB * G::RB);
                const int z = clampi(Z0 - 1 - M + pz, dm.Z), y = clampi(Y0 - 1 - M + r, dm.Y),
                          x = clampi(X0 - G::HXB + c, dm.X);
                sB[idx] = __ldg(src + ((size_t)z * dm.Y + y) * dm.X + x);
            }
        }
        __syncthreads();

        Acc4 acc[RZ];
#pragma unroll
        for (int o = 0; o < RZ; ++o)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                acc[o].z[i] = 0.f;
                acc[o].n[i] = 0.f;
                acc[o].b[i] = INFINITY;
            }

        const float *aRow = sA + lane * G::PA + x0;
        constexpr int E = 2 * M + 1;
#pragma unroll 1
        for (int k = 0; k < E * E; ++k) {
            // start with (ty, tz) = (0, 0): the zero offset is usually the best match, so the
            // reference exponent is set once and the cold path stays cold
            const int kk = (k + (E * E) / 2) % (E * E);
            const int tz = kk / E, ty = kk % E;   // 0 .. 2M  (offset + M)
            const float *bRow = sB + (tz * G::RB + (lane + ty)) * G::PB + x0;
            tiled_row_of_offsets<M, RZ>(aRow, bRow, dm.c2, acc);
        }

        // ---- a5: Jacobi combine (Eq. 8).  Direction 0 writes mu/(2+mu) g + NLM-/(2+mu); direction 1
        // adds NLM+/(2+mu) to the value this same thread wrote (no other thread touches the voxel).
        const int y = Y0 - 1 + lane;
        const bool row_ok = (lane >= 1) && (lane <= kTiledRowsOut) && (y < dm.Y);
#pragma unroll
        for (int o = 0; o < RZ; ++o) {
            const int z = Z0 + o;
            if (row_ok && z < dm.z_end) {
                const size_t base = (size_t)ph * V + ((size_t)z * dm.Y + y) * dm.X + X0 + x0;
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (X0 + x0 + i < dm.X) {
                        const float nlm = __fdividef(acc[o].n[i], acc[o].z[i]);
                        if (s == 0)
                            f_out[base + i] = fmaf(dm.a_g, __ldg(g + base + i), dm.a_n * nlm);
                        else
                            f_out[base + i] = fmaf(dm.a_n, nlm, f_out[base + i]);
                    }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
constexpr int kTiledRZ = 8;

inline bool tiled_supported(const tnlm_params &p)
{
    return p.patch_radius == 1 && p.search_radius >= 1 && p.search_radius <= 4;
}
inline size_t tiled_scratch_bytes(const tnlm_params &) { return 0; }
inline const char *tiled_name(const tnlm_params &p)
{
    switch (p.search_radius) {
        case 1: return "tnlm_tiled_kernel<M=1,RZ=8>";
        case 2: return "tnlm_tiled_kernel<M=2,RZ=8>";
        case 3: return "tnlm_tiled_kernel<M=3,RZ=8>";
        default: return "tnlm_tiled_kernel<M=4,RZ=8>";
    }
}
inline int tiled_launches_per_sweep(const tnlm_params &) { return 1; }

template <int M, int RZ>
cudaError_t launch_tiled_t(const Dims &dm, const float *f, const float *g, float *f_out, cudaStream_t st)
{
    using S = TiledSmem<M, RZ>;
    static bool configured = false;   // per template instance; attribute is per-device-function, idempotent
    cudaError_t e;
    if (!configured) {
        e = cudaFuncSetAttribute(tnlm_tiled_kernel<M, RZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::BYTES);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    const int tiles_x = (dm.X + kTiledTX - 1) / kTiledTX;
    const int tiles_y = (dm.Y + kTiledRowsOut - 1) / kTiledRowsOut;
    const int tiles_z = (dm.z_end - dm.z_begin + RZ - 1) / RZ;
    const long long blocks = (long long)tiles_x * tiles_y * tiles_z * dm.P;
    if (blocks <= 0 || blocks > 2147483647LL) return cudaErrorInvalidConfiguration;
    tnlm_tiled_kernel<M, RZ><<<(unsigned)blocks, 32 * kTiledWarps, S::BYTES, st>>>(f, g, f_out, dm, tiles_x, tiles_y,
                                                                                  tiles_z);
    return cudaGetLastError();
}

inline int tiled_rz()
{
    static int rz = [] {
        const char *e = getenv("TNLM_TILED_RZ");   // tuning knob for experiments; default = kTiledRZ
        const int v = e ? atoi(e) : kTiledRZ;
        return (v == 4 || v == 6 || v == 8) ? v : kTiledRZ;
    }();
    return rz;
}

template <int M>
cudaError_t launch_tiled_m(const Dims &dm, const float *f, const float *g, float *f_out, cudaStream_t st)
{
    switch (tiled_rz()) {
        case 4: return launch_tiled_t<M, 4>(dm, f, g, f_out, st);
        case 6: return launch_tiled_t<M, 6>(dm, f, g, f_out, st);
        default: return launch_tiled_t<M, 8>(dm, f, g, f_out, st);
    }
}

// ref must be f (TNLM-E); the caller falls back to the generic kernel otherwise.
inline cudaError_t launch_tiled(const tnlm_params &p, const Dims &dm, const float *f, const float *g, const float *ref,
                                float *f_out, void *, size_t, cudaStream_t st)
{
    if (ref != f) return cudaErrorNotSupported;
    switch (p.search_radius) {
        case 1: return launch_tiled_m<1>(dm, f, g, f_out, st);
        case 2: return launch_tiled_m<2>(dm, f, g, f_out, st);
        case 3: return launch_tiled_m<3>(dm, f, g, f_out, st);
        case 4: return launch_tiled_m<4>(dm, f, g, f_out, st);
        default: return cudaErrorNotSupported;
    }
}

}  // namespace tnlm
