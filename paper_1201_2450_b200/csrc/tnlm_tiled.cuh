// Tiled sm_100a TNLM sweep kernel for 3^3 patches (d = 1), search radius M in {1,2,3,4}.
//
// One CTA = one (phase i, 32-wide x-tile, 30-row y-group, RZ-plane z-slab) and both neighbour
// phases j = i-1, i+1 (Eq. 8).  The CTA stages a halo tile of ref_i (halo d) and of
// ref_j = f_j (halo d+M; clamp-to-edge applied while staging: reading P4) in shared memory, then
// every warp runs without any block-level synchronisation until the tile is done:
//
//   lane        = one y-row (32 rows per warp; rows 0 and 31 are the d-halo: 30 output rows)
//   thread      = an x-run of XR voxels x 1 row x a column of RZ output planes
//   registers   = the accumulators (Z, N, reference exponent) of its XR*RZ outputs for the whole
//                 search window; nothing per-offset ever leaves the register file
//   per (ty,tz) = a "pass": march the RZ+2 planes of the slab; per plane
//       a1  diffs ref_i - ref_j(+t) for up to 5 consecutive tx at once, from one vector-loaded row window
//       a2x 3-tap x-sum of squares in registers; neighbouring outputs share the middle pair
//       a2y 3-tap y-sum through two warp shuffles (lanes are rows)
//       a2z 3-tap z-sum from a two-plane register ring
//       a3  u = ex2(bias - c2*D): one FFMA + one MUFU (bias = lazily maintained reference exponent)
//       a4  Z += u, N += u * f_j(x+t)   (the candidate value is the centre of the row window, in registers)
//   epilogue    = a5: f_out = mu/(2+mu) g + (N-/Z- + N+/Z+)/(2+mu)
//
// Reference exponent (reading P3: weights relative to the best candidate): a pass adds its terms
// optimistically and checks its partial normaliser; only if a term left the 2^60 guard band (or on
// first use, bias = +inf) is the output re-based on the best candidate of the pass (cold path).
// The result equals the shifted softmax up to rounding.
#pragma once
#include <cstdlib>

#include "tnlm_common.cuh"

namespace tnlm {

constexpr int kTiledTX = 32;                   // x extent of a CTA tile
constexpr int kTiledRowsOut = 30;              // output rows per CTA (32 lanes - 2 halo rows)
constexpr float kGuard = 1.152921504606847e18f;   // 2^60

__host__ __device__ constexpr int round_up_pitch(int min_words, int v)   // smallest p >= min_words with p = v * odd
{
    int p = (min_words + v - 1) / v * v;
    return ((p / v) % 2 == 1) ? p : p + v;
}
__host__ __device__ constexpr int cdiv(int a, int b) { return (a + b - 1) / b; }
__host__ __device__ constexpr int cmax(int a, int b) { return a > b ? a : b; }

// Offsets tx = -M..M are processed in chunks of at most 5 whose first word is vector aligned.
template <int M> struct Chunks {
    static constexpr int W0 = (2 * M + 1 <= 5) ? 2 * M + 1 : 4;   // first chunk
    static constexpr int W1 = 2 * M + 1 - W0;                     // second chunk (0 if none), starts at word 4
};

template <int M, int XR> struct TiledGeom {
    using C = Chunks<M>;
    static constexpr int NW = kTiledTX / XR;                       // warps per CTA, one x-run each
    static constexpr int NT = 32 * NW;
    static constexpr int HXB = M + 1;                              // B col c <-> x = X0 - HXB + c
    static constexpr int AV = cdiv(XR + 2, XR);                    // vectors of an A row window
    static constexpr int BV0 = cdiv(XR + C::W0 + 1, XR);           // vectors of chunk 0's B row window
    static constexpr int BV1 = C::W1 ? cdiv(XR + C::W1 + 1, XR) : 0;
    static constexpr int BWORDS = cmax(BV0 * XR, C::W1 ? 4 + BV1 * XR : 0);
    static constexpr int PA = round_up_pitch(kTiledTX - XR + AV * XR, XR);   // conflict-free vector LDS (lanes = rows)
    static constexpr int PB = round_up_pitch(kTiledTX - XR + BWORDS, XR);
    static constexpr int RA = 32;                                  // A rows
    static constexpr int RB = 32 + 2 * M;                          // B rows
};

template <int M, int XR, int RZ> struct TiledSmem {
    using G = TiledGeom<M, XR>;
    static constexpr int NA = RZ + 2, NB = RZ + 2 + 2 * M;
    static constexpr int A_WORDS = NA * G::RA * G::PA;
    static constexpr int B_WORDS = NB * G::RB * G::PB;
    static constexpr int STASH_WORDS = RZ * XR * G::NT;            // NLM of the first direction
    static constexpr size_t BYTES = (size_t)(A_WORDS + B_WORDS + STASH_WORDS) * sizeof(float);
};

template <int XR> struct AccRun { float z[XR], n[XR], b[XR]; };   // normaliser, weighted sum, reference exponent

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

template <int XR, int NV>
__device__ __forceinline__ void load_row(const float *__restrict__ p, float (&dst)[NV * XR])
{
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        if constexpr (XR == 4) {
            const float4 t = *reinterpret_cast<const float4 *>(p + 4 * v);
            dst[4 * v] = t.x; dst[4 * v + 1] = t.y; dst[4 * v + 2] = t.z; dst[4 * v + 3] = t.w;
        } else {
            const float2 t = *reinterpret_cast<const float2 *>(p + 2 * v);
            dst[2 * v] = t.x; dst[2 * v + 1] = t.y;
        }
    }
}

// One pass: W consecutive x-offsets at fixed (ty, tz), marching the RZ+2 planes.
//   aRow: &A[plane 0][row lane][x0]              word k <-> x = x0 - 1 + k
//   bRow: &B[plane tz][row lane + ty][x0 + c0]   word k + q pairs with a[k] for the q-th offset of the chunk
template <int XR, int RZ, int W, int A_PLANE, int B_PLANE>
__device__ __forceinline__ void tiled_pass(const float *__restrict__ aRow, const float *__restrict__ bRow,
                                           const float c2, AccRun<XR> (&acc)[RZ])
{
    constexpr int AV = cdiv(XR + 2, XR), BV = cdiv(XR + W + 1, XR);
    float ring0[W][XR], ring1[W][XR];
    float bprev[BV * XR];
#pragma unroll
    for (int p = 0; p < RZ + 2; ++p) {
        float a[AV * XR], b[BV * XR];
        load_row<XR, AV>(aRow + p * A_PLANE, a);
        load_row<XR, BV>(bRow + p * B_PLANE, b);
        float Y[W][XR];
#pragma unroll
        for (int q = 0; q < W; ++q) {
            float d[XR + 2], X[XR];
#pragma unroll
            for (int k = 0; k < XR + 2; ++k) d[k] = a[k] - b[k + q];                       // a1
#pragma unroll
            for (int i = 0; i < XR; i += 2) {                                              // a2x
                const float mid = fmaf(d[i + 2], d[i + 2], d[i + 1] * d[i + 1]);
                X[i] = fmaf(d[i], d[i], mid);
                X[i + 1] = fmaf(d[i + 3], d[i + 3], mid);
            }
#pragma unroll
            for (int i = 0; i < XR; ++i)                                                   // a2y: rows are lanes
                Y[q][i] = X[i] + __shfl_up_sync(0xffffffffu, X[i], 1) + __shfl_down_sync(0xffffffffu, X[i], 1);
        }
        if (p >= 2) {
            AccRun<XR> &ac = acc[p - 2];
#pragma unroll
            for (int i0 = 0; i0 < XR; i0 += 2) {   // two outputs per guard check
                float D[2][W], zp[2], np[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int i = i0 + e;
                    zp[e] = 0.f;
                    np[e] = 0.f;
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        D[e][q] = ring0[q][i] + ring1[q][i] + Y[q][i];                     // a2z
                        const float u = ex2(fmaf(-c2, D[e][q], ac.b[i]));                  // a3
                        zp[e] += u;                                                        // a4
                        np[e] = fmaf(u, bprev[i + 1 + q], np[e]);
                    }
                }
                if (fmaxf(zp[0], zp[1]) <= kGuard) {
                    ac.z[i0] += zp[0]; ac.n[i0] += np[0];
                    ac.z[i0 + 1] += zp[1]; ac.n[i0 + 1] += np[1];
                } else {   // a term left the guard band (or first use, bias = +inf): cold path
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int i = i0 + e;
                        if (zp[e] <= kGuard) {
                            ac.z[i] += zp[e];
                            ac.n[i] += np[e];
                        } else {
                            const float3 r = rebase_and_add<W>(
                                ac.z[i], ac.n[i], ac.b[i], c2, D[e][0], D[e][W > 1 ? 1 : 0], D[e][W > 2 ? 2 : 0],
                                D[e][W > 3 ? 3 : 0], D[e][W > 4 ? 4 : 0], bprev[i + 1], bprev[i + 1 + (W > 1 ? 1 : 0)],
                                bprev[i + 1 + (W > 2 ? 2 : 0)], bprev[i + 1 + (W > 3 ? 3 : 0)],
                                bprev[i + 1 + (W > 4 ? 4 : 0)]);
                            ac.z[i] = r.x; ac.n[i] = r.y; ac.b[i] = r.z;
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int q = 0; q < W; ++q)
#pragma unroll
            for (int i = 0; i < XR; ++i) {
                ring0[q][i] = ring1[q][i];
                ring1[q][i] = Y[q][i];
            }
#pragma unroll
        for (int k = 0; k < BV * XR; ++k) bprev[k] = b[k];
    }
}

// Stage a clamped halo tile: dst[pz][r][c] <- src(clamp(zo+pz), clamp(yo+r), clamp(xo+c)); 8 loads in flight.
template <int PITCH, int ROWS, int WORDS, int NT>
__device__ __forceinline__ void stage_tile(float *__restrict__ dst, const float *__restrict__ src, const int zo,
                                           const int yo, const int xo, const Dims &dm, const int tid)
{
    constexpr int U = 8;
#pragma unroll 1
    for (int base = tid; base < WORDS; base += NT * U) {
        float v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int idx = base + u * NT;
            if (idx < WORDS) {
                const int c = idx % PITCH, r = (idx / PITCH) % ROWS, pz = idx / (PITCH * ROWS);
                const int z = clampi(zo + pz, dm.Z), y = clampi(yo + r, dm.Y), x = clampi(xo + c, dm.X);
                v[u] = __ldg(src + ((size_t)z * dm.Y + y) * dm.X + x);
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int idx = base + u * NT;
            if (idx < WORDS) dst[idx] = v[u];
        }
    }
}

template <int M, int XR, int RZ>
__global__ void __launch_bounds__(TiledGeom<M, XR>::NT, 1)
tnlm_tiled_kernel(const float *__restrict__ f, const float *__restrict__ g, float *__restrict__ f_out, const Dims dm,
                  const int tiles_x, const int tiles_y, const int tiles_z)
{
    using G = TiledGeom<M, XR>;
    using S = TiledSmem<M, XR, RZ>;
    using C = Chunks<M>;
    constexpr int AP = G::RA * G::PA, BP = G::RB * G::PB;
    extern __shared__ __align__(16) float smem[];
    float *sA = smem;
    float *sB = smem + S::A_WORDS;
    float *sStash = sB + S::B_WORDS;

    int t = blockIdx.x;
    const int bx = t % tiles_x; t /= tiles_x;
    const int by = t % tiles_y; t /= tiles_y;
    const int bz = t % tiles_z; t /= tiles_z;
    const int ph = t;
    const int X0 = bx * kTiledTX, Y0 = by * kTiledRowsOut, Z0 = dm.z_begin + bz * RZ;
    const size_t V = (size_t)dm.Z * dm.Y * dm.X;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int x0 = XR * warp;

    // ref_i tile (halo 1): A[pz][r][c] <-> (Z0-1+pz, Y0-1+r, X0-1+c)
    stage_tile<G::PA, G::RA, S::A_WORDS, G::NT>(sA, f + (size_t)ph * V, Z0 - 1, Y0 - 1, X0 - 1, dm, tid);

#pragma unroll 1
    for (int s = 0; s < 2; ++s) {
        const int j = (ph + (s ? 1 : dm.P - 1)) % dm.P;
        __syncthreads();   // everyone is done with the previous B tile
        // f_j tile (halo 1+M): B[pz][r][c] <-> (Z0-1-M+pz, Y0-1-M+r, X0-1-M+c)
        stage_tile<G::PB, G::RB, S::B_WORDS, G::NT>(sB, f + (size_t)j * V, Z0 - 1 - M, Y0 - 1 - M, X0 - G::HXB, dm, tid);
        __syncthreads();

        AccRun<XR> acc[RZ];
#pragma unroll
        for (int o = 0; o < RZ; ++o)
#pragma unroll
            for (int i = 0; i < XR; ++i) {
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
            const int tz = kk / E, ty = kk % E;   // offset + M
            const float *bRow = sB + (tz * G::RB + (lane + ty)) * G::PB + x0;
            tiled_pass<XR, RZ, C::W0, AP, BP>(aRow, bRow, dm.c2, acc);
            if constexpr (C::W1 > 0) tiled_pass<XR, RZ, C::W1, AP, BP>(aRow, bRow + 4, dm.c2, acc);
        }

        if (s == 0) {
            // park NLM- of this thread's outputs (own slots, lanes consecutive: conflict-free)
#pragma unroll
            for (int o = 0; o < RZ; ++o)
#pragma unroll
                for (int i = 0; i < XR; ++i)
                    sStash[(o * XR + i) * G::NT + tid] = __fdividef(acc[o].n[i], acc[o].z[i]);
        } else {
            // a5: Jacobi combine (Eq. 8)
            const int y = Y0 - 1 + lane;
            const bool row_ok = (lane >= 1) && (lane <= kTiledRowsOut) && (y < dm.Y);
            const bool vec_ok = (dm.X % XR) == 0;   // then every run start is vector aligned and fully inside
            if (row_ok && X0 + x0 < dm.X) {
                float gv[RZ][XR];
                const size_t base0 = (size_t)ph * V + ((size_t)Z0 * dm.Y + y) * dm.X + X0 + x0;
                const size_t zstride = (size_t)dm.Y * dm.X;
#pragma unroll
                for (int o = 0; o < RZ; ++o) {
                    if (Z0 + o < dm.z_end) {
                        if (vec_ok) {
                            if constexpr (XR == 4) {
                                const float4 tv = __ldg(reinterpret_cast<const float4 *>(g + base0 + o * zstride));
                                gv[o][0] = tv.x; gv[o][1] = tv.y; gv[o][2] = tv.z; gv[o][3] = tv.w;
                            } else {
                                const float2 tv = __ldg(reinterpret_cast<const float2 *>(g + base0 + o * zstride));
                                gv[o][0] = tv.x; gv[o][1] = tv.y;
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < XR; ++i)
                                gv[o][i] = (X0 + x0 + i < dm.X) ? __ldg(g + base0 + o * zstride + i) : 0.f;
                        }
                    }
                }
#pragma unroll
                for (int o = 0; o < RZ; ++o) {
                    if (Z0 + o < dm.z_end) {
                        float r[XR];
#pragma unroll
                        for (int i = 0; i < XR; ++i) {
                            const float nlm = sStash[(o * XR + i) * G::NT + tid] + __fdividef(acc[o].n[i], acc[o].z[i]);
                            r[i] = fmaf(dm.a_g, gv[o][i], dm.a_n * nlm);
                        }
                        float *dst = f_out + base0 + o * zstride;
                        if (vec_ok) {
                            if constexpr (XR == 4)
                                *reinterpret_cast<float4 *>(dst) = make_float4(r[0], r[1], r[2], r[3]);
                            else
                                *reinterpret_cast<float2 *>(dst) = make_float2(r[0], r[1]);
                        } else {
#pragma unroll
                            for (int i = 0; i < XR; ++i)
                                if (X0 + x0 + i < dm.X) dst[i] = r[i];
                        }
                    }
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
constexpr int kTiledRZ = 8;
constexpr int kTiledXR = 2;

inline bool tiled_supported(const tnlm_params &p)
{
    return p.patch_radius == 1 && p.search_radius >= 1 && p.search_radius <= 4;
}
inline size_t tiled_scratch_bytes(const tnlm_params &) { return 0; }
inline const char *tiled_name(const tnlm_params &p)
{
    switch (p.search_radius) {
        case 1: return "tnlm_tiled_kernel<M=1>";
        case 2: return "tnlm_tiled_kernel<M=2>";
        case 3: return "tnlm_tiled_kernel<M=3>";
        default: return "tnlm_tiled_kernel<M=4>";
    }
}
inline int tiled_launches_per_sweep(const tnlm_params &) { return 1; }

template <int M, int XR, int RZ>
cudaError_t launch_tiled_t(const Dims &dm, const float *f, const float *g, float *f_out, cudaStream_t st)
{
    using S = TiledSmem<M, XR, RZ>;
    using G = TiledGeom<M, XR>;
    static std::atomic<uint64_t> configured{0};   // per template instance: one bit per device
    cudaError_t e = ensure_dynamic_smem(tnlm_tiled_kernel<M, XR, RZ>, S::BYTES, configured);
    if (e != cudaSuccess) return e;
    const int tiles_x = (dm.X + kTiledTX - 1) / kTiledTX;
    const int tiles_y = (dm.Y + kTiledRowsOut - 1) / kTiledRowsOut;
    const int tiles_z = (dm.z_end - dm.z_begin + RZ - 1) / RZ;
    const long long blocks = (long long)tiles_x * tiles_y * tiles_z * dm.P;
    if (blocks <= 0 || blocks > 2147483647LL) return cudaErrorInvalidConfiguration;
    tnlm_tiled_kernel<M, XR, RZ><<<(unsigned)blocks, G::NT, S::BYTES, st>>>(f, g, f_out, dm, tiles_x, tiles_y, tiles_z);
    return cudaGetLastError();
}

template <int M>
cudaError_t launch_tiled_m(const Dims &dm, const float *f, const float *g, float *f_out, cudaStream_t st)
{
    return launch_tiled_t<M, kTiledXR, kTiledRZ>(dm, f, g, f_out, st);
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
