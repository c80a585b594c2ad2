// Row-pair packed sm_100a TNLM sweep kernel for 5^3 patches (d = 2), search radius M in {1,2,3,4}.
//
// Same design as tnlm_pair.cuh (read its header first): float2 = the same quantity for tile rows 2l and
// 2l+1, packed FADD2 / FMUL2 / FFMA2 arithmetic, even/odd row-pair copies of the neighbour phase in
// shared memory, accumulators and reference exponents in registers, hot/careful pass forms.  What a
// 5^3 patch (PAPER.md:105, :221 with d = 2) changes:
//   tile halo    2 (A) and 2+M (B); half-warp = 32 tile rows = 28 output rows (tile rows 2..29)
//   a1/a2x       6 differences per x-run of 2 outputs; the two 5-tap x-sums share their 4 middle squares
//   a2z          5-tap z-sum from a four-plane register ring; the candidate plane is two planes back
//   a2y          own two rows + two rows from the lane above + two from the lane below: 4 SHFL per pair
//   x-offsets    chunks of W = 2 (the last one 3) so that the four-plane ring fits in registers
#pragma once
#include "tnlm_pair.cuh"

namespace tnlm {

constexpr int kPair5RowsOut = 28;

// chunk c of the 2M+1 x-offsets: starts at q0 = 2c; width 2, the last chunk (c = M-1) 3
__host__ __device__ constexpr int chunk5_w(int M, int c) { return c == M - 1 ? 3 : 2; }

template <int M, int RZ, int TX, bool SEP = false> struct Pair5Geom {
    static constexpr int E = 2 * M + 1;
    static constexpr int NRUN = TX / 2, NT = NRUN * 16;
    static constexpr int ACOLS = TX + 4, BCOLS = TX + 2 * M + 4;      // staged columns
    // columns a B window may touch: x0_max + q0_max + 2 * NVB(3) with NVB(W) = (W + 6) / 2
    static constexpr int BREAD = TX - 2 + 2 * (M - 1) + 8;
    static constexpr int PA2 = pitch2(cmax(ACOLS, TX - 2 + 6));
    static constexpr int PB2 = pitch2(cmax(BCOLS, BREAD));
    static constexpr int NPA = 16, NPE = 16 + M, NPO = 15 + M, NPB = NPE + NPO;
    static constexpr int NAP = RZ + 4, NBP = RZ + 4 + 2 * M;
    static constexpr int NFP = SEP ? RZ + 2 * M : 0;                  // candidate tile F (ref != f): B planes 2 .. NBP-3
    static constexpr int A_F2 = NAP * NPA * PA2, B_F2 = NBP * NPB * PB2, F_F2 = NFP * NPB * PB2;
    static constexpr size_t BYTES = (size_t)(A_F2 + B_F2 + F_F2) * sizeof(float2);
};

// One pass of the 5^3-patch kernel: W consecutive x-offsets at fixed (ty, tz), marching the RZ+4 planes.
//   aRow: &A2[plane 0][pair l][x0]                 element k <-> x = X0 + x0 - 2 + k   (negated values)
//   bRow: &B?[plane tz][pair l + ty/2][x0 + q0]    element k + q pairs with a[k] for the q-th offset of the chunk
//   fRow (SEP only): &F?[plane tz][pair l + ty/2][x0 + q0], F plane k <-> B plane k + 2
// CAREFUL and SEP as in pair_pass (tnlm_pair.cuh).
template <int RZ, int W, bool CAREFUL, int A_PLANE, int B_PLANE, bool SEP = false>
__device__ __forceinline__ unsigned pair5_pass(const float2 *__restrict__ aRow, const float2 *__restrict__ bRow,
                                               const float2 *__restrict__ fRow, const float c2, AccPair (&acc)[RZ],
                                               const unsigned mask)
{
    constexpr int NVB = (W + 6) / 2;   // 6 + W - 1 positions
    const float2 nc2 = make_float2(-c2, -c2);
    float2 ring[4][W][2];              // x-summed planes p-4 .. p-1
    float2 cand1[W + 1], cand2[W + 1]; // candidate values f_j(x+t) of planes p-1 and p-2: elements 2 .. W+2 of b
    unsigned fail = 0u;
#pragma unroll
    for (int p = 0; p < RZ + 4; ++p) {
        float2 a[6], b[2 * NVB];
        load_pairs<3>(aRow + p * A_PLANE, a);
        load_pairs<NVB>(bRow + p * B_PLANE, b);
        float2 X[W][2];
#pragma unroll
        for (int q = 0; q < W; ++q) {
            float2 d[6];
#pragma unroll
            for (int k = 0; k < 6; ++k) d[k] = add2(b[k + q], a[k]);                      // a1 (a is -ref_i)
            float2 mid = mul2(d[1], d[1]);                                                // a2x
            mid = fma2(d[2], d[2], mid);
            mid = fma2(d[3], d[3], mid);
            mid = fma2(d[4], d[4], mid);
            X[q][0] = fma2(d[0], d[0], mid);
            X[q][1] = fma2(d[5], d[5], mid);
        }
        if (p >= 4) {
            AccPair &ac = acc[p - 4];
            if (SEP) {   // candidates f_j(x+t) of the centre plane: window elements 2 .. W+2
                float2 fw[2 * NVB];
                load_pairs<NVB>(fRow + (p - 4) * B_PLANE, fw);
#pragma unroll
                for (int k = 0; k < W + 1; ++k) cand2[k] = fw[k + 2];
            }
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                float2 D[W];
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    const float2 S = add2(add2(add2(ring[0][q][i], ring[1][q][i]), add2(ring[2][q][i], ring[3][q][i])),
                                          X[q][i]);                                       // a2z
                    const float u0 = __shfl_up_sync(0xffffffffu, S.x, 1);                 // row 2l-2
                    const float u1 = __shfl_up_sync(0xffffffffu, S.y, 1);                 // row 2l-1
                    const float d0 = __shfl_down_sync(0xffffffffu, S.x, 1);               // row 2l+2
                    const float d1 = __shfl_down_sync(0xffffffffu, S.y, 1);               // row 2l+3
                    const float common = (S.x + S.y) + (u1 + d0);                         // a2y
                    D[q] = add2(make_float2(u0, d1), make_float2(common, common));
                }
                if (!CAREFUL) {
                    // hot form: optimistic partial sums relative to the reference exponents, one guard per row pair
                    float2 zp = make_float2(0.f, 0.f), np = make_float2(0.f, 0.f);
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        const float2 arg = fma2(D[q], nc2, ac.b[i]);                      // a3
                        const float2 u = make_float2(ex2(arg.x), ex2(arg.y));
                        zp = add2(zp, u);                                                 // a4
                        np = fma2(u, cand2[i + q], np);
                    }
                    if (fmaxf(zp.x, zp.y) <= kPairGuard) {
                        ac.z[i] = add2(ac.z[i], zp);
                        ac.n[i] = add2(ac.n[i], np);
                    } else {
                        fail |= 1u << (2 * (p - 4) + i);
                    }
                } else if ((mask >> (2 * (p - 4) + i)) & 1u) {
                    // careful form, straight-line: a row is re-based iff its best candidate of this chunk beats its
                    // reference by more than 2^97 (then the W terms could pass 2^100; on first use the reference is
                    // +inf); otherwise it keeps its reference (scale factor 1) and its terms are simply added
                    float2 dmin = D[0];
#pragma unroll
                    for (int q = 1; q < W; ++q) dmin = make_float2(fminf(dmin.x, D[q].x), fminf(dmin.y, D[q].y));
                    const float2 cb = make_float2(c2 * dmin.x, c2 * dmin.y);
                    const float2 nb = make_float2(ac.b[i].x - cb.x > kPairRebase ? cb.x - kPairHead : ac.b[i].x,
                                                  ac.b[i].y - cb.y > kPairRebase ? cb.y - kPairHead : ac.b[i].y);
                    // scale by 2^(nb - b) in two halves: the factor itself may be below 2^-126 when the product is not
                    const float2 sc = make_float2(ex2(0.5f * (nb.x - ac.b[i].x)), ex2(0.5f * (nb.y - ac.b[i].y)));
                    float2 zz = mul2(mul2(ac.z[i], sc), sc), nn = mul2(mul2(ac.n[i], sc), sc);
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        const float2 ar = fma2(D[q], nc2, nb);
                        const float2 u = make_float2(ex2(ar.x), ex2(ar.y));
                        zz = add2(zz, u);
                        nn = fma2(u, cand2[i + q], nn);
                    }
                    ac.z[i] = zz; ac.n[i] = nn; ac.b[i] = nb;
                }
            }
        }
#pragma unroll
        for (int q = 0; q < W; ++q)
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                ring[0][q][i] = ring[1][q][i];
                ring[1][q][i] = ring[2][q][i];
                ring[2][q][i] = ring[3][q][i];
                ring[3][q][i] = X[q][i];
            }
        // output x-index i, offset q reads the candidate at window element i + 2 + q
        if (!SEP) {
#pragma unroll
            for (int k = 0; k < W + 1; ++k) {
                cand2[k] = cand1[k];
                cand1[k] = b[k + 2];
            }
        }
    }
    return fail;
}

template <int M, int RZ, int TX, int NCTA, bool SEP = false>
__global__ void __launch_bounds__(Pair5Geom<M, RZ, TX, SEP>::NT, NCTA)
tnlm_pair5_kernel(const float *__restrict__ f, const float *__restrict__ g, const float *__restrict__ ref, float *f_out,
                  const Dims dm, const int tiles_x, const int tiles_y, const int tiles_z)
{
    using G = Pair5Geom<M, RZ, TX, SEP>;
    constexpr int AP = G::NPA * G::PA2, BP = G::NPB * G::PB2;   // plane strides (float2)
    extern __shared__ __align__(16) float smem[];
    float2 *sA = reinterpret_cast<float2 *>(smem);
    float2 *sBE = sA + G::A_F2;
    float2 *sBO = sBE + G::NPE * G::PB2;   // odd pairs of plane 0
    float2 *sFE = sBE + G::B_F2;           // SEP: candidate tile, same plane layout as B
    float2 *sFO = sFE + G::NPE * G::PB2;

    int t = blockIdx.x;
    const int bx = t % tiles_x; t /= tiles_x;
    const int by = t % tiles_y; t /= tiles_y;
    const int bz = t % tiles_z; t /= tiles_z;
    const int ph = t;
    // z-tiles aligned to absolute multiples of RZ (slab-invariant rounding, as in tnlm_pair_kernel)
    const int X0 = bx * TX, Y0 = by * kPair5RowsOut, Z0 = (dm.z_begin / RZ + bz) * RZ;
    const size_t V = (size_t)dm.Z * dm.Y * dm.X;
    const int tid = threadIdx.x;
    const int l = tid & 15;            // row pair: tile rows 2l, 2l+1
    const int x0 = 2 * (tid >> 4);     // first x of the run, tile relative

    // -ref_i tile (halo 2): rows <-> y = Y0-2+r, cols <-> x = X0-2+c, planes <-> z = Z0-2+pz
    stage_pairs<G::PA2, 32, G::ACOLS, G::NAP, G::NPA, 0, true, G::NT>(
        reinterpret_cast<float *>(sA), nullptr, ref + (size_t)ph * V, Z0 - 2, Y0 - 2, X0 - 2, dm, tid);

    const size_t zstride = (size_t)dm.Y * dm.X;
    const bool vec_ok = (dm.X % 2) == 0;
    const bool col_ok = X0 + x0 < dm.X;

#pragma unroll 1
    for (int s = 0; s < 2; ++s) {
        const int j = (ph + (s ? 1 : dm.P - 1)) % dm.P;
        __syncthreads();   // everyone is done with the previous B tiles
        // ref_j tiles (halo 2+M): rows <-> y = Y0-2-M+r, cols <-> x = X0-2-M+c, planes <-> z = Z0-2-M+pz
        stage_pairs<G::PB2, 32 + 2 * M, G::BCOLS, G::NBP, G::NPE, G::NPO, false, G::NT>(
            reinterpret_cast<float *>(sBE), reinterpret_cast<float *>(sBO), ref + (size_t)j * V, Z0 - 2 - M, Y0 - 2 - M,
            X0 - 2 - M, dm, tid);
        if constexpr (SEP)   // f_j, same rows and columns, planes <-> z = Z0-M+pz
            stage_pairs<G::PB2, 32 + 2 * M, G::BCOLS, G::NFP, G::NPE, G::NPO, false, G::NT>(
                reinterpret_cast<float *>(sFE), reinterpret_cast<float *>(sFO), f + (size_t)j * V, Z0 - M, Y0 - 2 - M,
                X0 - 2 - M, dm, tid);
        __syncthreads();

        AccPair acc[RZ];
#pragma unroll
        for (int o = 0; o < RZ; ++o)
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                acc[o].z[i] = make_float2(0.f, 0.f);
                acc[o].n[i] = make_float2(0.f, 0.f);
                acc[o].b[i] = make_float2(INFINITY, INFINITY);   // first use takes the re-base path
            }
        const float2 *aRow = sA + l * G::PA2 + x0;
        auto run_chunk = [&](auto wtag, const float2 *bRow, const bool first) {
            constexpr int W = decltype(wtag)::value;
            const float2 *fRow = bRow + (sFE - sBE);   // same (plane, pair, column) of the candidate tile
            unsigned fail = 0xffffffffu;   // first use: every reference exponent is still +inf
            if (!first) fail = pair5_pass<RZ, W, false, AP, BP, SEP>(aRow, bRow, fRow, dm.c2, acc, 0u);
            if (__any_sync(0xffffffffu, fail != 0u)) pair5_pass<RZ, W, true, AP, BP, SEP>(aRow, bRow, fRow, dm.c2, acc, fail);
        };
#pragma unroll 1
        for (int k = 0; k < G::E * G::E; ++k) {
            const int kk = (k + (G::E * G::E) / 2) % (G::E * G::E);   // zero y/z offset first
            const int tz = kk / G::E, ty = kk % G::E;                 // offset + M
            const float2 *bRow = ((ty & 1) ? sBO : sBE) + (tz * G::NPB + l + (ty >> 1)) * G::PB2 + x0;
            // the chunk holding the zero x-offset (q = M) goes first, so that the first careful pass sets
            // the reference exponents from the best candidates
#pragma unroll 1
            for (int cc = 0; cc < M; ++cc) {
                const int c = (cc + M / 2) % M;
                if (c == M - 1) run_chunk(std::integral_constant<int, 3>{}, bRow + 2 * c, k == 0 && cc == 0);
                else run_chunk(std::integral_constant<int, 2>{}, bRow + 2 * c, k == 0 && cc == 0);
            }
        }

        // epilogue: rows 2l (.x) and 2l+1 (.y); tile rows 2..29 are outputs
        bool row_ok[2];
        size_t base0[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int r = 2 * l + e, y = Y0 - 2 + r;
            row_ok[e] = r >= 2 && r <= kPair5RowsOut + 1 && y < dm.Y && col_ok;
            base0[e] = (size_t)ph * V + ((size_t)Z0 * dm.Y + min(max(y, 0), dm.Y - 1)) * dm.X + X0 + x0;
        }
#pragma unroll
        for (int e = 0; e < 2; ++e)
#pragma unroll
            for (int o = 0; o < RZ; ++o) {
                if (row_ok[e] && Z0 + o >= dm.z_begin && Z0 + o < dm.z_end) {
                    const float n0 = e ? __fdividef(acc[o].n[0].y, acc[o].z[0].y) : __fdividef(acc[o].n[0].x, acc[o].z[0].x);
                    const float n1 = e ? __fdividef(acc[o].n[1].y, acc[o].z[1].y) : __fdividef(acc[o].n[1].x, acc[o].z[1].x);
                    float *dst = f_out + base0[e] + o * zstride;
                    const bool two = X0 + x0 + 1 < dm.X;
                    if (s == 0) {
                        // park NLM- in f_out; the same thread reads it back after the second direction
                        if (vec_ok) {
                            *reinterpret_cast<float2 *>(dst) = make_float2(n0, n1);
                        } else {
                            dst[0] = n0;
                            if (two) dst[1] = n1;
                        }
                    } else {
                        // a5: Jacobi combine (Eq. 8)
                        const float *gp = g + base0[e] + o * zstride;
                        if (vec_ok) {
                            const float2 gv = __ldg(reinterpret_cast<const float2 *>(gp));
                            const float2 pv = *reinterpret_cast<const float2 *>(dst);
                            *reinterpret_cast<float2 *>(dst) = make_float2(fmaf(dm.a_g, gv.x, dm.a_n * (pv.x + n0)),
                                                                           fmaf(dm.a_g, gv.y, dm.a_n * (pv.y + n1)));
                        } else {
                            dst[0] = fmaf(dm.a_g, __ldg(gp), dm.a_n * (dst[0] + n0));
                            if (two) dst[1] = fmaf(dm.a_g, __ldg(gp + 1), dm.a_n * (dst[1] + n1));
                        }
                    }
                }
            }
    }
}

// ---------------------------------------------------------------------------------------------
inline bool pair5_supported(const tnlm_params &p)
{
    return p.patch_radius == 2 && p.search_radius >= 1 && p.search_radius <= 4;
}
inline const char *pair5_name(const tnlm_params &p)
{
    switch (p.search_radius) {
        case 1: return "tnlm_pair5_kernel<M=1>";
        case 2: return "tnlm_pair5_kernel<M=2>";
        case 3: return "tnlm_pair5_kernel<M=3>";
        default: return "tnlm_pair5_kernel<M=4>";
    }
}

template <int M, int RZ, int TX, int NCTA, bool SEP = false>
cudaError_t launch_pair5_t(const Dims &dm, const float *f, const float *g, const float *ref, float *f_out, cudaStream_t st)
{
    using G = Pair5Geom<M, RZ, TX, SEP>;
    static_assert(NCTA * (G::BYTES + 1024) <= 228 * 1024, "NCTA tiles of the pair5 kernel do not fit in shared memory");
    static std::atomic<uint64_t> configured{0};   // per template instance: one bit per device
    cudaError_t e = ensure_dynamic_smem(tnlm_pair5_kernel<M, RZ, TX, NCTA, SEP>, G::BYTES, configured);
    if (e != cudaSuccess) return e;
    const int tiles_x = (dm.X + TX - 1) / TX;
    const int tiles_y = (dm.Y + kPair5RowsOut - 1) / kPair5RowsOut;
    const int tiles_z = (dm.z_end + RZ - 1) / RZ - dm.z_begin / RZ;   // tiles aligned to multiples of RZ
    const long long blocks = (long long)tiles_x * tiles_y * tiles_z * dm.P;
    if (blocks <= 0 || blocks > 2147483647LL) return cudaErrorInvalidConfiguration;
    tnlm_pair5_kernel<M, RZ, TX, NCTA, SEP><<<(unsigned)blocks, G::NT, G::BYTES, st>>>(f, g, ref, f_out, dm, tiles_x, tiles_y, tiles_z);
    return cudaGetLastError();
}

// With a separate ref stack the candidate tile F needs room of its own: shallower or narrower tiles (see launch_pair).
inline cudaError_t launch_pair5(const tnlm_params &p, const Dims &dm, const float *f, const float *g, const float *ref,
                                float *f_out, cudaStream_t st)
{
    if (ref == f) {
        switch (p.search_radius) {
            case 1: return launch_pair5_t<1, 6, 16, 2>(dm, f, g, f, f_out, st);
            case 2: return launch_pair5_t<2, 4, 16, 2>(dm, f, g, f, f_out, st);
            case 3: return launch_pair5_t<3, 4, 32, 1>(dm, f, g, f, f_out, st);
            case 4: return launch_pair5_t<4, 2, 32, 1>(dm, f, g, f, f_out, st);
            default: return cudaErrorNotSupported;
        }
    }
    switch (p.search_radius) {
        case 1: return launch_pair5_t<1, 4, 32, 1, true>(dm, f, g, ref, f_out, st);
        case 2: return launch_pair5_t<2, 2, 32, 1, true>(dm, f, g, ref, f_out, st);
        case 3: return launch_pair5_t<3, 2, 16, 1, true>(dm, f, g, ref, f_out, st);
        case 4: return launch_pair5_t<4, 2, 8, 1, true>(dm, f, g, ref, f_out, st);
        default: return cudaErrorNotSupported;
    }
}

}  // namespace tnlm
