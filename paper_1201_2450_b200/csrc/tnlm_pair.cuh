// Row-pair packed sm_100a TNLM sweep kernel for 3^3 patches (d = 1), search radius M in {1,2,3,4}.
//
// Blackwell's FP32 pipe executes FADD2 / FMUL2 / FFMA2 (two fp32 lanes of a 64-bit register pair per
// thread) at the same lane rate as the scalar forms but for half the issue slots; the scalar tiled
// kernel (tnlm_tiled.cuh) is issue bound.  Here every value of the distance pipeline is a float2 that
// holds the SAME quantity for two vertically adjacent voxels (rows 2l and 2l+1 of the tile), so a1-a4
// all run packed, and each thread needs one shuffle per output for the y-sum instead of two.
//
// One CTA = one (phase i, TX-wide x-tile, 30-row y-group, RZ-plane z-slab), both neighbour phases in turn
// (Eq. 8).  Shared memory holds float2 row-pair tiles:
//   A2 [RZ+2   ][16  ][PA2]   -ref_i, pair k = tile rows (2k, 2k+1), halo d = 1 (stored negated: a1 is an add)
//   B  [RZ+2+2M][31+2M][PB2]   ref_j, halo 1+M; each plane holds two copies of its rows:
//        BE = pairs 0..15+M,  pair k = tile rows (2k,   2k+1)   used when the y-offset is even
//        BO = pairs 16+M..,   pair k = tile rows (2k+1, 2k+2)   used when the y-offset is odd
// (clamp-to-edge applied while staging: reading P4).  The second copy of B keeps the operand of every
// packed op an aligned register pair for any y-offset.
//
//   half-warp   = 16 lanes = 16 row pairs = 32 tile rows (rows 0 and 31 are the d-halo: 30 output rows)
//   thread      = 2 rows x an x-run of 2 voxels x a column of RZ output planes = 4*RZ outputs
//   registers   = (Z, N, reference exponent) of its outputs for the whole search window
//   per (ty,tz) = a "pass": march the RZ+2 planes; per plane, for W consecutive tx at once
//       a1  d = b + (-a)                                      FADD2, operands straight from LDS.128 windows
//       a2x 3-tap x-sum of squares; the two outputs share the middle pair    FMUL2 + 3 FFMA2 per 2 outputs
//       a2z 3-tap z-sum from a two-plane register ring; even/odd outputs share a pair sum   1.5 FADD2
//       a2y S.lo + S.hi (own two rows) + one row from the lane above / below  1 FADD + 2 SHFL + 1 FADD2
//       a3  u = ex2(bias - c2*D)                                              FFMA2 + 2 MUFU.EX2
//       a4  Z += u, N += u * f_j(x+t)                                         FADD2 + FFMA2
//   epilogue    = NLM of the first direction is parked in f_out (same thread reads it back), then
//                 a5: f_out = mu/(2+mu) g + (NLM- + NLM+)/(2+mu)
// SEP = true (ref != f: weights from another stack than the one that is averaged): a third tile F holds
// f_j in the layout of B (both copies) for the planes that carry candidates; the candidate window of a pass is read
// from F instead of being the centre of the B window of the previous plane.
// Reference exponent (reading P3: weights relative to the best candidate).  Every output keeps a
// reference exponent b; a pass sums its W terms ex2(b - c2*D) optimistically.  If the partial
// normaliser stays below 2^100 (no candidate ~2^100 times better than the reference) it is added as
// it is; otherwise (first use, b = +inf; later only at moving high-contrast edges) nothing is added,
// the row pair is flagged, and the warp re-does that pass in a careful form that re-bases flagged
// pairs on min(b, c2*Dmin of the pass - 90) and re-evaluates their terms (the 90 binades of headroom make a
// second re-base of the same output rare even on noise-dominated stacks).  The result equals the shifted
// softmax up to rounding.
#pragma once
#include <cstdlib>
#include <type_traits>

#include "tnlm_common.cuh"
#include "tnlm_tiled.cuh"

namespace tnlm {

constexpr int kPairRowsOut = 30;

__host__ __device__ constexpr int pitch2(int n)   // smallest p >= n with p = 2 (mod 4): conflict-free LDS.128
{
    int p = n;
    while (p % 4 != 2) ++p;
    return p;
}

__device__ __forceinline__ float2 add2(const float2 a, const float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 mul2(const float2 a, const float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(const float2 a, const float2 b, const float2 c) { return __ffma2_rn(a, b, c); }

template <int M, int RZ, int TX, bool SEP = false> struct PairGeom {
    using C = Chunks<M>;
    static constexpr int E = 2 * M + 1;
    static constexpr int NRUN = TX / 2;             // x-runs of 2 voxels
    static constexpr int NT = NRUN * 16;            // 16 row-pair lanes per run
    static constexpr int NVB0 = (C::W0 + 4) / 2;    // LDS.128 per B row window (2 + W + 1 positions)
    static constexpr int NVB1 = C::W1 ? (C::W1 + 4) / 2 : 0;
    static constexpr int ACOLS = TX + 2, BCOLS = TX + 2 * M + 2;   // staged columns
    static constexpr int BREAD = cmax(TX - 2 + 2 * NVB0, C::W1 ? TX - 2 + 4 + 2 * NVB1 : 0);   // columns a window may touch
    static constexpr int PA2 = pitch2(ACOLS);
    static constexpr int PB2 = pitch2(cmax(BCOLS, BREAD));
    static constexpr int NPA = 16, NPE = 16 + M, NPO = 15 + M;     // row pairs per plane
    static constexpr int NPB = NPE + NPO;                          // a B plane = its BE pairs, then its BO pairs
    static constexpr int NAP = RZ + 2, NBP = RZ + 2 + 2 * M;       // planes
    static constexpr int NFP = SEP ? RZ + 2 * M : 0;               // planes of the candidate tile F: B planes 1 .. NBP-2
    static constexpr int A_F2 = NAP * NPA * PA2, B_F2 = NBP * NPB * PB2, F_F2 = NFP * NPB * PB2;
    static constexpr size_t BYTES = (size_t)(A_F2 + B_F2 + F_F2) * sizeof(float2);
};

struct AccPair { float2 z[2], n[2], b[2]; };   // [x of the run]; .x = row 2l, .y = row 2l+1

// Guard band and headroom of the reference exponents.  Partial sums up to 2^100 (relative to the reference) are added
// as they are: Z stays below 2^107 (inside __fdividef's range) and N below 2^107 * max|f|, finite for |f| < 2^20
// (a 2^80 band would cover |f| < 2^40 but re-bases noise-dominated stacks 15 % more often).
// A re-base puts the best candidate seen so far at 2^-90, not at 1: later candidates may be up to 2^190 times better
// before the guard trips again, while terms down to 2^-36 of the best stay normal (125 * 2^-36 = 2e-9 of the sum).
constexpr float kPairHead = 90.f;
constexpr float kPairRebase = 97.f;   // careful form: re-base a row whose best term would exceed 2^97 (5 such terms stay below 2^100)
constexpr float kPairGuard = 1.2676506002282294e30f;   // 2^100

template <int NV>
__device__ __forceinline__ void load_pairs(const float2 *__restrict__ p, float2 (&dst)[2 * NV])
{
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        const float4 t = *reinterpret_cast<const float4 *>(p + 2 * v);
        dst[2 * v] = make_float2(t.x, t.y);
        dst[2 * v + 1] = make_float2(t.z, t.w);
    }
}

// One pass: W consecutive x-offsets at fixed (ty, tz), marching the RZ+2 planes.
//   aRow: &A2[plane 0][pair l][x0]                 element k <-> x = X0 + x0 - 1 + k   (negated values)
//   bRow: &B?[plane tz][pair l + ty/2][x0 + q0]    element k + q pairs with a[k] for the q-th offset of the chunk
// CAREFUL = false (hot): the W terms of a row pair are summed optimistically relative to its reference
//   exponents and added if the partial normaliser stayed inside the guard band; otherwise nothing is
//   added and bit 2*o + i of the returned mask is set.
// CAREFUL = true: only the row pairs named in `mask` are touched; each of the two rows is re-based on
//   c2*Dmin of the chunk (with headroom) if that beats its reference by more than 2^97, branch-free, and the
//   terms are evaluated once.  Used for the first chunk (reference = +inf) and to re-do a chunk that reported failures.
// Both forms execute the same shuffles, so a warp may run them with different masks per lane.
//   fRow (SEP only): &F?[plane tz][pair l + ty/2][x0 + q0], F plane k <-> B plane k + 1
template <int RZ, int W, bool CAREFUL, int A_PLANE, int B_PLANE, bool SEP = false>
__device__ __forceinline__ unsigned pair_pass(const float2 *__restrict__ aRow, const float2 *__restrict__ bRow,
                                              const float2 *__restrict__ fRow, const float c2, AccPair (&acc)[RZ],
                                              const unsigned mask)
{
    constexpr int NVB = (W + 4) / 2;
    const float2 nc2 = make_float2(-c2, -c2);
    float2 ring0[W][2], ring1[W][2];
    float2 bprev[2 * NVB];
    unsigned fail = 0u;
#pragma unroll
    for (int p = 0; p < RZ + 2; ++p) {
        float2 a[4], b[2 * NVB];
        load_pairs<2>(aRow + p * A_PLANE, a);
        load_pairs<NVB>(bRow + p * B_PLANE, b);
        float2 X[W][2];
#pragma unroll
        for (int q = 0; q < W; ++q) {
            float2 d[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) d[k] = add2(b[k + q], a[k]);                      // a1 (a is -ref_i)
            const float2 mid = fma2(d[2], d[2], mul2(d[1], d[1]));                        // a2x
            X[q][0] = fma2(d[0], d[0], mid);
            X[q][1] = fma2(d[3], d[3], mid);
        }
        if (p >= 2) {
            AccPair &ac = acc[p - 2];
            if (SEP) load_pairs<NVB>(fRow + (p - 2) * B_PLANE, bprev);   // candidates f_j(x+t) of the centre plane
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                float2 D[W];
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    // a2z: outputs (o, o+1), o even, share X[o+1] + X[o+2]: 3 adds per 2 outputs
                    float2 S;
                    if ((p & 1) == 0) {
                        ring1[q][i] = add2(ring1[q][i], X[q][i]);    // X[o+1] + X[o+2]
                        S = add2(ring0[q][i], ring1[q][i]);
                    } else {
                        S = add2(ring0[q][i], X[q][i]);              // ring0 holds the shared pair sum
                    }
                    const float own = S.x + S.y;                                          // a2y
                    const float up = __shfl_up_sync(0xffffffffu, S.y, 1);                 // row 2l-1
                    const float dn = __shfl_down_sync(0xffffffffu, S.x, 1);               // row 2l+2
                    D[q] = add2(make_float2(up, dn), make_float2(own, own));
                }
                if (!CAREFUL) {
                    // hot form: optimistic partial sums relative to the reference exponents, one guard per row pair
                    float2 zp = make_float2(0.f, 0.f), np = make_float2(0.f, 0.f);
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        const float2 arg = fma2(D[q], nc2, ac.b[i]);                      // a3
                        const float2 u = make_float2(ex2(arg.x), ex2(arg.y));
                        zp = add2(zp, u);                                                 // a4
                        np = fma2(u, bprev[i + 1 + q], np);
                    }
                    if (fmaxf(zp.x, zp.y) <= kPairGuard) {
                        ac.z[i] = add2(ac.z[i], zp);
                        ac.n[i] = add2(ac.n[i], np);
                    } else {
                        fail |= 1u << (2 * (p - 2) + i);
                    }
                } else if ((mask >> (2 * (p - 2) + i)) & 1u) {
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
                        nn = fma2(u, bprev[i + 1 + q], nn);
                    }
                    ac.z[i] = zz; ac.n[i] = nn; ac.b[i] = nb;
                }
            }
        }
        // ring state after plane p: p < 2 or p odd -> (X[p-1], X[p]); p even -> (X[p-1] + X[p], X[p])
#pragma unroll
        for (int q = 0; q < W; ++q)
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                ring0[q][i] = ring1[q][i];
                ring1[q][i] = X[q][i];
            }
        if (!SEP) {
#pragma unroll
            for (int k = 0; k < 2 * NVB; ++k) bprev[k] = b[k];
        }
    }
    return fail;
}

// Stage a clamped halo tile into row-pair layout(s):
//   tile element (pz, r, c) <- sign * src(clamp(zo+pz), clamp(yo+r), clamp(xo+c))
//   dstE pair r/2 (half r&1); dstO (optional) pair (r-1)/2 (half (r-1)&1) for r >= 1
// The (r, c) of a thread's k-th element is the same in every plane, so its global offset inside a
// plane and its shared-memory offsets are tabulated once; the plane loop is then LDG + STS only,
// four or five planes in flight per thread.
template <int PITCH2, int ROWS, int COLS, int PLANES, int NP, int NPO, bool NEGATE, int NT>
__device__ __forceinline__ void stage_pairs(float *__restrict__ dstE, float *__restrict__ dstO,
                                            const float *__restrict__ src, const int zo, const int yo, const int xo,
                                            const Dims &dm, const int tid)
{
    constexpr int K = (ROWS * COLS + NT - 1) / NT;
    constexpr bool ODD = NPO > 0;
    constexpr int PLANE_F = (NP + NPO) * PITCH2 * 2;   // floats per shared-memory plane (even pairs, then odd pairs)
    constexpr int PF = (PLANES % 7 == 0 && K <= 4) ? 7 : (PLANES % 5 == 0 && K <= 8) ? 5 : 4;   // planes in flight
    int goff[K], eoff[K], ooff[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int idx = tid + k * NT;
        const int r = idx / COLS, c = idx - r * COLS;
        const bool ok = idx < ROWS * COLS;
        goff[k] = clampi(yo + r, dm.Y) * dm.X + clampi(xo + c, dm.X);
        eoff[k] = ok ? (((r >> 1) * PITCH2 + c) * 2 + (r & 1)) : -1;
        const int ro = r - 1;
        ooff[k] = (ok && ro >= 0 && (ro >> 1) < NPO) ? (((ro >> 1) * PITCH2 + c) * 2 + (ro & 1)) : -1;
        if (!ok) goff[k] = 0;
    }
    const size_t plane = (size_t)dm.Y * dm.X;
#pragma unroll 1
    for (int pz = 0; pz < PLANES; pz += PF) {
        float v[PF][K];
#pragma unroll
        for (int h = 0; h < PF; ++h) {
            const float *sp = src + (size_t)clampi(zo + min(pz + h, PLANES - 1), dm.Z) * plane;
#pragma unroll
            for (int k = 0; k < K; ++k) v[h][k] = __ldg(sp + goff[k]);
        }
#pragma unroll
        for (int h = 0; h < PF; ++h) {
            if (pz + h < PLANES) {
                float *dE = dstE + (pz + h) * PLANE_F;
                float *dO = dstO + (pz + h) * PLANE_F;
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    const float val = NEGATE ? -v[h][k] : v[h][k];
                    if (eoff[k] >= 0) dE[eoff[k]] = val;
                    if (ODD && ooff[k] >= 0) dO[ooff[k]] = val;
                }
            }
        }
    }
}

template <int M, int RZ, int TX, int NCTA, bool SEP = false>
__global__ void __launch_bounds__(PairGeom<M, RZ, TX, SEP>::NT, NCTA)
tnlm_pair_kernel(const float *__restrict__ f, const float *__restrict__ g, const float *__restrict__ ref, float *f_out,
                 const Dims dm, const int tiles_x, const int tiles_y, const int tiles_z)
{
    using G = PairGeom<M, RZ, TX, SEP>;
    using C = Chunks<M>;
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
    // z-tiles are aligned to absolute multiples of RZ, so a voxel is computed at the same place of a tile
    // (same rounding) whatever output slab [z_begin, z_end) the call covers
    const int X0 = bx * TX, Y0 = by * kPairRowsOut, Z0 = (dm.z_begin / RZ + bz) * RZ;
    const size_t V = (size_t)dm.Z * dm.Y * dm.X;
    const int tid = threadIdx.x;
    const int l = tid & 15;            // row pair: tile rows 2l, 2l+1
    const int x0 = 2 * (tid >> 4);     // first x of the run, tile relative

    // -ref_i tile (halo 1): rows <-> y = Y0-1+r, cols <-> x = X0-1+c, planes <-> z = Z0-1+pz
    stage_pairs<G::PA2, 32, G::ACOLS, G::NAP, G::NPA, 0, true, G::NT>(
        reinterpret_cast<float *>(sA), nullptr, ref + (size_t)ph * V, Z0 - 1, Y0 - 1, X0 - 1, dm, tid);

    const size_t zstride = (size_t)dm.Y * dm.X;
    const bool vec_ok = (dm.X % 2) == 0;
    const bool col_ok = X0 + x0 < dm.X;

#pragma unroll 1
    for (int s = 0; s < 2; ++s) {
        const int j = (ph + (s ? 1 : dm.P - 1)) % dm.P;
        __syncthreads();   // everyone is done with the previous B tiles
        // ref_j tiles (halo 1+M): rows <-> y = Y0-1-M+r, cols <-> x = X0-1-M+c, planes <-> z = Z0-1-M+pz
        stage_pairs<G::PB2, 32 + 2 * M, G::BCOLS, G::NBP, G::NPE, G::NPO, false, G::NT>(
            reinterpret_cast<float *>(sBE), reinterpret_cast<float *>(sBO), ref + (size_t)j * V, Z0 - 1 - M, Y0 - 1 - M,
            X0 - 1 - M, dm, tid);
        if constexpr (SEP)   // f_j, same rows and columns, planes <-> z = Z0-M+pz
            stage_pairs<G::PB2, 32 + 2 * M, G::BCOLS, G::NFP, G::NPE, G::NPO, false, G::NT>(
                reinterpret_cast<float *>(sFE), reinterpret_cast<float *>(sFO), f + (size_t)j * V, Z0 - M, Y0 - 1 - M,
                X0 - 1 - M, dm, tid);
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
        // a chunk of a pass: hot form first; if any lane of the warp reports guard failures, the whole
        // warp re-does the chunk in the careful form (each lane with its own mask of failed row pairs)
        auto run_chunk = [&](auto wtag, const float2 *bRow, const bool first) {
            constexpr int W = decltype(wtag)::value;
            const float2 *fRow = bRow + (sFE - sBE);   // same (plane, pair, column) of the candidate tile
            unsigned fail = 0xffffffffu;   // first use: every reference exponent is still +inf
            if (!first) fail = pair_pass<RZ, W, false, AP, BP, SEP>(aRow, bRow, fRow, dm.c2, acc, 0u);
            if (__any_sync(0xffffffffu, fail != 0u)) pair_pass<RZ, W, true, AP, BP, SEP>(aRow, bRow, fRow, dm.c2, acc, fail);
        };
#pragma unroll 1
        for (int k = 0; k < G::E * G::E; ++k) {
            // start with (ty, tz) = (0, 0): the zero offset is usually the best match, so the reference
            // exponents are set once, in the first pass, and the careful form stays cold afterwards
            const int kk = (k + (G::E * G::E) / 2) % (G::E * G::E);
            const int tz = kk / G::E, ty = kk % G::E;   // offset + M
            const float2 *bRow = ((ty & 1) ? sBO : sBE) + (tz * G::NPB + l + (ty >> 1)) * G::PB2 + x0;
            run_chunk(std::integral_constant<int, C::W0>{}, bRow, k == 0);
            if constexpr (C::W1 > 0) run_chunk(std::integral_constant<int, C::W1>{}, bRow + 4, false);
        }

        // epilogue: rows 2l (.x) and 2l+1 (.y); tile rows 1..30 are outputs
        bool row_ok[2];
        size_t base0[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int r = 2 * l + e, y = Y0 - 1 + r;
            row_ok[e] = r >= 1 && r <= kPairRowsOut && y < dm.Y && col_ok;
            base0[e] = (size_t)ph * V + ((size_t)Z0 * dm.Y + min(y, dm.Y - 1)) * dm.X + X0 + x0;
        }
        if (s == 0) {
            // park NLM- in f_out; the same thread reads it back after the second direction
#pragma unroll
            for (int e = 0; e < 2; ++e)
#pragma unroll
                for (int o = 0; o < RZ; ++o) {
                    if (row_ok[e] && Z0 + o >= dm.z_begin && Z0 + o < dm.z_end) {
                        const float n0 = e ? __fdividef(acc[o].n[0].y, acc[o].z[0].y) : __fdividef(acc[o].n[0].x, acc[o].z[0].x);
                        const float n1 = e ? __fdividef(acc[o].n[1].y, acc[o].z[1].y) : __fdividef(acc[o].n[1].x, acc[o].z[1].x);
                        float *dst = f_out + base0[e] + o * zstride;
                        if (vec_ok) {
                            *reinterpret_cast<float2 *>(dst) = make_float2(n0, n1);
                        } else {
                            dst[0] = n0;
                            if (X0 + x0 + 1 < dm.X) dst[1] = n1;
                        }
                    }
                }
        } else {
            // a5: Jacobi combine (Eq. 8); all loads are issued before the first dependent use
            float2 gv[2][RZ], pv[2][RZ];
#pragma unroll
            for (int e = 0; e < 2; ++e)
#pragma unroll
                for (int o = 0; o < RZ; ++o) {
                    gv[e][o] = pv[e][o] = make_float2(0.f, 0.f);
                    if (row_ok[e] && Z0 + o >= dm.z_begin && Z0 + o < dm.z_end) {
                        const float *gp = g + base0[e] + o * zstride;
                        const float *pp = f_out + base0[e] + o * zstride;
                        if (vec_ok) {
                            gv[e][o] = __ldg(reinterpret_cast<const float2 *>(gp));
                            pv[e][o] = *reinterpret_cast<const float2 *>(pp);
                        } else {
                            gv[e][o].x = __ldg(gp);
                            pv[e][o].x = pp[0];
                            if (X0 + x0 + 1 < dm.X) {
                                gv[e][o].y = __ldg(gp + 1);
                                pv[e][o].y = pp[1];
                            }
                        }
                    }
                }
#pragma unroll
            for (int e = 0; e < 2; ++e)
#pragma unroll
                for (int o = 0; o < RZ; ++o) {
                    if (row_ok[e] && Z0 + o >= dm.z_begin && Z0 + o < dm.z_end) {
                        const float n0 = e ? __fdividef(acc[o].n[0].y, acc[o].z[0].y) : __fdividef(acc[o].n[0].x, acc[o].z[0].x);
                        const float n1 = e ? __fdividef(acc[o].n[1].y, acc[o].z[1].y) : __fdividef(acc[o].n[1].x, acc[o].z[1].x);
                        const float r0 = fmaf(dm.a_g, gv[e][o].x, dm.a_n * (pv[e][o].x + n0));
                        const float r1 = fmaf(dm.a_g, gv[e][o].y, dm.a_n * (pv[e][o].y + n1));
                        float *dst = f_out + base0[e] + o * zstride;
                        if (vec_ok) {
                            *reinterpret_cast<float2 *>(dst) = make_float2(r0, r1);
                        } else {
                            dst[0] = r0;
                            if (X0 + x0 + 1 < dm.X) dst[1] = r1;
                        }
                    }
                }
        }
    }
}

// ---------------------------------------------------------------------------------------------
inline bool pair_supported(const tnlm_params &p)
{
    return p.patch_radius == 1 && p.search_radius >= 1 && p.search_radius <= 4;
}
inline const char *pair_name(const tnlm_params &p)
{
    switch (p.search_radius) {
        case 1: return "tnlm_pair_kernel<M=1>";
        case 2: return "tnlm_pair_kernel<M=2>";
        case 3: return "tnlm_pair_kernel<M=3>";
        default: return "tnlm_pair_kernel<M=4>";
    }
}

template <int M, int RZ, int TX, int NCTA, bool SEP = false>
cudaError_t launch_pair_t(const Dims &dm, const float *f, const float *g, const float *ref, float *f_out, cudaStream_t st)
{
    using G = PairGeom<M, RZ, TX, SEP>;
    static_assert(NCTA * (G::BYTES + 1024) <= 228 * 1024, "NCTA tiles of the pair kernel do not fit in shared memory");
    static std::atomic<uint64_t> configured{0};   // per template instance: one bit per device
    cudaError_t e = ensure_dynamic_smem(tnlm_pair_kernel<M, RZ, TX, NCTA, SEP>, G::BYTES, configured);
    if (e != cudaSuccess) return e;
    const int tiles_x = (dm.X + TX - 1) / TX;
    const int tiles_y = (dm.Y + kPairRowsOut - 1) / kPairRowsOut;
    const int tiles_z = (dm.z_end + RZ - 1) / RZ - dm.z_begin / RZ;   // tiles aligned to multiples of RZ
    const long long blocks = (long long)tiles_x * tiles_y * tiles_z * dm.P;
    if (blocks <= 0 || blocks > 2147483647LL) return cudaErrorInvalidConfiguration;
    tnlm_pair_kernel<M, RZ, TX, NCTA, SEP><<<(unsigned)blocks, G::NT, G::BYTES, st>>>(f, g, ref, f_out, dm, tiles_x, tiles_y, tiles_z);
    return cudaGetLastError();
}

// <M, RZ, TX, CTAs per SM>: the shapes that measured best on the thorax phantoms.  With a
// separate ref stack the candidate tile F needs room of its own: shallower or narrower tiles, fewer CTAs per SM.
inline cudaError_t launch_pair(const tnlm_params &p, const Dims &dm, const float *f, const float *g, const float *ref,
                               float *f_out, cudaStream_t st)
{
    if (ref == f) {
        switch (p.search_radius) {
            case 1: return launch_pair_t<1, 4, 16, 3>(dm, f, g, f, f_out, st);
            case 2: return launch_pair_t<2, 4, 16, 3>(dm, f, g, f, f_out, st);
            case 3: return launch_pair_t<3, 6, 32, 1>(dm, f, g, f, f_out, st);
            case 4: return launch_pair_t<4, 4, 32, 1>(dm, f, g, f, f_out, st);
            default: return cudaErrorNotSupported;
        }
    }
    switch (p.search_radius) {
        case 1: return launch_pair_t<1, 4, 16, 2, true>(dm, f, g, ref, f_out, st);
        case 2: return launch_pair_t<2, 4, 32, 1, true>(dm, f, g, ref, f_out, st);
        case 3: return launch_pair_t<3, 2, 24, 1, true>(dm, f, g, ref, f_out, st);
        case 4: return launch_pair_t<4, 2, 16, 1, true>(dm, f, g, ref, f_out, st);
        default: return cudaErrorNotSupported;
    }
}

}  // namespace tnlm
