// 5^3-patch sweep kernel (d = 2, ref == f) with the thread-private operands in tensor memory and a rolling ref_j window.
//
// tnlm_pair5_kernel's arithmetic (read tnlm_pair5.cuh first: 6 differences per 2-voxel run, 5-tap x-sums that share
// their four middle squares, 5-tap z-sum, 5-tap y-sum from four shuffles per row pair) with the two changes that took the
// 3^3-patch kernels of the 7^3 / 9^3 windows from one CTA per SM to three / two (tnlm_pair_tm.cuh, tnlm_pair_tmr.cuh):
//   * TMEM holds what only its own thread touches: the -ref_i windows (6 columns x 2 rows = 12 words per plane, RZ+4
//     planes) and (Z, N, b) of the 4 RZ outputs (16 words per output plane).  96 + 64 = 160 columns per thread at RZ = 4
//     (allocated as 128 + 32), 120 + 96 = 216 at RZ = 6 (128 + 128: two CTAs use all 512 columns of the SM).
//   * shared memory holds a ring of NR = RZ+4+M planes of the doubled ref_j tile instead of all RZ+4+2M: the centre row of
//     offsets first (its planes [M, M+RZ+4) are in the initial fill), then tz ascending; the slot of a dead plane is
//     refilled with cp.async M+1 pass groups before its first use.
// and two that the room so gained pays for:
//   * the 5-tap z-sums of the output planes share their pair sums (two additions per output instead of four, ZSHARE below);
//   * with two CTAs per SM (~250 registers per thread instead of 168 at three) the x-offsets go in chunks of 4-5 instead
//     of 2-3 and, where the ring fits twice (M = 2, 3), the tile is 6 planes deep.  Measured best in every shape
//     (launch_pair_tm below); the three-CTA form <2,4,3> of the 5^3 window reaches 0.427 of the FP32 roofline, <2,6,2>
//     0.473.
// The order of the passes differs from tnlm_pair5_kernel's, so the two agree to rounding, not bit for bit.
#pragma once
#include "tnlm_pair5.cuh"
#include "tnlm_pair_tmr.cuh"

namespace tnlm {

template <int M, int RZ> struct Pair5TmGeom {
    static constexpr int TX = 16, NT = 128;
    static constexpr int E = 2 * M + 1;
    static constexpr int BCOLS = TX + 2 * M + 4;
    static constexpr int BREAD = TX - 2 + 2 * (M - 1) + 8;
    static constexpr int PB2 = pitch2(cmax(BCOLS, BREAD));
    static constexpr int NPE = 16 + M, NPO = 15 + M, NPB = NPE + NPO;
    static constexpr int NAP = RZ + 4, NBP = RZ + 4 + 2 * M;
    static constexpr int NR = RZ + 4 + M;            // ring slots; the initial fill [0, NR) holds the centre window
    static constexpr int R_F2 = NR * NPB * PB2;
    static constexpr size_t BYTES = (size_t)R_F2 * sizeof(float2) + 16;
    // TMEM columns of a thread: a-planes (12 words each), then 16-word accumulator blocks Z[2] N[2] b[2] pad
    static constexpr int TM_A = 0, TM_ACC = (12 * NAP + 15) / 16 * 16, TM_END = TM_ACC + 16 * RZ;
    static constexpr int TM_COLS2 = TM_END > 128 ? (TM_END > 160 ? (TM_END > 192 ? 128 : 64) : 32) : 0;
    static_assert(TM_END <= 128 + TM_COLS2 && TM_END <= 256, "thread-private operands do not fit the CTA's TMEM columns");
    static_assert(12 * NAP <= 128 && (TM_ACC >= 128 || (128 - TM_ACC) % 16 == 0), "a block would straddle the two allocations");
};

// TMEM address of logical column c (c and the block it starts are compile-time; a block never straddles column 128)
__device__ __forceinline__ unsigned tm_at(const int c, const unsigned t1, const unsigned t2) { return c < 128 ? t1 + c : t2 + (c - 128); }

// One pass: W consecutive x-offsets at fixed (ty, tz), marching the RZ+4 planes (pair5_pass with TMEM operands and ring slots).
// ZSHARE: the z-sums of the four output planes share their pair sums (below); otherwise a four-plane ring.
template <typename G, int RZ, int W, bool CAREFUL, bool ZSHARE>
__device__ __forceinline__ unsigned pair5_pass_tm(const unsigned t1, const unsigned t2, const float2 *__restrict__ bRow,
                                                  const float c2, const unsigned mask, const int s0)
{
    constexpr int NVB = (W + 6) / 2, B_PLANE = G::NPB * G::PB2, NR = G::NR;
    static_assert(!ZSHARE || RZ % 2 == 0, "the shared z-sums pair the output planes");
    const float2 nc2 = make_float2(-c2, -c2);
    float2 zr[4][W][2];                                    // z-sum state: the last four planes' X (ring) ...
    float2 ze[2][W][2], zo[W][2], zp[W][2], zq[W][2];      // ... or the shared sums of ZSHARE (a2z below)
    float2 cand1[W + 1], cand2[W + 1];
    unsigned fail = 0u;
    float a8[2][8], a4[2][4], zn[2][8], bt[2][4];   // double-buffered TMEM loads
    tm_ld8(tm_at(G::TM_A, t1, t2), a8[0]);
    tm_ld4(tm_at(G::TM_A + 8, t1, t2), a4[0]);
#pragma unroll
    for (int p = 0; p < RZ + 4; ++p) {
        float2 b[2 * NVB];
        {
            const int sl = s0 + p;
            load_pairs<NVB>(bRow + (sl >= NR ? sl - NR : sl) * B_PLANE, b);
        }
        tm_wait_ld();
        if (p + 1 < RZ + 4) {
            tm_ld8(tm_at(G::TM_A + 12 * (p + 1), t1, t2), a8[(p + 1) & 1]);
            tm_ld4(tm_at(G::TM_A + 12 * (p + 1) + 8, t1, t2), a4[(p + 1) & 1]);
        }
        if (p + 1 >= 4 && p + 1 < RZ + 4) {
            tm_ld8(tm_at(G::TM_ACC + 16 * (p - 3), t1, t2), zn[(p + 1) & 1]);
            tm_ld4(tm_at(G::TM_ACC + 16 * (p - 3) + 8, t1, t2), bt[(p + 1) & 1]);
        }
        float2 a[6];
#pragma unroll
        for (int k = 0; k < 4; ++k) a[k] = make_float2(a8[p & 1][2 * k], a8[p & 1][2 * k + 1]);
        a[4] = make_float2(a4[p & 1][0], a4[p & 1][1]);
        a[5] = make_float2(a4[p & 1][2], a4[p & 1][3]);
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
            float (&acc)[8] = zn[p & 1];
            float (&bb)[4] = bt[p & 1];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                float2 D[W];
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    // a2z: S_o = X_o + .. + X_o+4.  ZSHARE: with the pair sums P_k = X_k + X_k+1 (k odd) and
                    // Q_k = P_k + P_k+2 the outputs (o, o+1), o even, share Q_o+1: S_o = X_o + Q_o+1 at plane o+4,
                    // S_o+1 = Q_o+1 + X_o+5 at plane o+5 -- two additions per output instead of four; direct sums, no
                    // differences.  State: the even planes' X (two alive), the last odd X, the last P, the last Q.
                    float2 S;
                    if (!ZSHARE) {
                        S = add2(add2(add2(zr[0][q][i], zr[1][q][i]), add2(zr[2][q][i], zr[3][q][i])), X[q][i]);
                    } else if ((p & 1) == 0) {
                        const float2 pn = add2(zo[q][i], X[q][i]);                        // P_p-1
                        zq[q][i] = add2(zp[q][i], pn);                                    // Q_p-3
                        zp[q][i] = pn;
                        S = add2(ze[(p >> 1) & 1][q][i], zq[q][i]);                       // X_p-4 + Q_p-3
                    } else {
                        S = add2(zq[q][i], X[q][i]);                                      // Q_p-4 + X_p
                    }
                    const float u0 = __shfl_up_sync(0xffffffffu, S.x, 1);                 // row 2l-2
                    const float u1 = __shfl_up_sync(0xffffffffu, S.y, 1);                 // row 2l-1
                    const float d0 = __shfl_down_sync(0xffffffffu, S.x, 1);               // row 2l+2
                    const float d1 = __shfl_down_sync(0xffffffffu, S.y, 1);               // row 2l+3
                    const float common = (S.x + S.y) + (u1 + d0);                         // a2y
                    D[q] = add2(make_float2(u0, d1), make_float2(common, common));
                }
                const float2 bx = make_float2(bb[2 * i], bb[2 * i + 1]);
                float2 zi = make_float2(acc[2 * i], acc[2 * i + 1]), ni = make_float2(acc[4 + 2 * i], acc[5 + 2 * i]);
                if (!CAREFUL) {
                    float2 zp = make_float2(0.f, 0.f), np = make_float2(0.f, 0.f);
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        const float2 arg = fma2(D[q], nc2, bx);                           // a3
                        const float2 u = make_float2(ex2(arg.x), ex2(arg.y));
                        zp = add2(zp, u);                                                 // a4
                        np = fma2(u, cand2[i + q], np);
                    }
                    if (fmaxf(zp.x, zp.y) <= kPairGuard) {
                        zi = add2(zi, zp);
                        ni = add2(ni, np);
                    } else {
                        fail |= 1u << (2 * (p - 4) + i);
                    }
                } else if ((mask >> (2 * (p - 4) + i)) & 1u) {
                    float2 dmin = D[0];
#pragma unroll
                    for (int q = 1; q < W; ++q) dmin = make_float2(fminf(dmin.x, D[q].x), fminf(dmin.y, D[q].y));
                    const float2 cb = make_float2(c2 * dmin.x, c2 * dmin.y);
                    const float2 nb = make_float2(bx.x - cb.x > kPairRebase ? cb.x - kPairHead : bx.x,
                                                  bx.y - cb.y > kPairRebase ? cb.y - kPairHead : bx.y);
                    const float2 sc = make_float2(ex2(0.5f * (nb.x - bx.x)), ex2(0.5f * (nb.y - bx.y)));
                    float2 zz = mul2(mul2(zi, sc), sc), nn = mul2(mul2(ni, sc), sc);
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        const float2 ar = fma2(D[q], nc2, nb);
                        const float2 u = make_float2(ex2(ar.x), ex2(ar.y));
                        zz = add2(zz, u);
                        nn = fma2(u, cand2[i + q], nn);
                    }
                    zi = zz; ni = nn;
                    bb[2 * i] = nb.x; bb[2 * i + 1] = nb.y;
                }
                acc[2 * i] = zi.x; acc[2 * i + 1] = zi.y;
                acc[4 + 2 * i] = ni.x; acc[5 + 2 * i] = ni.y;
            }
            tm_st8(tm_at(G::TM_ACC + 16 * (p - 4), t1, t2), acc);
            if (CAREFUL) tm_st4(tm_at(G::TM_ACC + 16 * (p - 4) + 8, t1, t2), bb);
        }
#pragma unroll
        for (int q = 0; q < W; ++q)
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                if (!ZSHARE) {
                    zr[0][q][i] = zr[1][q][i];
                    zr[1][q][i] = zr[2][q][i];
                    zr[2][q][i] = zr[3][q][i];
                    zr[3][q][i] = X[q][i];
                    continue;
                }
                if (p & 1) {
                    zo[q][i] = X[q][i];                                                   // the odd plane of the next P
                } else {
                    if (p == 2) zp[q][i] = add2(zo[q][i], X[q][i]);                       // P_1
                    ze[(p >> 1) & 1][q][i] = X[q][i];                                     // X_p replaces X_p-4
                }
            }
        // output x-index i, offset q reads the candidate at window element i + 2 + q of the plane two back
#pragma unroll
        for (int k = 0; k < W + 1; ++k) {
            cand2[k] = cand1[k];
            cand1[k] = b[k + 2];
        }
    }
    tm_wait_st();
    return fail;
}

template <int M, int RZ, int NCTA>
__global__ void __launch_bounds__(128, NCTA)
tnlm_pair5_tmr_kernel(const float *__restrict__ f, const float *__restrict__ g, float *f_out, const Dims dm, const int tiles_x,
                      const int tiles_y, const int tiles_z)
{
    using G = Pair5TmGeom<M, RZ>;
    constexpr int TX = 16, NR = G::NR, E = G::E;
    constexpr bool kZShare = RZ % 2 == 0;   // shared z-sums (pair5_pass_tm) wherever the output planes pair up
    constexpr bool kWide = NCTA == 2;       // two CTAs per SM have the registers for chunks of four or five x-offsets
    extern __shared__ __align__(16) float smem[];
    float2 *sBE = reinterpret_cast<float2 *>(smem);
    float2 *sBO = sBE + G::NPE * G::PB2;
    unsigned *slot = reinterpret_cast<unsigned *>(sBE + G::R_F2);

    int t = blockIdx.x;
    const int bx = t % tiles_x; t /= tiles_x;
    const int by = t % tiles_y; t /= tiles_y;
    const int bz = t % tiles_z; t /= tiles_z;
    const int ph = t;
    const int X0 = bx * TX, Y0 = by * kPair5RowsOut, Z0 = (dm.z_begin / RZ + bz) * RZ;
    const size_t V = (size_t)dm.Z * dm.Y * dm.X;
    const size_t zstride = (size_t)dm.Y * dm.X;
    const int tid = threadIdx.x;
    const int l = tid & 15;
    const int x0 = 2 * (tid >> 4);

    if (tid < 32) {
        const unsigned sa = (unsigned)__cvta_generic_to_shared(slot);
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" :: "r"(sa) : "memory");
        if (G::TM_COLS2 == 32) asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 32;" :: "r"(sa + 4) : "memory");
        if (G::TM_COLS2 == 64) asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 64;" :: "r"(sa + 4) : "memory");
        if (G::TM_COLS2 == 128) asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" :: "r"(sa + 4) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tm_base1 = slot[0], tm_base2 = G::TM_COLS2 ? slot[1] : 0u;
    const unsigned quarter = ((unsigned)(tid >> 5) * 32u) << 16;
    const unsigned t1 = tm_base1 + quarter, t2 = tm_base2 + quarter;

    {   // -ref_i windows into TMEM: rows y = Y0-2+2l+e, columns x = X0+x0-2+k (k < 6), planes z = Z0-2+p; clamp-to-edge (P4)
        const float *src = f + (size_t)ph * V;
        int xo[6], yo[2];
#pragma unroll
        for (int k = 0; k < 6; ++k) xo[k] = clampi(X0 + x0 - 2 + k, dm.X);
#pragma unroll
        for (int e = 0; e < 2; ++e) yo[e] = clampi(Y0 - 2 + 2 * l + e, dm.Y) * dm.X;
#pragma unroll
        for (int p = 0; p < G::NAP; ++p) {
            const float *sp = src + (size_t)clampi(Z0 - 2 + p, dm.Z) * zstride;
            float w8[8], w4[4];
#pragma unroll
            for (int k = 0; k < 4; ++k)
#pragma unroll
                for (int e = 0; e < 2; ++e) w8[2 * k + e] = -__ldg(sp + yo[e] + xo[k]);
#pragma unroll
            for (int k = 4; k < 6; ++k)
#pragma unroll
                for (int e = 0; e < 2; ++e) w4[2 * (k - 4) + e] = -__ldg(sp + yo[e] + xo[k]);
            tm_st8(tm_at(G::TM_A + 12 * p, t1, t2), w8);
            tm_st4(tm_at(G::TM_A + 12 * p + 8, t1, t2), w4);
        }
        tm_wait_st();
    }

    const bool vec_ok = (dm.X % 2) == 0;
    const bool col_ok = X0 + x0 < dm.X;

#pragma unroll 1
    for (int s = 0; s < 2; ++s) {
        const int j = (ph + (s ? 1 : dm.P - 1)) % dm.P;
        const float *fj = f + (size_t)j * V;
        __syncthreads();   // everyone is done with the previous direction's ring
        // initial fill: tile planes [0, NR) <-> z = Z0-2-M+pz, slot = plane; rows y = Y0-2-M+r, columns x = X0-2-M+c
        stage_pairs<G::PB2, 32 + 2 * M, G::BCOLS, NR, G::NPE, G::NPO, false, G::NT>(
            reinterpret_cast<float *>(sBE), reinterpret_cast<float *>(sBO), fj, Z0 - 2 - M, Y0 - 2 - M, X0 - 2 - M, dm, tid);
        {
            const float zero[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            const float inf4[4] = {INFINITY, INFINITY, INFINITY, INFINITY};   // first use takes the re-base path
#pragma unroll
            for (int o = 0; o < RZ; ++o) {
                tm_st8(tm_at(G::TM_ACC + 16 * o, t1, t2), zero);
                tm_st4(tm_at(G::TM_ACC + 16 * o + 8, t1, t2), inf4);
            }
            tm_wait_st();
        }
        __syncthreads();

        // one chunk of W x-offsets (starting at x-offset `start`, even) of the row of offsets (ty, tz)
        auto run_chunk = [&](auto wtag, const int start, const int ty, const int tz, const bool first) {
            constexpr int W = decltype(wtag)::value;
            const int s0 = tz % NR;
            const float2 *row = ((ty & 1) ? sBO : sBE) + (l + (ty >> 1)) * G::PB2 + x0 + start;
            unsigned fail = 0xffffffffu;   // first use: every reference exponent is still +inf
            if (!first) fail = pair5_pass_tm<G, RZ, W, false, kZShare>(t1, t2, row, dm.c2, 0u, s0);
            if (__any_sync(0xffffffffu, fail != 0u)) pair5_pass_tm<G, RZ, W, true, kZShare>(t1, t2, row, dm.c2, fail, s0);
        };
        // The rows of one tz (tz < 0: the centre row alone, first pass of the direction), CHUNK BY CHUNK: all rows with the
        // first chunk, then all rows with the second.  Row by row the two unrolled pass bodies (W = 4 and W = 3 at ten planes
        // each) evict each other from the instruction cache (stall reason no_instruction 0.9 per issued instruction at the
        // 7^3 window); chunk by chunk each body runs 2M+1 times in a row.  The chunk holding the zero x-offset goes first,
        // so that the first careful pass sets the reference exponents from the best candidates.
        auto run_rows = [&](const int tz_or_centre) {
            const bool centre = tz_or_centre < 0;
            const int tz = centre ? M : tz_or_centre;
            auto rows_of = [&](auto wtag, const int start, const bool first_chunk) {
                if (centre) {
                    run_chunk(wtag, start, M, M, first_chunk);
                } else {
#pragma unroll 1
                    for (int ty = 0; ty < E; ++ty)
                        if (!(tz == M && ty == M)) run_chunk(wtag, start, ty, tz, false);
                }
            };
            if constexpr (kWide && M == 2) {          // x-offsets 0-4
                rows_of(std::integral_constant<int, 5>{}, 0, true);
            } else if constexpr (kWide && M == 3) {   // x-offsets 0-3, 4-6
                rows_of(std::integral_constant<int, 4>{}, 0, true);
                rows_of(std::integral_constant<int, 3>{}, 4, false);
            } else if constexpr (kWide && M == 4) {   // x-offsets 4-8 (the zero offset is among them), then 0-3
                rows_of(std::integral_constant<int, 5>{}, 4, true);
                rows_of(std::integral_constant<int, 4>{}, 0, false);
            } else {                                   // chunks of 2, the last one of 3
#pragma unroll 1
                for (int cc = 0; cc < M; ++cc) {
                    const int c = (cc + M / 2) % M;
                    if (c == M - 1) rows_of(std::integral_constant<int, 3>{}, 2 * c, cc == 0);
                    else rows_of(std::integral_constant<int, 2>{}, 2 * c, cc == 0);
                }
            }
        };
        auto refill = [&](const int tz) {   // before the rows of tz >= 1: plane tz - 1 is dead, plane tz - 1 + NR takes its slot
            cp_async_wait_all();
            __syncthreads();   // the plane fetched during the previous group is visible; every warp is done with plane tz - 1
            const int pz = tz - 1 + NR;
            if (pz < G::NBP)
                stage_plane_async<G>(reinterpret_cast<float *>(sBE), reinterpret_cast<float *>(sBO),
                                     fj + (size_t)clampi(Z0 - 2 - M + pz, dm.Z) * zstride, (tz - 1) % NR, Y0 - 2 - M, X0 - 2 - M, dm, tid);
        };
        run_rows(-1);   // centre row first
#pragma unroll 1
        for (int tz = 0; tz < E; ++tz) {
            if (tz >= 1) refill(tz);
            run_rows(tz);
        }
        cp_async_wait_all();

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
        for (int o = 0; o < RZ; ++o) {
            float zn[8];
            tm_ld8(tm_at(G::TM_ACC + 16 * o, t1, t2), zn);
            tm_wait_ld();
            const bool z_ok = Z0 + o >= dm.z_begin && Z0 + o < dm.z_end;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                if (row_ok[e] && z_ok) {
                    const float n0 = __fdividef(zn[4 + e], zn[e]);
                    const float n1 = __fdividef(zn[6 + e], zn[2 + e]);
                    float *dst = f_out + base0[e] + o * zstride;
                    const bool two = X0 + x0 + 1 < dm.X;
                    if (s == 0) {
                        if (vec_ok) {
                            *reinterpret_cast<float2 *>(dst) = make_float2(n0, n1);
                        } else {
                            dst[0] = n0;
                            if (two) dst[1] = n1;
                        }
                    } else {
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
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (tid < 32) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" :: "r"(tm_base1) : "memory");
        if (G::TM_COLS2 == 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 32;" :: "r"(tm_base2) : "memory");
        if (G::TM_COLS2 == 64) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 64;" :: "r"(tm_base2) : "memory");
        if (G::TM_COLS2 == 128) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" :: "r"(tm_base2) : "memory");
    }
}

template <int M, int RZ, int NCTA>
cudaError_t launch_pair5_tmr_t(const Dims &dm, const float *f, const float *g, float *f_out, cudaStream_t st)
{
    using G = Pair5TmGeom<M, RZ>;
    static_assert(NCTA * (G::BYTES + 1024) <= 228 * 1024, "NCTA rings of the rolling pair5 kernel do not fit in shared memory");
    static_assert(NCTA * (128 + G::TM_COLS2) <= 512, "NCTA allocations do not fit the SM's 512 TMEM columns");
    static std::atomic<uint64_t> configured{0};
    cudaError_t e = ensure_dynamic_smem(tnlm_pair5_tmr_kernel<M, RZ, NCTA>, G::BYTES, configured);
    if (e != cudaSuccess) return e;
    const int tiles_x = (dm.X + 15) / 16;
    const int tiles_y = (dm.Y + kPair5RowsOut - 1) / kPair5RowsOut;
    const int tiles_z = (dm.z_end + RZ - 1) / RZ - dm.z_begin / RZ;
    const long long blocks = (long long)tiles_x * tiles_y * tiles_z * dm.P;
    if (blocks <= 0 || blocks > 2147483647LL) return cudaErrorInvalidConfiguration;
    tnlm_pair5_tmr_kernel<M, RZ, NCTA><<<(unsigned)blocks, 128, G::BYTES, st>>>(f, g, f_out, dm, tiles_x, tiles_y, tiles_z);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------
// TNLM_VARIANT_PAIRED_TMEM (ref == f): 3^3 patch: whole tile resident at M = 2 (tnlm_pair_tm_kernel), rolling window at
// M = 3, 4 (tnlm_pair_tmr_kernel); 5^3 patch: rolling window at M = 2, 3, 4 (tnlm_pair5_tmr_kernel).  The 3^3 windows
// stay on tnlm_pair_kernel / tnlm_pair5_kernel (measured: no gain there).
// 3^3 patch at M = 3, 4: two CTAs per SM, 6-plane tiles (a CTA may then take 256 TMEM columns; z-halo of the march 8/6
// instead of 6/4) and all 2M+1 x-offsets of a row in one pass (tnlm_pair_tmr.cuh).
// 5^3 patch: every shape runs TWO CTAs per SM with ~250 registers, which pays for x-offset chunks of 4-5 instead of 2-3
// (the -ref_i loads, the accumulator round trip and the guard of a pass are spread over twice the offsets) and, where the
// ring still fits twice (M = 2, 3), for 6-plane tiles (z-halo 10/6 instead of 8/4): 0.427 -> 0.474, 0.415 -> 0.468,
// 0.429 -> 0.49 of the FP32 roofline at config 5 (profiles/r02_config5_sweep.md).  Chunks: (5), (4, 3), (5, 4); chunk starts
// are even so that the LDS.128 of a row window stay aligned.
inline bool pair_tm_supported(const tnlm_params &p)
{
    return (p.patch_radius == 1 || p.patch_radius == 2) && p.search_radius >= 2 && p.search_radius <= 4;
}
inline const char *pair_tm_name(const tnlm_params &p)
{
    if (p.patch_radius == 2) {
        switch (p.search_radius) {
            case 2: return "tnlm_pair5_tmr_kernel<M=2>";
            case 3: return "tnlm_pair5_tmr_kernel<M=3>";
            default: return "tnlm_pair5_tmr_kernel<M=4>";
        }
    }
    switch (p.search_radius) {
        case 2: return "tnlm_pair_tm_kernel<M=2>";
        case 3: return "tnlm_pair_tmr_kernel<M=3>";
        default: return "tnlm_pair_tmr_kernel<M=4>";
    }
}

// ref must be f (TNLM-E)
inline cudaError_t launch_pair_tm(const tnlm_params &p, const Dims &dm, const float *f, const float *g, float *f_out,
                                  cudaStream_t st)
{
    if (p.patch_radius == 2) {
        switch (p.search_radius) {
            case 2: return launch_pair5_tmr_t<2, 6, 2>(dm, f, g, f_out, st);           // <M, RZ, CTAs per SM>
            case 3: return launch_pair5_tmr_t<3, 6, 2>(dm, f, g, f_out, st);           // deep tile: 128 + 128 TMEM columns
            case 4: return launch_pair5_tmr_t<4, 4, 2>(dm, f, g, f_out, st);
            default: return cudaErrorNotSupported;
        }
    }
    switch (p.search_radius) {
        case 2: return launch_pair_tm_t<2, 4, 16, 3, true>(dm, f, g, f_out, st);   // <M, RZ, TX, CTAs per SM, b in TMEM>
        case 3: return launch_pair_tmr_t<3, 6, 2>(dm, f, g, f_out, st);            // <M, RZ, CTAs per SM>; 256 TMEM columns
        case 4: return launch_pair_tmr_t<4, 6, 2>(dm, f, g, f_out, st);            // deep tile: 256 TMEM columns
        default: return cudaErrorNotSupported;
    }
}

}  // namespace tnlm
