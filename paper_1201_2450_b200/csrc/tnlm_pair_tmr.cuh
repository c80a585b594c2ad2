// TMEM pair kernel with a ROLLING ref_j window, for the wide search windows (d = 1, M = 3, ref == f).
//
// tnlm_pair_kernel keeps all RZ+2+2M planes of the doubled ref_j tile in shared memory, which at M = 3 leaves room for
// one 256-thread CTA per SM (8 warps) -- and a kernel bound by issue slots wants more warps than that to fill them
// (profiles/r02_issue_model.md: 0.78 slots per cycle at 8 warps against 0.91 at 12).  But a pass at z-offset tz only
// reads planes [tz, tz+RZ+2) of the tile, and the passes can be ordered by tz.  This kernel keeps a ring of
// NR = RZ+2+M planes: the centre row of offsets runs first (it sets the reference exponents, as in tnlm_pair.cuh; its
// planes [M, M+RZ+2) are in the initial fill [0, NR)), then tz = 0 .. 2M in order; when the CTA has finished the
// passes of tz, plane tz is dead and plane tz+NR is fetched into its slot with cp.async, M+1 groups of passes before
// it is first read.  With the -ref_i windows and (Z, N, b) in TMEM (tnlm_pair_tm.cuh) a CTA needs 69 KB at M = 3,
// RZ = 4: three CTAs per SM, 12 warps.  Same arithmetic per pass; the ORDER of the passes differs from
// tnlm_pair_kernel's (centre row, then tz ascending), so results agree with it to rounding, not bit for bit.
// Two CTAs per SM (NCTA = 2) are a different trade: 6-plane tiles (160 TMEM columns per thread out of an allocation of
// 256; z-halo of the march 8/6 instead of 6/4) and every x-offset of a row in one pass of 7 or 9 offsets, which ~250
// registers hold.  Fewer instructions beat the third CTA: 7^3 window 0.543 -> 0.580 of the FP32 roofline at config 4
// (<3,6,2> against <3,4,3>), 9^3 window 0.549 -> 0.609 (<4,6,2> against <4,4,2> in chunks of 4 + 5).
#pragma once
#include "tnlm_pair_tm.cuh"

namespace tnlm {

__device__ __forceinline__ void cp_async4(float *smem_dst, const float *gmem_src)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Tile geometry (PairTmGeom's for TX = 16 with (Z, N, b) in TMEM, plus the ring).  Deep tiles need more than 128 TMEM
// columns per thread (RZ = 6: 64 + 96 = 160): the CTA then allocates 256, which leaves room for two CTAs per SM.
template <int M, int RZ> struct PairTmrGeom {
    using C = Chunks<M>;
    static constexpr int TX = 16, NT = 128;
    static constexpr int E = 2 * M + 1;
    static constexpr int NVB0 = (C::W0 + 4) / 2;
    static constexpr int NVB1 = C::W1 ? (C::W1 + 4) / 2 : 0;
    static constexpr int BCOLS = TX + 2 * M + 2;
    static constexpr int BREAD = cmax(TX - 2 + 2 * NVB0, C::W1 ? TX - 2 + 4 + 2 * NVB1 : 0);
    static constexpr int PB2 = pitch2(cmax(BCOLS, BREAD));
    static constexpr int NPE = 16 + M, NPO = 15 + M, NPB = NPE + NPO;
    static constexpr int NAP = RZ + 2, NBP = RZ + 2 + 2 * M;
    static constexpr int NR = RZ + 2 + M;            // ring slots; the initial fill [0, NR) holds the centre window
    static constexpr int R_F2 = NR * NPB * PB2;
    static constexpr size_t BYTES = (size_t)R_F2 * sizeof(float2) + 16;   // + the TMEM base-address slot
    static constexpr int ACC_W = 16;                 // words per output plane: Z[2], N[2], b[2], 4 words of padding
    static constexpr int TM_A = 0, TM_ACC = 8 * NAP;
    static constexpr int TM_COLS = TM_ACC + ACC_W * RZ <= 128 ? 128 : 256;   // columns the CTA allocates
    static_assert(TM_ACC + ACC_W * RZ <= TM_COLS, "thread-private operands do not fit the CTA's TMEM columns");
};

// Fetch plane `pz` of the clamped ref_j tile (rows y = yo + r, columns x = xo + c) into ring slot `slot`, both row-pair
// copies, with 4-byte cp.async (the layout interleaves two rows per element, so nothing wider applies).
template <typename G>
__device__ __forceinline__ void stage_plane_async(float *sE, float *sO, const float *__restrict__ src_plane, const int slot,
                                                  const int yo, const int xo, const Dims &dm, const int tid)
{
    constexpr int ROWS = 32 + 2 * (G::E / 2), COLS = G::BCOLS;
    constexpr int K = (ROWS * COLS + G::NT - 1) / G::NT;
    constexpr int PLANE_F = G::NPB * G::PB2 * 2;
    float *dE = sE + slot * PLANE_F, *dO = sO + slot * PLANE_F;
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int idx = tid + k * G::NT;
        if (idx < ROWS * COLS) {
            const int r = idx / COLS, c = idx - r * COLS;
            const float *sp = src_plane + clampi(yo + r, dm.Y) * dm.X + clampi(xo + c, dm.X);
            cp_async4(dE + ((r >> 1) * G::PB2 + c) * 2 + (r & 1), sp);
            const int ro = r - 1;
            if (ro >= 0 && (ro >> 1) < G::NPO) cp_async4(dO + ((ro >> 1) * G::PB2 + c) * 2 + (ro & 1), sp);
        }
    }
    cp_async_commit();
}

template <int M, int RZ, int NCTA>
__global__ void __launch_bounds__(128, NCTA)
tnlm_pair_tmr_kernel(const float *__restrict__ f, const float *__restrict__ g, float *f_out, const Dims dm, const int tiles_x,
                     const int tiles_y, const int tiles_z)
{
    using G = PairTmrGeom<M, RZ>;
    using C = Chunks<M>;
    constexpr int TX = 16, NR = G::NR, ACC_W = G::ACC_W, E = G::E;
    // two CTAs per SM (up to 255 registers) take all 2M+1 x-offsets of a row in ONE pass: the -ref_i loads, the accumulator
    // round trip through TMEM and the guard are paid once per row instead of once per chunk of 4-5
    constexpr bool kOneChunk = NCTA == 2;
    static_assert(!kOneChunk || TX - 2 + 2 * ((E + 4) / 2) <= G::PB2, "a one-chunk row window would leave the tile row");
    constexpr int BP = G::NPB * G::PB2;
    extern __shared__ __align__(16) float smem[];
    float2 *sBE = reinterpret_cast<float2 *>(smem);
    float2 *sBO = sBE + G::NPE * G::PB2;
    unsigned *slot = reinterpret_cast<unsigned *>(sBE + G::R_F2);

    int t = blockIdx.x;
    const int bx = t % tiles_x; t /= tiles_x;
    const int by = t % tiles_y; t /= tiles_y;
    const int bz = t % tiles_z; t /= tiles_z;
    const int ph = t;
    const int X0 = bx * TX, Y0 = by * kPairRowsOut, Z0 = (dm.z_begin / RZ + bz) * RZ;
    const size_t V = (size_t)dm.Z * dm.Y * dm.X;
    const size_t zstride = (size_t)dm.Y * dm.X;
    const int tid = threadIdx.x;
    const int l = tid & 15;
    const int x0 = 2 * (tid >> 4);

    const unsigned tm_base = tm_alloc<G::TM_COLS>(slot);
    const unsigned tbase = tm_base + (((unsigned)(tid >> 5) * 32u) << 16);
    const unsigned ta = tbase + G::TM_A, tacc = tbase + G::TM_ACC;

    {   // -ref_i windows into TMEM (as tnlm_pair_tm_kernel)
        const float *src = f + (size_t)ph * V;
        int xo[4], yo[2];
#pragma unroll
        for (int k = 0; k < 4; ++k) xo[k] = clampi(X0 + x0 - 1 + k, dm.X);
#pragma unroll
        for (int e = 0; e < 2; ++e) yo[e] = clampi(Y0 - 1 + 2 * l + e, dm.Y) * dm.X;
#pragma unroll
        for (int p = 0; p < G::NAP; ++p) {
            const float *sp = src + (size_t)clampi(Z0 - 1 + p, dm.Z) * zstride;
            float w[8];
#pragma unroll
            for (int k = 0; k < 4; ++k)
#pragma unroll
                for (int e = 0; e < 2; ++e) w[2 * k + e] = -__ldg(sp + yo[e] + xo[k]);
            tm_st8(ta + 8 * p, w);
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
        // initial fill: tile planes [0, NR) <-> z = Z0-1-M+pz, slot = plane
        stage_pairs<G::PB2, 32 + 2 * M, G::BCOLS, NR, G::NPE, G::NPO, false, G::NT>(
            reinterpret_cast<float *>(sBE), reinterpret_cast<float *>(sBO), fj, Z0 - 1 - M, Y0 - 1 - M, X0 - 1 - M, dm, tid);
        {
            const float zero[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            const float inf4[4] = {INFINITY, INFINITY, INFINITY, INFINITY};
#pragma unroll
            for (int o = 0; o < RZ; ++o) {
                tm_st8(tacc + ACC_W * o, zero);
                tm_st4(tacc + ACC_W * o + 8, inf4);
            }
            tm_wait_st();
        }
        __syncthreads();

        float2 bexp[1][2];
        bexp[0][0] = bexp[0][1] = make_float2(INFINITY, INFINITY);   // (unused: the exponents live in TMEM)
        auto run_row = [&](const int ty, const int tz, const bool first) {
            const int s0 = tz % NR;                                  // slot of the march's plane 0
            const float2 *bRow = ((ty & 1) ? sBO : sBE) + (l + (ty >> 1)) * G::PB2 + x0;
            auto run_chunk = [&](auto wtag, const float2 *row, const bool frst) {
                constexpr int W = decltype(wtag)::value;
                unsigned fail = 0xffffffffu;   // first use: every reference exponent is still +inf
                if (!frst) fail = pair_pass_tm<RZ, W, false, BP, true, NR>(ta, tacc, row, dm.c2, bexp, 0u, s0);
                if (__any_sync(0xffffffffu, fail != 0u)) pair_pass_tm<RZ, W, true, BP, true, NR>(ta, tacc, row, dm.c2, bexp, fail, s0);
            };
            if constexpr (kOneChunk) {
                run_chunk(std::integral_constant<int, E>{}, bRow, first);
            } else {
                run_chunk(std::integral_constant<int, C::W0>{}, bRow, first);
                if constexpr (C::W1 > 0) run_chunk(std::integral_constant<int, C::W1>{}, bRow + 4, false);
            }
        };
        // the centre row first: the zero offset is usually the best match, so it sets the reference exponents
        run_row(M, M, true);
#pragma unroll 1
        for (int tz = 0; tz < E; ++tz) {
            if (tz >= 1) {
                cp_async_wait_all();   // the plane fetched during the previous group has landed (needed M groups from now)
                __syncthreads();       // ... for every thread, and every warp has finished the passes of tz - 1
                const int pz = tz - 1 + NR;
                if (pz < G::NBP)
                    stage_plane_async<G>(reinterpret_cast<float *>(sBE), reinterpret_cast<float *>(sBO),
                                         fj + (size_t)clampi(Z0 - 1 - M + pz, dm.Z) * zstride, (tz - 1) % NR, Y0 - 1 - M, X0 - 1 - M, dm, tid);
            }
#pragma unroll 1
            for (int ty = 0; ty < E; ++ty)
                if (!(tz == M && ty == M)) run_row(ty, tz, false);
        }
        cp_async_wait_all();

        // epilogue (as tnlm_pair_tm_kernel): rows 2l (.x) and 2l+1 (.y); tile rows 1..30 are outputs
        bool row_ok[2];
        size_t base0[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int r = 2 * l + e, y = Y0 - 1 + r;
            row_ok[e] = r >= 1 && r <= kPairRowsOut && y < dm.Y && col_ok;
            base0[e] = (size_t)ph * V + ((size_t)Z0 * dm.Y + min(y, dm.Y - 1)) * dm.X + X0 + x0;
        }
#pragma unroll
        for (int o = 0; o < RZ; ++o) {
            float zn[8];
            tm_ld8(tacc + ACC_W * o, zn);
            tm_wait_ld();
            const bool z_ok = Z0 + o >= dm.z_begin && Z0 + o < dm.z_end;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                if (row_ok[e] && z_ok) {
                    const float n0 = __fdividef(zn[4 + e], zn[e]);
                    const float n1 = __fdividef(zn[6 + e], zn[2 + e]);
                    float *dst = f_out + base0[e] + o * zstride;
                    if (s == 0) {
                        if (vec_ok) {
                            *reinterpret_cast<float2 *>(dst) = make_float2(n0, n1);
                        } else {
                            dst[0] = n0;
                            if (X0 + x0 + 1 < dm.X) dst[1] = n1;
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
                            if (X0 + x0 + 1 < dm.X) dst[1] = fmaf(dm.a_g, __ldg(gp + 1), dm.a_n * (dst[1] + n1));
                        }
                    }
                }
            }
        }
    }
    tm_free<G::TM_COLS>(tm_base);
}

template <int M, int RZ, int NCTA>
cudaError_t launch_pair_tmr_t(const Dims &dm, const float *f, const float *g, float *f_out, cudaStream_t st)
{
    using G = PairTmrGeom<M, RZ>;
    static_assert(NCTA * (G::BYTES + 1024) <= 228 * 1024, "NCTA rings of the rolling pair kernel do not fit in shared memory");
    static_assert(NCTA * G::TM_COLS <= 512, "NCTA allocations do not fit the SM's 512 TMEM columns");
    static std::atomic<uint64_t> configured{0};
    cudaError_t e = ensure_dynamic_smem(tnlm_pair_tmr_kernel<M, RZ, NCTA>, G::BYTES, configured);
    if (e != cudaSuccess) return e;
    const int tiles_x = (dm.X + 15) / 16;
    const int tiles_y = (dm.Y + kPairRowsOut - 1) / kPairRowsOut;
    const int tiles_z = (dm.z_end + RZ - 1) / RZ - dm.z_begin / RZ;
    const long long blocks = (long long)tiles_x * tiles_y * tiles_z * dm.P;
    if (blocks <= 0 || blocks > 2147483647LL) return cudaErrorInvalidConfiguration;
    tnlm_pair_tmr_kernel<M, RZ, NCTA><<<(unsigned)blocks, 128, G::BYTES, st>>>(f, g, f_out, dm, tiles_x, tiles_y, tiles_z);
    return cudaGetLastError();
}

}  // namespace tnlm
