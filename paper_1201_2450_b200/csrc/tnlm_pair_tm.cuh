// Row-pair packed sweep kernel for 3^3 patches (d = 1, ref == f) with the thread-private operands in tensor
// memory (TMEM).
//
// The arithmetic is tnlm_pair.cuh's (same passes, same reference-exponent scheme, same order of operations inside a
// pass); what changes is where the thread-private arrays live.  In tnlm_pair_kernel the -ref_i tile sits in shared
// memory although a thread only ever reads its own four columns of its own row pair from it (the same 8 words per
// plane in every one of the 2 x (2M+1)^2 passes), and (Z, N, reference exponent) of all outputs sit in registers
// although a pass touches those of one plane at a time.  Blackwell's 256 KB of tensor memory per SM is addressed as
// 128 lanes x 512 columns of 32-bit words, and a warp's tcgen05.ld / tcgen05.st .32x32b moves "lane = thread, n
// consecutive columns" between it and registers: a per-thread scratch array that costs neither shared-memory
// capacity, nor LDS wavefronts, nor registers.  No tcgen05.mma is issued (the path is not a contraction, DESIGN.md
// section 5); TMEM is storage only.
//
//   TMEM columns of a thread (the CTA allocates 128 columns per four warps; 3 CTAs per SM use 384 of the 512)
//     [0, 8(RZ+2))        plane p -> -ref_i as float2 a[4] (columns x0-1 .. x0+2 of row pair l)
//     [8(RZ+2), ...)      output plane o -> 16 words: Z[2], N[2] as float2 (index = x of the run; .x = row 2l,
//                         .y = row 2l+1), then the reference exponents b[2] (BTM) and 4 words of padding
//   registers             z-ring, row windows, the pass's partial sums (and b if not BTM)
//   shared memory         the ref_j tiles BE / BO only (layout of tnlm_pair.cuh)
//
// What it buys (profiles/r02_*): the sweep is bound by issue slots -- a packed FP32 instruction holds the issue port
// for two cycles and nothing issues in its shadow -- and with 48 accumulator registers and a
// third of the LDS.128 gone the same instruction stream issues at 91 % of that bound instead of 86 %.
#pragma once
#include "tnlm_pair.cuh"

namespace tnlm {

__device__ __forceinline__ void tm_ld8(const unsigned addr, float (&r)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7])
                 : "r"(addr));
}
__device__ __forceinline__ void tm_st8(const unsigned addr, const float (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "r"(addr), "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]), "f"(r[4]), "f"(r[5]), "f"(r[6]), "f"(r[7]));
}
// the loaded registers may be read only after wait::ld; a location may be re-read only after wait::st of its store
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;"); }

constexpr int kTmColsPerThread = 128;   // columns of a thread's scratch block

__device__ __forceinline__ void tm_ld4(const unsigned addr, float (&r)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void tm_st4(const unsigned addr, const float (&r)[4])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};"
                 :: "r"(addr), "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]));
}

// Warp 0 allocates the CTA's columns (a power of two >= 32) and publishes the base address through shared memory.
template <int kTmCols>
__device__ __forceinline__ unsigned tm_alloc(unsigned *slot)
{
    if (threadIdx.x < 32) {
        const unsigned sa = (unsigned)__cvta_generic_to_shared(slot);
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(sa), "n"(kTmCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    return *slot;
}
template <int kTmCols>
__device__ __forceinline__ void tm_free(const unsigned base)
{
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (threadIdx.x < 32)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(base), "n"(kTmCols) : "memory");
}

template <int M, int RZ, int TX_, bool BTM> struct PairTmGeom {
    using C = Chunks<M>;
    static constexpr int TX = TX_;                   // 16: four warps (one TMEM lane quarter each); 32: eight warps (two column blocks)
    static constexpr int E = 2 * M + 1;
    static constexpr int NT = TX * 8;
    static_assert(TX == 16 || TX == 32, "a CTA is one or two warps per TMEM lane quarter");
    static constexpr int NVB0 = (C::W0 + 4) / 2;
    static constexpr int NVB1 = C::W1 ? (C::W1 + 4) / 2 : 0;
    static constexpr int BCOLS = TX + 2 * M + 2;
    static constexpr int BREAD = cmax(TX - 2 + 2 * NVB0, C::W1 ? TX - 2 + 4 + 2 * NVB1 : 0);
    static constexpr int PB2 = pitch2(cmax(BCOLS, BREAD));
    static constexpr int NPE = 16 + M, NPO = 15 + M, NPB = NPE + NPO;
    static constexpr int NAP = RZ + 2, NBP = RZ + 2 + 2 * M;
    static constexpr int B_F2 = NBP * NPB * PB2;
    static constexpr size_t BYTES = (size_t)B_F2 * sizeof(float2) + 16;   // + the TMEM base-address slot
    static constexpr int ACC_W = BTM ? 16 : 8;       // words per output plane: Z[2], N[2] (and b[2] + 4 words of padding)
    static constexpr int TM_A = 0, TM_ACC = 8 * NAP;
    static constexpr int TM_COLS = (NT / 128) * kTmColsPerThread;   // columns the CTA allocates
    static_assert(TM_ACC + ACC_W * RZ <= kTmColsPerThread, "thread-private operands do not fit the thread's TMEM columns");
};

// One pass (W consecutive x-offsets at fixed (ty, tz), marching the RZ+2 planes): pair_pass of tnlm_pair.cuh with
// the -ref_i windows and the (Z, N) sums in TMEM.  ta / tz: TMEM addresses of the thread's a-block / accumulator block.
// NR > 0: the ref_j planes live in a ring of NR shared-memory slots, plane p of the march in slot (s0 + p) mod NR.
template <int RZ, int W, bool CAREFUL, int B_PLANE, bool BTM, int NR = 0>
__device__ __forceinline__ unsigned pair_pass_tm(const unsigned ta, const unsigned tacc, const float2 *__restrict__ bRow,
                                                 const float c2, float2 (&bexp)[BTM ? 1 : RZ][2], const unsigned mask,
                                                 const int s0 = 0)
{
    constexpr int ACC_W = BTM ? 16 : 8;
    constexpr int NVB = (W + 4) / 2;
    const float2 nc2 = make_float2(-c2, -c2);
    float2 ring0[W][2], ring1[W][2];
    float2 bprev[2 * NVB];
    unsigned fail = 0u;
    float av[2][8], zn[2][8], bt[2][4];   // double-buffered TMEM loads: the loads of plane p+1 are in flight during plane p
    tm_ld8(ta, av[0]);
#pragma unroll
    for (int p = 0; p < RZ + 2; ++p) {
        float2 b[2 * NVB];
        if constexpr (NR == 0) {
            load_pairs<NVB>(bRow + p * B_PLANE, b);
        } else {
            const int sl = s0 + p;
            load_pairs<NVB>(bRow + (sl >= NR ? sl - NR : sl) * B_PLANE, b);
        }
        tm_wait_ld();
        if (p + 1 < RZ + 2) tm_ld8(ta + 8 * (p + 1), av[(p + 1) & 1]);
        if (p + 1 >= 2 && p + 1 < RZ + 2) {
            tm_ld8(tacc + ACC_W * (p - 1), zn[(p + 1) & 1]);
            if (BTM) tm_ld4(tacc + ACC_W * (p - 1) + 8, bt[(p + 1) & 1]);
        }
        const float (&aw)[8] = av[p & 1];
        float2 X[W][2];
#pragma unroll
        for (int q = 0; q < W; ++q) {
            float2 d[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) d[k] = add2(b[k + q], make_float2(aw[2 * k], aw[2 * k + 1]));   // a1 (a is -ref_i)
            const float2 mid = fma2(d[2], d[2], mul2(d[1], d[1]));                                       // a2x
            X[q][0] = fma2(d[0], d[0], mid);
            X[q][1] = fma2(d[3], d[3], mid);
        }
        if (p >= 2) {
            float (&acc)[8] = zn[p & 1];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                float2 D[W];
#pragma unroll
                for (int q = 0; q < W; ++q) {
                    float2 S;
                    if ((p & 1) == 0) {
                        ring1[q][i] = add2(ring1[q][i], X[q][i]);
                        S = add2(ring0[q][i], ring1[q][i]);
                    } else {
                        S = add2(ring0[q][i], X[q][i]);
                    }
                    const float own = S.x + S.y;
                    const float up = __shfl_up_sync(0xffffffffu, S.y, 1);
                    const float dn = __shfl_down_sync(0xffffffffu, S.x, 1);
                    D[q] = add2(make_float2(up, dn), make_float2(own, own));
                }
                float2 bx = BTM ? make_float2(bt[p & 1][2 * i], bt[p & 1][2 * i + 1]) : bexp[BTM ? 0 : p - 2][i];
                float2 zi = make_float2(acc[2 * i], acc[2 * i + 1]), ni = make_float2(acc[4 + 2 * i], acc[5 + 2 * i]);
                if (!CAREFUL) {
                    float2 zp = make_float2(0.f, 0.f), np = make_float2(0.f, 0.f);
#pragma unroll
                    for (int q = 0; q < W; ++q) {
                        const float2 arg = fma2(D[q], nc2, bx);
                        const float2 u = make_float2(ex2(arg.x), ex2(arg.y));
                        zp = add2(zp, u);
                        np = fma2(u, bprev[i + 1 + q], np);
                    }
                    if (fmaxf(zp.x, zp.y) <= kPairGuard) {
                        zi = add2(zi, zp);
                        ni = add2(ni, np);
                    } else {
                        fail |= 1u << (2 * (p - 2) + i);
                    }
                } else if ((mask >> (2 * (p - 2) + i)) & 1u) {
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
                        nn = fma2(u, bprev[i + 1 + q], nn);
                    }
                    zi = zz; ni = nn; bx = nb;
                    if (BTM) { bt[p & 1][2 * i] = nb.x; bt[p & 1][2 * i + 1] = nb.y; } else { bexp[BTM ? 0 : p - 2][i] = nb; }
                }
                acc[2 * i] = zi.x; acc[2 * i + 1] = zi.y;
                acc[4 + 2 * i] = ni.x; acc[5 + 2 * i] = ni.y;
            }
            tm_st8(tacc + ACC_W * (p - 2), acc);
            if (BTM && CAREFUL) tm_st4(tacc + ACC_W * (p - 2) + 8, bt[p & 1]);
        }
#pragma unroll
        for (int q = 0; q < W; ++q)
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                ring0[q][i] = ring1[q][i];
                ring1[q][i] = X[q][i];
            }
#pragma unroll
        for (int k = 0; k < 2 * NVB; ++k) bprev[k] = b[k];
    }
    tm_wait_st();   // the next pass (or the epilogue) reads these sums back
    return fail;
}

template <int M, int RZ, int TX_, int NCTA, bool BTM>
__global__ void __launch_bounds__(PairTmGeom<M, RZ, TX_, BTM>::NT, NCTA)
tnlm_pair_tm_kernel(const float *__restrict__ f, const float *__restrict__ g, float *f_out, const Dims dm,
                    const int tiles_x, const int tiles_y, const int tiles_z)
{
    using G = PairTmGeom<M, RZ, TX_, BTM>;
    using C = Chunks<M>;
    constexpr int TX = G::TX;
    constexpr int ACC_W = G::ACC_W;
    constexpr int BP = G::NPB * G::PB2;
    extern __shared__ __align__(16) float smem[];
    float2 *sBE = reinterpret_cast<float2 *>(smem);
    float2 *sBO = sBE + G::NPE * G::PB2;
    unsigned *slot = reinterpret_cast<unsigned *>(sBE + G::B_F2);

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
    // warp w: lane quarter w % 4, column block w / 4
    const unsigned tbase = tm_base + ((((unsigned)(tid >> 5) & 3u) * 32u) << 16) + (unsigned)(tid >> 7) * kTmColsPerThread;
    const unsigned ta = tbase + G::TM_A, tacc = tbase + G::TM_ACC;

    // -ref_i windows straight from global memory into TMEM (clamp-to-edge, reading P4): rows y = Y0-1+2l+e,
    // columns x = X0+x0-1+k, planes z = Z0-1+p
    {
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
        __syncthreads();
        stage_pairs<G::PB2, 32 + 2 * M, G::BCOLS, G::NBP, G::NPE, G::NPO, false, G::NT>(
            reinterpret_cast<float *>(sBE), reinterpret_cast<float *>(sBO), f + (size_t)j * V, Z0 - 1 - M, Y0 - 1 - M,
            X0 - 1 - M, dm, tid);
        {
            const float zero[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            const float inf4[4] = {INFINITY, INFINITY, INFINITY, INFINITY};
#pragma unroll
            for (int o = 0; o < RZ; ++o) {
                tm_st8(tacc + ACC_W * o, zero);
                if (BTM) tm_st4(tacc + ACC_W * o + 8, inf4);
            }
            tm_wait_st();
        }
        __syncthreads();

        float2 bexp[BTM ? 1 : RZ][2];
#pragma unroll
        for (int o = 0; o < (BTM ? 1 : RZ); ++o)
#pragma unroll
            for (int i = 0; i < 2; ++i) bexp[o][i] = make_float2(INFINITY, INFINITY);   // first use takes the re-base path
        auto run_chunk = [&](auto wtag, const float2 *bRow, const bool first) {
            constexpr int W = decltype(wtag)::value;
            unsigned fail = 0xffffffffu;
            if (!first) fail = pair_pass_tm<RZ, W, false, BP, BTM>(ta, tacc, bRow, dm.c2, bexp, 0u);
            if (__any_sync(0xffffffffu, fail != 0u)) pair_pass_tm<RZ, W, true, BP, BTM>(ta, tacc, bRow, dm.c2, bexp, fail);
        };
#pragma unroll 1
        for (int k = 0; k < G::E * G::E; ++k) {
            const int kk = (k + (G::E * G::E) / 2) % (G::E * G::E);
            const int tz = kk / G::E, ty = kk % G::E;
            const float2 *bRow = ((ty & 1) ? sBO : sBE) + (tz * G::NPB + l + (ty >> 1)) * G::PB2 + x0;
            run_chunk(std::integral_constant<int, C::W0>{}, bRow, k == 0);
            if constexpr (C::W1 > 0) run_chunk(std::integral_constant<int, C::W1>{}, bRow + 4, false);
        }

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
                    // words: Z[i].x Z[i].y at 2i, 2i+1; N[i] at 4+2i, 5+2i; .x = row 2l (e = 0), .y = row 2l+1
                    const float n0 = __fdividef(zn[4 + e], zn[e]);
                    const float n1 = __fdividef(zn[6 + e], zn[2 + e]);
                    float *dst = f_out + base0[e] + o * zstride;
                    if (s == 0) {
                        // park NLM- in f_out; the same thread reads it back after the second direction
                        if (vec_ok) {
                            *reinterpret_cast<float2 *>(dst) = make_float2(n0, n1);
                        } else {
                            dst[0] = n0;
                            if (X0 + x0 + 1 < dm.X) dst[1] = n1;
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
                            if (X0 + x0 + 1 < dm.X) dst[1] = fmaf(dm.a_g, __ldg(gp + 1), dm.a_n * (dst[1] + n1));
                        }
                    }
                }
            }
        }
    }
    tm_free<G::TM_COLS>(tm_base);
}

template <int M, int RZ, int TX_, int NCTA, bool BTM>
cudaError_t launch_pair_tm_t(const Dims &dm, const float *f, const float *g, float *f_out, cudaStream_t st)
{
    using G = PairTmGeom<M, RZ, TX_, BTM>;
    static_assert(NCTA * (G::BYTES + 1024) <= 228 * 1024, "NCTA tiles of the TMEM pair kernel do not fit in shared memory");
    static_assert(NCTA * G::TM_COLS <= 512, "NCTA allocations do not fit the SM's 512 TMEM columns");
    static std::atomic<uint64_t> configured{0};
    cudaError_t e = ensure_dynamic_smem(tnlm_pair_tm_kernel<M, RZ, TX_, NCTA, BTM>, G::BYTES, configured);
    if (e != cudaSuccess) return e;
    const int tiles_x = (dm.X + G::TX - 1) / G::TX;
    const int tiles_y = (dm.Y + kPairRowsOut - 1) / kPairRowsOut;
    const int tiles_z = (dm.z_end + RZ - 1) / RZ - dm.z_begin / RZ;
    const long long blocks = (long long)tiles_x * tiles_y * tiles_z * dm.P;
    if (blocks <= 0 || blocks > 2147483647LL) return cudaErrorInvalidConfiguration;
    tnlm_pair_tm_kernel<M, RZ, TX_, NCTA, BTM><<<(unsigned)blocks, G::NT, G::BYTES, st>>>(f, g, f_out, dm, tiles_x, tiles_y, tiles_z);
    return cudaGetLastError();
}

}  // namespace tnlm
