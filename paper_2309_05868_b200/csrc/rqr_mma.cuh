// rqr_mma.cuh -- device building blocks shared by the FP64 DMMA kernels (rqr_tall_mma.cu: n <= 64,
// rqr_tall_panel.cu: 64 < n <= 256): PTX helpers (mma.sync m8n8k4.f64, mbarrier, bulk async copy),
// triangular-factor B fragments, the per-warp blocked substitution on 8 column blocks, the swizzled
// Gram staging block and the per-warp landing ring.
#pragma once
#include "rqr_common.cuh"
#include "rqr_tall.cuh"
#include <type_traits>

#ifndef GRAM_WARPS
#define GRAM_WARPS 8      // A4: 248 registers/thread (36 Gram accumulators) => 8 warps per SM
#endif
#ifndef GRAM_STAGES
#define GRAM_STAGES 3
#endif
#ifndef APPLY_WARPS
#define APPLY_WARPS 12    // A6: ~90 registers/thread
#endif
#ifndef APPLY_STAGES
#define APPLY_STAGES 2
#endif
#define LDL_PAD 8         // landing rows: LD = n8 + 8  (conflict-free 128-bit C-fragment reads)

// ------------------------------------------------------------------------------------------
// PTX helpers
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
                 :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        :: "r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        :: "r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// ------------------------------------------------------------------------------------------
// Triangular-factor fragments in shared memory, built by every CTA in its prologue:
//   Tf [J][s][lane]      = T_J[2(lane%4) + s][lane/4],     T_J = inv(R[J,J])   (B fragments)
//   nRf[p(J,J')][s][lane] = -R[8J + 2(lane%4) + s][8J' + lane/4],  J < J'
// R is n x n; columns/rows >= n are padded with the identity.
// ------------------------------------------------------------------------------------------
template <int NB>
struct TriFrags {
    static constexpr int NPAIR = NB * (NB - 1) / 2;
    static constexpr int DOUBLES = NB * 64 + NPAIR * 64;
    __device__ static int pair(int J, int Jp) { return J * NB - J * (J + 1) / 2 + (Jp - J - 1); }
};

__device__ __forceinline__ double r_padded(const double* __restrict__ R, int n, int i, int c)
{
    return (i < n && c < n) ? __ldg(R + i * n + c) : ((i == c) ? 1.0 : 0.0);
}

// `stage`: (8 NB)^2 doubles of shared memory that are free in the prologue (the callers pass their landing ring
// and zero it afterwards).  The diagonal panel of R is staged there with coalesced loads first, so the back
// substitution (64 threads, a dependent chain) and the fragment fills read shared memory instead of L2, and the
// divisions by the diagonal are 8 independent reciprocals up front: 11 -> 3 us of prologue at n = 64.
template <int NB>
__device__ void build_tri_frags(const double* __restrict__ R, int n, double* __restrict__ Tf,
                                double* __restrict__ nRf, double* __restrict__ scratch /* NB*64 */,
                                double* __restrict__ stage /* (8 NB)^2 */,
                                int base = 0 /* first row/column of the diagonal panel */)
{
    constexpr int N = 8 * NB;
    const int tid = threadIdx.x;
#pragma unroll 4
    for (int t = tid; t < N * N; t += blockDim.x) {                 // unrolled: 4 loads of L2 latency in flight
        const int i = t / N, c = t - i * N;
        stage[t] = r_padded(R, n, base + i, base + c);
    }
    __syncthreads();
    // T_J column c by back substitution: R_JJ t = e_c  (one thread per (J, c))
    for (int t = tid; t < NB * 8; t += blockDim.x) {
        const int J = t >> 3, c = t & 7;
        const double* D = stage + (8 * J) * N + 8 * J;
        double rinv[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) rinv[i] = 1.0 / D[i * N + i];
        double tc[8];
#pragma unroll
        for (int i = 7; i >= 0; --i) {
            double s = (i == c) ? 1.0 : 0.0;
#pragma unroll
            for (int k = 7; k > i; --k) s = fma(-D[i * N + k], tc[k], s);
            tc[i] = (i <= c) ? s * rinv[i] : 0.0;
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) scratch[J * 64 + i * 8 + c] = tc[i];
    }
    __syncthreads();
    for (int t = tid; t < NB * 64; t += blockDim.x) {
        const int J = t >> 6, h = (t >> 5) & 1, lane = t & 31;
        Tf[t] = scratch[J * 64 + (2 * (lane & 3) + h) * 8 + (lane >> 2)];
    }
    for (int t = tid; t < TriFrags<NB>::NPAIR * 64; t += blockDim.x) {
        const int p = t >> 6, h = (t >> 5) & 1, lane = t & 31;
        // invert p -> (J, J')
        int J = 0, rem = p;
        while (rem >= NB - 1 - J) { rem -= NB - 1 - J; ++J; }
        const int Jp = J + 1 + rem;
        nRf[t] = -stage[(8 * J + 2 * (lane & 3) + h) * N + 8 * Jp + (lane >> 2)];
    }
    __syncthreads();
}

// ------------------------------------------------------------------------------------------
// xs: per-warp 8 x N8 block, 16-byte units XOR-swizzled by g(r) = 4 (r&1) + (r&2).
// Element (r, c) lives at r*LD + (((c>>1) ^ g(r)) << 1) + (c&1), LD = N8 rounded up to 16.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int xs_swz(int r) { return ((r & 1) << 2) | (r & 2); }

template <int N8>
struct XsAddr {
    // the XOR swizzle permutes the 8 units of a 16-double group, so a row occupies a multiple of 16 doubles
    // (odd column-block counts leave 8 pad doubles per row that are never read)
    static constexpr int LD = (N8 + 15) & ~15;
    int c_base;   // C fragment of block J:  c_base + ((8J) ^ c_x)      (double2)
    int c_x;
    int a_base;   // A fragment (J, h):      a_base + ((8J + 4h) ^ a_x)
    int a_x;
    int g_base[2];// Gram fragment (h, a):   g_base[h] + ((8a) ^ g_x[h])
    int g_x[2];
    __device__ __forceinline__ explicit XsAddr(int lane)
    {
        const int r = lane >> 2, q = lane & 3;
        // C: (r, 8J + 2q): unit 4J + q ^ g(r)
        c_base = r * LD; c_x = ((q ^ xs_swz(r)) << 1);
        // A: (r, 8J + 4h + q): unit (4J + 2h + (q>>1)) ^ g(r), word q&1
        a_base = r * LD + (q & 1); a_x = (((q >> 1) ^ xs_swz(r)) << 1);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            // Gram: (row 4h + q, col 8a + r): unit (4a + (r>>1)) ^ g(row), word r&1
            const int row = 4 * h + q;
            g_base[h] = row * LD + (r & 1); g_x[h] = (((r >> 1) ^ xs_swz(row)) << 1);
        }
    }
    __device__ __forceinline__ int c(int J) const { return c_base + ((8 * J) ^ c_x); }
    __device__ __forceinline__ int a(int J, int h) const { return a_base + ((8 * J + 4 * h) ^ a_x); }
    __device__ __forceinline__ int g(int h, int a_) const { return g_base[h] + ((8 * a_) ^ g_x[h]); }
};

// t-th Gram DMMA of a row-block, t in [0, 2*NBLK): slab h = t / NBLK, then (a, b), a <= b, row-major
template <int NB>
__device__ __forceinline__ constexpr int gram_a(int t)
{
    int rem = t % (NB * (NB + 1) / 2), a = 0;
    while (rem >= NB - a) { rem -= NB - a; ++a; }
    return a;
}
template <int NB>
__device__ __forceinline__ constexpr int gram_b(int t)
{
    int rem = t % (NB * (NB + 1) / 2), a = 0;
    while (rem >= NB - a) { rem -= NB - a; ++a; }
    return a + rem;
}

template <int I, int N, class F>
__device__ __forceinline__ void static_for(F&& f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

// Gram DMMAs [T0, T1) of the row-block held in xsp; g = fragment registers carried across calls.
template <int NB, int N8, int T0, int T1>
__device__ __forceinline__ void gram_chunk(const double* __restrict__ xsp, const XsAddr<N8>& ad,
                                           double (&g)[NB], double (&G)[NB * (NB + 1) / 2][2])
{
    constexpr int NBLK = NB * (NB + 1) / 2;
    static_for<T0, T1>([&](auto tc) {
        constexpr int t = decltype(tc)::value;
        if constexpr (t % NBLK == 0) {
            constexpr int h = t / NBLK;
#pragma unroll
            for (int a_ = 0; a_ < NB; ++a_) g[a_] = xsp[ad.g(h, a_)];
        }
        constexpr int idx = t % NBLK;
        dmma(G[idx][0], G[idx][1], g[gram_a<NB>(t)], g[gram_b<NB>(t)]);
    });
}

// ------------------------------------------------------------------------------------------
// One 8-row block:  X = A R^-1 by blocked substitution (DMMA), A given as C fragments in acc; on
// return acc holds X (C fragments).  X is also written (swizzled) to xsc if XS, and to global
// memory if gout != nullptr.  When GRAM is set the NB+1 Gram DMMAs per step of the PREVIOUS
// row-block (held in xsp) are issued in four groups placed in the dependent-issue gaps of the
// chain  T(s=0) -> T(s=1) -> U(J+1, s=0) -> U(J+1, s=1) -> next step.
// The arithmetic on (acc, Tf, nRf) is the same instruction sequence for every caller (H1).
// ------------------------------------------------------------------------------------------
// Per-lane output state of a row-block: gp = address of (row r, column 2q) in the output or
// nullptr when this lane's row is not stored; colmask bit 2J = "columns 8J+2q and 8J+2q+1 both
// exist", bit 2J+1 = "column 8J+2q exists" (computed once per kernel by col_mask()).
template <int NB>
__device__ __forceinline__ uint32_t col_mask(int n, int lane)
{
    uint32_t msk = 0;
#pragma unroll
    for (int J = 0; J < NB; ++J) {
        const int c = 8 * J + 2 * (lane & 3);
        msk |= (uint32_t)(c + 1 < n) << (2 * J);
        msk |= (uint32_t)(c < n) << (2 * J + 1);
    }
    return msk;
}

// `after_first` runs once after step 0 has issued its updates: every acc register loaded from the
// landing block has been consumed by a DMMA by then, so the hook may refill that block.
template <int NB, bool GRAM, bool XS, bool FULL, class Hook>
__device__ __forceinline__ void trsm_rowblock(double (&acc)[NB][2], double* __restrict__ xsc,
                                              const double* __restrict__ xsp,
                                              const XsAddr<8 * NB>& ad, const double* __restrict__ Tf,
                                              const double* __restrict__ nRf, double* __restrict__ gp,
                                              uint32_t colmask, int lane,
                                              double (&g)[NB], double (&G)[NB * (NB + 1) / 2][2],
                                              Hook&& after_first)
{
    constexpr int N8 = 8 * NB;
    constexpr int GP = NB + 1;                       // Gram DMMAs per step
    constexpr int E1 = GP / 4, E2 = GP / 2, E3 = (3 * GP) / 4;
    static_for<0, NB>([&](auto Jc) {
        constexpr int J = decltype(Jc)::value;
        double x0 = 0.0, x1 = 0.0;
        dmma(x0, x1, acc[J][0], Tf[J * 64 + lane]);
        if constexpr (GRAM) gram_chunk<NB, N8, J * GP, J * GP + E1>(xsp, ad, g, G);
        dmma(x0, x1, acc[J][1], Tf[J * 64 + 32 + lane]);
        if constexpr (GRAM) gram_chunk<NB, N8, J * GP + E1, J * GP + E2>(xsp, ad, g, G);
#pragma unroll
        for (int Jp = J + 1; Jp < NB; ++Jp)
            dmma(acc[Jp][0], acc[Jp][1], x0, nRf[TriFrags<NB>::pair(J, Jp) * 64 + lane]);
        if constexpr (GRAM) gram_chunk<NB, N8, J * GP + E2, J * GP + E3>(xsp, ad, g, G);
#pragma unroll
        for (int Jp = J + 1; Jp < NB; ++Jp)
            dmma(acc[Jp][0], acc[Jp][1], x1, nRf[TriFrags<NB>::pair(J, Jp) * 64 + 32 + lane]);
        acc[J][0] = x0; acc[J][1] = x1;
        if constexpr (J == 0) after_first();
        if constexpr (GRAM) gram_chunk<NB, N8, J * GP + E3, (J + 1) * GP>(xsp, ad, g, G);
        // stores last: x has long been produced, the warp does not stall on the DMMA result
        if constexpr (XS) *reinterpret_cast<double2*>(xsc + ad.c(J)) = make_double2(x0, x1);
        if (gp != nullptr) {
            if (FULL || ((colmask >> (2 * J)) & 1u)) *reinterpret_cast<double2*>(gp + 8 * J) = make_double2(x0, x1);
            else if ((colmask >> (2 * J + 1)) & 1u) gp[8 * J] = x0;
        }
    });
    if constexpr (XS) __syncwarp();
}

// The same routine (same instruction sequence on acc, Tf, nRf: H1) with the interleaved independent
// work given as a functor: gf.template chunk<J, PART>() is called at the four gaps of step J.
template <int NB, bool XS, bool FULL, class Hook, class GF>
__device__ __forceinline__ void trsm_rowblock_gf(double (&acc)[NB][2], double* __restrict__ xsc,
                                                 const XsAddr<8 * NB>& ad, const double* __restrict__ Tf,
                                                 const double* __restrict__ nRf, double* __restrict__ gp,
                                                 uint32_t colmask, int lane, Hook&& after_first, GF&& gf)
{
    static_for<0, NB>([&](auto Jc) {
        constexpr int J = decltype(Jc)::value;
        double x0 = 0.0, x1 = 0.0;
        dmma(x0, x1, acc[J][0], Tf[J * 64 + lane]);
        gf.template chunk<J, 0>();
        dmma(x0, x1, acc[J][1], Tf[J * 64 + 32 + lane]);
        gf.template chunk<J, 1>();
#pragma unroll
        for (int Jp = J + 1; Jp < NB; ++Jp)
            dmma(acc[Jp][0], acc[Jp][1], x0, nRf[TriFrags<NB>::pair(J, Jp) * 64 + lane]);
        gf.template chunk<J, 2>();
#pragma unroll
        for (int Jp = J + 1; Jp < NB; ++Jp)
            dmma(acc[Jp][0], acc[Jp][1], x1, nRf[TriFrags<NB>::pair(J, Jp) * 64 + 32 + lane]);
        acc[J][0] = x0; acc[J][1] = x1;
        if constexpr (J == 0) after_first();
        gf.template chunk<J, 3>();
        if constexpr (XS) *reinterpret_cast<double2*>(xsc + ad.c(J)) = make_double2(x0, x1);
        if (gp != nullptr) {
            if (FULL || ((colmask >> (2 * J)) & 1u)) *reinterpret_cast<double2*>(gp + 8 * J) = make_double2(x0, x1);
            else if ((colmask >> (2 * J + 1)) & 1u) gp[8 * J] = x0;
        }
    });
    if constexpr (XS) __syncwarp();
}

// Two row-blocks through the same triangular factor at once (A6): every B fragment (T_J, -R[J,J']) is read from
// shared memory ONCE for both, and the warp carries two independent substitution chains, so a dependent DMMA of one
// chain issues in the shadow of the other's.  The arithmetic on each row-block is the instruction sequence of
// trsm_rowblock (H1: same bits); which blocks are paired does not enter it.
template <int NB, bool FULL, class Hook>
__device__ __forceinline__ void trsm_rowblock_x2(double (&accA)[NB][2], double (&accB)[NB][2],
                                                 const double* __restrict__ Tf, const double* __restrict__ nRf,
                                                 double* __restrict__ gpA, double* __restrict__ gpB, uint32_t colmask,
                                                 int lane, Hook&& after_first)
{
    static_for<0, NB>([&](auto Jc) {
        constexpr int J = decltype(Jc)::value;
        double xa0 = 0.0, xa1 = 0.0, xb0 = 0.0, xb1 = 0.0;
        const double t0 = Tf[J * 64 + lane];
        dmma(xa0, xa1, accA[J][0], t0);
        dmma(xb0, xb1, accB[J][0], t0);
        const double t1 = Tf[J * 64 + 32 + lane];
        dmma(xa0, xa1, accA[J][1], t1);
        dmma(xb0, xb1, accB[J][1], t1);
#pragma unroll
        for (int Jp = J + 1; Jp < NB; ++Jp) {
            const double r0 = nRf[TriFrags<NB>::pair(J, Jp) * 64 + lane];
            dmma(accA[Jp][0], accA[Jp][1], xa0, r0);
            dmma(accB[Jp][0], accB[Jp][1], xb0, r0);
        }
#pragma unroll
        for (int Jp = J + 1; Jp < NB; ++Jp) {
            const double r1 = nRf[TriFrags<NB>::pair(J, Jp) * 64 + 32 + lane];
            dmma(accA[Jp][0], accA[Jp][1], xa1, r1);
            dmma(accB[Jp][0], accB[Jp][1], xb1, r1);
        }
        accA[J][0] = xa0; accA[J][1] = xa1;
        accB[J][0] = xb0; accB[J][1] = xb1;
        if constexpr (J == 0) after_first();
        if (gpA != nullptr) {
            if (FULL || ((colmask >> (2 * J)) & 1u)) *reinterpret_cast<double2*>(gpA + 8 * J) = make_double2(xa0, xa1);
            else if ((colmask >> (2 * J + 1)) & 1u) gpA[8 * J] = xa0;
        }
        if (gpB != nullptr) {
            if (FULL || ((colmask >> (2 * J)) & 1u)) *reinterpret_cast<double2*>(gpB + 8 * J) = make_double2(xb0, xb1);
            else if ((colmask >> (2 * J + 1)) & 1u) gpB[8 * J] = xb0;
        }
    });
}

// Per-warp ring of landing row-blocks fed by bulk async copies.
template <int LD>
struct WarpRing {
    double* buf;          // STAGES x 8 x LD doubles (this warp's)
    uint64_t* bar;        // STAGES mbarriers (this warp's)
    const double* V;
    int64_t ldv, m;
    int n;
    int ld = LD;          // landing row stride: LD (padded rows, one bulk copy per row) or n (BLOCK mode: ldv == n,
                          // the 8 rows are contiguous in memory and land packed with ONE bulk copy; stage stride stays 8 LD)

    __device__ __forceinline__ void issue(int stage, int64_t rblk, int lane) const
    {
        // rows 8*rblk .. 8*rblk+7
        const int64_t row = rblk * 8 + lane;
        const int valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
        if (lane == 0) mbar_expect_tx(bar + stage, (uint32_t)(valid * n * 8));
        __syncwarp();
        if (ld != LD) {       // BLOCK mode: narrow rows are bound by the NUMBER of bulk copies, not by their bytes
            if (lane == 0) bulk_g2s(buf + stage * 8 * LD, V + rblk * 8 * ldv, (uint32_t)(valid * n * 8), bar + stage);
        } else if (lane < valid) {                    // lane i < 8 copies row i (8n bytes) into its padded slot
            bulk_g2s(buf + (stage * 8 + lane) * LD, V + row * ldv, (uint32_t)(n * 8), bar + stage);
        }
    }
};

template <int NB> struct TallCfg {
    static constexpr int N8 = 8 * NB;
    static constexpr int LDL = 8 * NB + LDL_PAD;
    static constexpr int NBLK = NB * (NB + 1) / 2;
    static constexpr int FRAG_DOUBLES = TriFrags<NB>::DOUBLES;         // Tf + nRf
};

// shared-memory carve-up (doubles): [frag sets][scratch NB*64][bars][xs: WARPS x 2 x 8 x N8][ring]
template <int NB, int WARPS, int STAGES, int NSETS, int XSBUF>
struct SmemPlan {
    static constexpr int LDL = TallCfg<NB>::LDL;
    static constexpr int N8 = TallCfg<NB>::N8;
    static constexpr size_t scratch = (size_t)NSETS * TallCfg<NB>::FRAG_DOUBLES;
    static constexpr size_t bars = scratch + NB * 64;
    static constexpr size_t xs = bars + ((WARPS * STAGES + 1) & ~1);
    static constexpr int XLD = (N8 + 15) & ~15;                        // row of an xs block (XsAddr<N8>::LD)
    static constexpr size_t ring = xs + (size_t)WARPS * XSBUF * 8 * XLD;
    static constexpr size_t ring_doubles = (size_t)WARPS * STAGES * 8 * LDL;
    static constexpr size_t red_doubles = XSBUF ? (size_t)WARPS * TallCfg<NB>::NBLK * 64 : 0;   // A4 only
    static constexpr size_t total_doubles =
        (ring + ring_doubles) > red_doubles ? (ring + ring_doubles) : red_doubles;
    static constexpr size_t bytes = total_doubles * sizeof(double);
};

// load the C fragments of a landing row-block (row stride ld).  ld == LDL: rows are padded with zeros up to 8 NB
// columns.  BLOCK mode (ld == n < LDL, rows packed): the columns past n of the last block hold the next row's data and
// are masked with the lane's column mask (col_mask()).
template <int NB, int LDL>
__device__ __forceinline__ void load_acc(double (&acc)[NB][2], const double* __restrict__ rb, int lane, int ld = LDL,
                                         uint32_t colmask = 0xffffffffu)
{
    const int r = lane >> 2, q = lane & 3;
    const double* p = rb + r * ld + 2 * q;
#pragma unroll
    for (int J = 0; J < NB; ++J) {
        double2 v = *reinterpret_cast<const double2*>(p + 8 * J);
        acc[J][0] = v.x; acc[J][1] = v.y;
    }
    if (ld != LDL && ld != 8 * NB) {                  // packed rows narrower than the column blocks: mask the last block
        if (!((colmask >> (2 * (NB - 1) + 1)) & 1u)) acc[NB - 1][0] = 0.0;
        if (!((colmask >> (2 * (NB - 1))) & 1u)) acc[NB - 1][1] = 0.0;
    }
}

