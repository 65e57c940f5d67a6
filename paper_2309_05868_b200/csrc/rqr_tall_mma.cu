// rqr_tall_mma.cu -- FP64 DMMA fast paths of A4 (rqr_trsm_gram) and A6 (rqr_apply), n <= 64.
//
// Design: one persistent CTA per SM, 8 warps, NO block-level
// synchronisation in the main loop.  Every warp is its own pipeline over 8-row blocks of V:
//   * a private ring of STAGES "landing" row-blocks in shared memory (8 rows x (n8+8) doubles),
//     filled by per-row cp.async.bulk (TMA bulk copy, SASS UBLKCP) completing on the warp's own
//     mbarriers; read once (128-bit C-fragment pattern, conflict free at this row stride);
//   * blocked forward substitution with 8x8 diagonal blocks (reading S7/H6):
//       X_J = acc_J T_J,  acc_J' -= X_J R[J,J']  (J' > J),  T_J = inv(R[J,J]) by substitution,
//     every product an mma.sync.m8n8k4.f64 (SASS DMMA).  The chain never leaves the register
//     file: an 8x8 product is two k=4 DMMAs, and the contraction index is PERMUTED so that
//     piece s in {0,1} contracts over columns {2k+s}: lane (r,k) of the A operand then needs
//     X[r][2k+s], which is exactly element s of the C fragment the same lane already holds.  The
//     B fragments (T_J, -R[J,J']) are built once per CTA with the matching row permutation;
//   * a private double-buffered 8 x n8 "xs" block (A4 only) through which X reaches the Gram
//     fragment layout (a transpose across lanes), 16-byte-unit XOR swizzle, conflict free;
//   * software pipelining inside the warp: the 72 independent Gram DMMAs of row-block i are
//     interleaved, 9 per substitution step, into the dependent-issue gaps of the chain of
//     row-block i+1;
//   * the Gram update G += X^T X on the upper block triangle, 36 (n = 64) 8x8 accumulators
//     held in the warp's registers for the whole kernel; X^T as A and X as B are the SAME
//     register (lane l holds X[l%4][l/4] of a 4-row slab).
// The same trsm routine serves rqr_apply, so V1 re-formed there has the same bits (H1).
#include "rqr_mma.cuh"

// ------------------------------------------------------------------------------------------
// A4: V1 = V R0^-1 (optional), store V1 (optional), partial Gram per CTA.
// ------------------------------------------------------------------------------------------
// warps per CTA of A4: bounded by registers (NB = 8: 248 per thread => 8 warps); the narrower
// shapes have small Gram tiles and little work per row-block, so they run more warps to hide the
// per-row-block latencies (mbarrier wait, chain start).  Measured at 2^22 x 32: 0.48 -> 0.37 ms.
// NB = 5, 6 (32 < n <= 48): 15 / 21 Gram blocks = 60 / 84 accumulator registers => 12 warps (168 registers each).
template <int NB> struct GramWarps { static constexpr int value = NB >= 7 ? 8 : (NB >= 5 ? 12 : (NB >= 3 ? 16 : 24)); };

template <int NB, bool HAS_R, bool FULL>
__global__ void __launch_bounds__(GramWarps<NB>::value * 32, 1)
k_trsm_gram_mma(const double* V, int64_t m, int n, int64_t ldv,          // V1 == V allowed: no restrict on either
                const double* __restrict__ R0, double* V1, int64_t ldq,
                double* __restrict__ part, int land_ld)
{
    using Plan = SmemPlan<NB, GramWarps<NB>::value, GRAM_STAGES, 1, 2>;
    constexpr int LDL = Plan::LDL, N8 = Plan::N8;
    constexpr int NBLK = TallCfg<NB>::NBLK;
    extern __shared__ __align__(16) double smem[];
    double* Tf = smem;
    double* nRf = smem + NB * 64;
    double* scratch = smem + Plan::scratch;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Plan::bars);
    double* ring = smem + Plan::ring;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int XB = 8 * Plan::XLD;                 // doubles of one xs block
    double* xs = smem + Plan::xs + (size_t)warp * 2 * XB;

    static_assert(Plan::ring_doubles >= 64 * NB * NB, "ring too small to stage R");
    if (threadIdx.x < GramWarps<NB>::value * GRAM_STAGES) mbar_init(bars + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (HAS_R) build_tri_frags<NB>(R0, n, Tf, nRf, scratch, ring);      // stages R in the (still unused) ring
    // rows of a partial last row-block that the bulk copies do not write must be zero (they enter the Gram)
    for (int i = threadIdx.x; i < (int)Plan::ring_doubles; i += blockDim.x) ring[i] = 0.0;
    fence_proxy_async();
    __syncthreads();

    WarpRing<LDL> wr{ring + (size_t)warp * GRAM_STAGES * 8 * LDL, bars + warp * GRAM_STAGES, V, ldv, m, n, land_ld};
    const XsAddr<N8> ad(lane);
    const int64_t nrb = (m + 7) / 8;
    const int64_t gw = (int64_t)blockIdx.x * GramWarps<NB>::value + warp;
    const int64_t stride = (int64_t)gridDim.x * GramWarps<NB>::value;
#pragma unroll
    for (int s = 0; s < GRAM_STAGES; ++s)
        if (gw + s * stride < nrb) wr.issue(s, gw + s * stride, lane);

    double G[NBLK][2];
#pragma unroll
    for (int b = 0; b < NBLK; ++b) { G[b][0] = 0.0; G[b][1] = 0.0; }
    double g[NB];
    double acc[NB][2];
    const uint32_t colmask = col_mask<NB>(n, lane);
    const int64_t lane_off = (int64_t)(lane >> 2) * ldq + 2 * (lane & 3);

    int it = 0, stage = 0;
    uint32_t phase = 0;
    for (int64_t rblk = gw; rblk < nrb; rblk += stride, ++it) {
        mbar_wait(wr.bar + stage, phase);
        double* rb = wr.buf + stage * 8 * LDL;
        const int valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
        if (valid < 8) {
            for (int e = lane; e < (8 - valid) * wr.ld; e += 32) rb[valid * wr.ld + e] = 0.0;
            __syncwarp();
        }
        load_acc<NB, LDL>(acc, rb, lane, wr.ld, colmask);
        // refill of the landing block once its values have been consumed (registers -> DMMA / xs)
        auto refill = [&]() {
            const int64_t next = rblk + (int64_t)GRAM_STAGES * stride;
            if (next < nrb) {
                fence_proxy_async();
                __syncwarp();
                wr.issue(stage, next, lane);
            }
        };
        double* xsc = xs + (it & 1) * XB;
        const double* xsp = xs + ((it & 1) ^ 1) * XB;
        if (HAS_R) {
            double* gp = (V1 && (lane >> 2) < valid) ? V1 + rblk * 8 * ldq + lane_off : nullptr;
            if (it > 0) trsm_rowblock<NB, true, true, FULL>(acc, xsc, xsp, ad, Tf, nRf, gp, colmask, lane, g, G, refill);
            else        trsm_rowblock<NB, false, true, FULL>(acc, xsc, xsp, ad, Tf, nRf, gp, colmask, lane, g, G, refill);
        } else {
            // plain Gram of V: move the row-block into xs, Gram of the previous one meanwhile
#pragma unroll
            for (int J = 0; J < NB; ++J)
                *reinterpret_cast<double2*>(xsc + ad.c(J)) = make_double2(acc[J][0], acc[J][1]);
            refill();
            if (it > 0) gram_chunk<NB, N8, 0, 2 * NBLK>(xsp, ad, g, G);
            __syncwarp();
        }
        if (++stage == GRAM_STAGES) { stage = 0; phase ^= 1u; }
    }
    if (it > 0) {
        __syncwarp();
        gram_chunk<NB, N8, 0, 2 * NBLK>(xs + ((it - 1) & 1) * XB, ad, g, G);
    }
    // fixed-order reduction of the warps' accumulators, then this CTA's partial (upper blocks)
    __syncthreads();
    double* red = smem;
#pragma unroll
    for (int b = 0; b < NBLK; ++b) {
        red[((size_t)warp * NBLK + b) * 64 + 2 * lane] = G[b][0];
        red[((size_t)warp * NBLK + b) * 64 + 2 * lane + 1] = G[b][1];
    }
    __syncthreads();
    double* P = part + (size_t)blockIdx.x * n * n;
    for (int e = threadIdx.x; e < NBLK * 64; e += blockDim.x) {
        const int b = e >> 6, l = (e >> 1) & 31, k = e & 1;
        double s = red[(size_t)b * 64 + 2 * l + k];
#pragma unroll
        for (int w = 1; w < GramWarps<NB>::value; ++w) s += red[((size_t)w * NBLK + b) * 64 + 2 * l + k];
        int a = 0, rem = b;
        while (rem >= NB - a) { rem -= NB - a; ++a; }
        const int bb = a + rem;
        const int row = 8 * a + (l >> 2), col = 8 * bb + 2 * (l & 3) + k;
        if (row < n && col < n) P[row * n + col] = s;
    }
}

// ------------------------------------------------------------------------------------------
// A4, pair version for 56 < n <= 64 (NB = 8; narrower shapes run k_trsm_gram_mma<NB> with NB = ceil(n / 8)).  The single-warp kernel above needs 248 registers
// (36 Gram accumulators), i.e. 2 warps per SM sub-partition, and loses ~15% of the DMMA pipe to
// moments when both are stalled.  Here two warps form a PAIR: each runs the substitution chain of its
// own row-block, both write X into a pair-shared staging block, and each accumulates HALF of the
// Gram blocks -- fold sets {0,7,1,6} / {2,5,3,4} of block rows, 18 blocks each -- over BOTH row-blocks.
// Same DMMA count per warp (72 chain + 72 Gram per iteration), half the accumulator registers:
// 12 warps per SM (3 per sub-partition).  One named barrier per pair and iteration.
// ------------------------------------------------------------------------------------------
#define PAIR_WARPS 12
#define PAIR_STAGES 2

template <int SIDE>
struct PairSet {
    __host__ __device__ static constexpr int row(int i)
    {
        return SIDE == 0 ? (i == 0 ? 0 : (i == 1 ? 7 : (i == 2 ? 1 : 6))) : (i == 0 ? 2 : (i == 1 ? 5 : (i == 2 ? 3 : 4)));
    }
    __host__ __device__ static constexpr int a(int k)
    {
        int i = 0;
        while (k >= 8 - row(i)) { k -= 8 - row(i); ++i; }
        return row(i);
    }
    __host__ __device__ static constexpr int b(int k)
    {
        int i = 0;
        while (k >= 8 - row(i)) { k -= 8 - row(i); ++i; }
        return row(i) + k;
    }
};

// (a << 4 | b) of Gram block k of side 0 (entries 0..17) and side 1 (18..35), for the epilogue
#define PAB(S, K) (unsigned char)((PairSet<S>::a(K) << 4) | PairSet<S>::b(K))
__constant__ unsigned char c_pair_ab[36] = {
    PAB(0, 0), PAB(0, 1), PAB(0, 2), PAB(0, 3), PAB(0, 4), PAB(0, 5), PAB(0, 6), PAB(0, 7), PAB(0, 8),
    PAB(0, 9), PAB(0, 10), PAB(0, 11), PAB(0, 12), PAB(0, 13), PAB(0, 14), PAB(0, 15), PAB(0, 16), PAB(0, 17),
    PAB(1, 0), PAB(1, 1), PAB(1, 2), PAB(1, 3), PAB(1, 4), PAB(1, 5), PAB(1, 6), PAB(1, 7), PAB(1, 8),
    PAB(1, 9), PAB(1, 10), PAB(1, 11), PAB(1, 12), PAB(1, 13), PAB(1, 14), PAB(1, 15), PAB(1, 16), PAB(1, 17)};
#undef PAB

// Gram DMMAs [T0, T1) of an iteration: t -> row-block t / 36 of the pair, slab (t % 36) / 18, block t % 18
template <int SIDE, int T0, int T1>
__device__ __forceinline__ void pair_gram_chunk(const double* __restrict__ xsp, const XsAddr<64>& ad,
                                                double (&g)[8], double (&G)[18][2])
{
    static_for<T0, T1>([&](auto tc) {
        constexpr int t = decltype(tc)::value;
        if constexpr (t % 18 == 0) {
            constexpr int rbk = t / 36, h = (t % 36) / 18;
#pragma unroll
            for (int a_ = (SIDE ? 2 : 0); a_ < 8; ++a_) g[a_] = xsp[rbk * 512 + ad.g(h, a_)];
        }
        constexpr int k = t % 18;
        dmma(G[k][0], G[k][1], g[PairSet<SIDE>::a(k)], g[PairSet<SIDE>::b(k)]);
    });
}

template <int SIDE, bool ON>
struct PairGram {
    const double* xsp;
    const XsAddr<64>& ad;
    double (&g)[8];
    double (&G)[18][2];
    template <int J, int PART>
    __device__ __forceinline__ void chunk()
    {
        if constexpr (ON) {
            constexpr int E[5] = {0, 2, 4, 6, 9};
            pair_gram_chunk<SIDE, 9 * J + E[PART], 9 * J + E[PART + 1]>(xsp, ad, g, G);
        }
    }
};

struct PairPlan {
    static constexpr int LDL = 64 + LDL_PAD;
    static constexpr size_t scratch = TriFrags<8>::DOUBLES;                      // after Tf, nRf
    static constexpr size_t bars = scratch + 8 * 64;
    static constexpr size_t xs = bars + PAIR_WARPS * PAIR_STAGES;
    static constexpr size_t ring = xs + (size_t)(PAIR_WARPS / 2) * 2 * 2 * 512;  // pair x buffer x row-block
    static constexpr size_t ring_doubles = (size_t)PAIR_WARPS * PAIR_STAGES * 8 * LDL;
    static constexpr size_t red_doubles = (size_t)PAIR_WARPS * 18 * 64;
    static constexpr size_t total = (ring + ring_doubles) > red_doubles ? (ring + ring_doubles) : red_doubles;
    static constexpr size_t bytes = total * sizeof(double);
};

template <int SIDE, bool FULL>
__device__ __forceinline__ void pair_body(const double* V, int64_t m, int n, int64_t ldv,
                                          double* V1, int64_t ldq, double* smem, double (&G)[18][2])
{
    constexpr int LDL = PairPlan::LDL;
    const double* Tf = smem;
    const double* nRf = smem + 8 * 64;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + PairPlan::bars);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, pair = warp >> 1;
    double* xs = smem + PairPlan::xs + (size_t)pair * 2 * 2 * 512;
    WarpRing<LDL> wr{smem + PairPlan::ring + (size_t)warp * PAIR_STAGES * 8 * LDL, bars + warp * PAIR_STAGES, V, ldv, m, n};
    const XsAddr<64> ad(lane);
    const int64_t nrb = (m + 7) / 8;
    const int64_t npairs = (int64_t)gridDim.x * (PAIR_WARPS / 2);
    const int64_t pg = (int64_t)blockIdx.x * (PAIR_WARPS / 2) + pair;
#pragma unroll
    for (int s = 0; s < PAIR_STAGES; ++s) {
        const int64_t rb = (s * npairs + pg) * 2 + SIDE;
        if (rb < nrb) wr.issue(s, rb, lane);
    }
    double g[8];
    double acc[8][2];
    const uint32_t colmask = col_mask<8>(n, lane);
    const int64_t lane_off = (int64_t)(lane >> 2) * ldq + 2 * (lane & 3);
    int t = 0, stage = 0;
    uint32_t phase = 0;
    for (;; ++t) {
        const int64_t base = ((int64_t)t * npairs + pg) * 2;
        if (base >= nrb) break;                              // pair-uniform
        const int64_t rblk = base + SIDE;
        const bool active = rblk < nrb;
        int valid = 0;
        if (active) {
            mbar_wait(wr.bar + stage, phase);
            double* rb = wr.buf + stage * 8 * LDL;
            valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
            if (valid < 8) {
                for (int e = lane; e < (8 - valid) * LDL; e += 32) rb[valid * LDL + e] = 0.0;
                __syncwarp();
            }
            load_acc<8, LDL>(acc, rb, lane);
        } else {
#pragma unroll
            for (int J = 0; J < 8; ++J) { acc[J][0] = 0.0; acc[J][1] = 0.0; }
        }
        auto refill = [&]() {
            const int64_t next = (((int64_t)t + PAIR_STAGES) * npairs + pg) * 2 + SIDE;
            if (active && next < nrb) {
                fence_proxy_async();
                __syncwarp();
                wr.issue(stage, next, lane);
            }
        };
        double* xsc = xs + (t & 1) * 1024 + SIDE * 512;
        const double* xsp = xs + ((t & 1) ^ 1) * 1024;
        double* gp = (V1 && active && (lane >> 2) < valid) ? V1 + rblk * 8 * ldq + lane_off : nullptr;
        if (t > 0) {
            PairGram<SIDE, true> gf{xsp, ad, g, G};
            trsm_rowblock_gf<8, true, FULL>(acc, xsc, ad, Tf, nRf, gp, colmask, lane, refill, gf);
        } else {
            PairGram<SIDE, false> gf{xsp, ad, g, G};
            trsm_rowblock_gf<8, true, FULL>(acc, xsc, ad, Tf, nRf, gp, colmask, lane, refill, gf);
        }
        // both X blocks of this iteration are complete, and the blocks read by this iteration's Gram may be reused
        asm volatile("bar.sync %0, 64;" :: "r"(1 + pair) : "memory");
        if (++stage == PAIR_STAGES) { stage = 0; phase ^= 1u; }
    }
    if (t > 0) pair_gram_chunk<SIDE, 0, 72>(xs + ((t - 1) & 1) * 1024, ad, g, G);
}

template <bool FULL>
__global__ void __launch_bounds__(PAIR_WARPS * 32, 1)
k_trsm_gram_pair(const double* V, int64_t m, int n, int64_t ldv, const double* __restrict__ R0,
                 double* V1, int64_t ldq, double* __restrict__ part)
{
    extern __shared__ __align__(16) double smem[];
    double* ring = smem + PairPlan::ring;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + PairPlan::bars);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    static_assert(PairPlan::ring_doubles >= 64 * 64, "ring too small to stage R");
    if (threadIdx.x < PAIR_WARPS * PAIR_STAGES) mbar_init(bars + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    build_tri_frags<8>(R0, n, smem, smem + 8 * 64, smem + PairPlan::scratch, ring);
    for (int i = threadIdx.x; i < (int)PairPlan::ring_doubles; i += blockDim.x) ring[i] = 0.0;
    fence_proxy_async();
    __syncthreads();

    double G[18][2];
#pragma unroll
    for (int b = 0; b < 18; ++b) { G[b][0] = 0.0; G[b][1] = 0.0; }
    if (warp & 1) pair_body<1, FULL>(V, m, n, ldv, V1, ldq, smem, G);
    else          pair_body<0, FULL>(V, m, n, ldv, V1, ldq, smem, G);

    // fixed-order reduction over the pairs, then this CTA's partial (upper blocks)
    __syncthreads();
    double* red = smem;
#pragma unroll
    for (int b = 0; b < 18; ++b) {
        red[((size_t)warp * 18 + b) * 64 + 2 * lane] = G[b][0];
        red[((size_t)warp * 18 + b) * 64 + 2 * lane + 1] = G[b][1];
    }
    __syncthreads();
    double* P = part + (size_t)blockIdx.x * n * n;
    // thread = (block j = side * 18 + k of the 36 upper blocks: threadIdx / 64 + 6 i, element threadIdx % 64)
    const int l = (threadIdx.x >> 1) & 31, kk = threadIdx.x & 1;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        const int j = (threadIdx.x >> 6) + (PAIR_WARPS * 32 / 64) * i;       // 384 threads: 6 blocks per pass
        if (j < 36) {
            const int side = j >= 18, k = j - 18 * side;
            double s = 0.0;
#pragma unroll
            for (int p = 0; p < PAIR_WARPS / 2; ++p) s += red[((size_t)(2 * p + side) * 18 + k) * 64 + 2 * l + kk];
            const int ab = c_pair_ab[j];
            const int row = 8 * (ab >> 4) + (l >> 2), col = 8 * (ab & 15) + 2 * (l & 3) + kk;
            if (row < n && col < n) P[row * n + col] = s;
        }
    }
}

// ------------------------------------------------------------------------------------------
// A6: Q = (V R0^-1) R1^-1  (TWO) or Q = V R1^-1.
// ------------------------------------------------------------------------------------------
// A6 launch shape, measured at 2^23 x 64 (profiles/r1_final_summary.md): the in-place pass (one chain per
// row-block, HBM-bound) is fastest with 8 warps x 3 stages (1.31 ms = 6.56 TB/s; 12 x 2: 1.44, 10 x 3: 1.53,
// 6 x 4: 1.71), the two-pass recompute mode (DMMA-bound) with 12 x 2 (2.22 ms; 8 x 3: 2.42).
// n <= 16 (tiny row-blocks) keeps 12 x 2 in both modes (2^22 x 16: 0.21 vs 0.25 ms).
template <int NB, bool TWO> struct ApplyCfg {
    static constexpr int WARPS = (TWO || NB < 4) ? 12 : 8;
    static constexpr int STAGES = (TWO || NB < 4) ? 2 : 3;
};

template <int NB, bool TWO, bool FULL>
__global__ void __launch_bounds__(ApplyCfg<NB, TWO>::WARPS * 32, 1)
k_apply_mma(const double* V, int64_t m, int n, int64_t ldv,              // Q == V allowed: no restrict on either
            const double* __restrict__ R0, const double* __restrict__ R1,
            double* Q, int64_t ldq, int land_ld)
{
    using Plan = SmemPlan<NB, ApplyCfg<NB, TWO>::WARPS, ApplyCfg<NB, TWO>::STAGES, 2, 0>;
    constexpr int LDL = Plan::LDL, N8 = Plan::N8;
    constexpr int FD = TallCfg<NB>::FRAG_DOUBLES;
    constexpr int NBLK = TallCfg<NB>::NBLK;
    extern __shared__ __align__(16) double smem[];
    double* Tf1 = smem;
    double* nRf1 = smem + NB * 64;
    double* Tf0 = smem + FD;
    double* nRf0 = smem + FD + NB * 64;
    double* scratch = smem + Plan::scratch;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Plan::bars);
    double* ring = smem + Plan::ring;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    static_assert(Plan::ring_doubles >= 64 * NB * NB, "ring too small to stage R");
    if (threadIdx.x < ApplyCfg<NB, TWO>::WARPS * ApplyCfg<NB, TWO>::STAGES) mbar_init(bars + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    build_tri_frags<NB>(R1, n, Tf1, nRf1, scratch, ring);
    if (TWO) build_tri_frags<NB>(R0, n, Tf0, nRf0, scratch, ring);
    for (int i = threadIdx.x; i < (int)Plan::ring_doubles; i += blockDim.x) ring[i] = 0.0;
    fence_proxy_async();
    __syncthreads();

    WarpRing<LDL> wr{ring + (size_t)warp * ApplyCfg<NB, TWO>::STAGES * 8 * LDL, bars + warp * ApplyCfg<NB, TWO>::STAGES, V, ldv, m, n, land_ld};
    const XsAddr<N8> ad(lane);
    const int64_t nrb = (m + 7) / 8;
    const int64_t gw = (int64_t)blockIdx.x * ApplyCfg<NB, TWO>::WARPS + warp;
    const int64_t stride = (int64_t)gridDim.x * ApplyCfg<NB, TWO>::WARPS;
#pragma unroll
    for (int s = 0; s < ApplyCfg<NB, TWO>::STAGES; ++s)
        if (gw + s * stride < nrb) wr.issue(s, gw + s * stride, lane);
    double acc[NB][2];
    double g[NB];
    double G[NBLK][2];      // unused (GRAM = false): optimised away
    const uint32_t colmask = col_mask<NB>(n, lane);
    const int64_t lane_off = (int64_t)(lane >> 2) * ldq + 2 * (lane & 3);
    int stage = 0;
    uint32_t phase = 0;
    for (int64_t rblk = gw; rblk < nrb; rblk += stride) {
        mbar_wait(wr.bar + stage, phase);
        double* rb = wr.buf + stage * 8 * LDL;
        const int valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
        if (valid < 8) {
            for (int e = lane; e < (8 - valid) * wr.ld; e += 32) rb[valid * wr.ld + e] = 0.0;
            __syncwarp();
        }
        load_acc<NB, LDL>(acc, rb, lane, wr.ld, colmask);
        auto refill = [&]() {
            const int64_t next = rblk + (int64_t)ApplyCfg<NB, TWO>::STAGES * stride;
            if (next < nrb) {
                fence_proxy_async();
                __syncwarp();
                wr.issue(stage, next, lane);
            }
        };
        auto nohook = []() {};
        double* gp = ((lane >> 2) < valid) ? Q + rblk * 8 * ldq + lane_off : nullptr;
        if (TWO) {
            trsm_rowblock<NB, false, false, FULL>(acc, nullptr, nullptr, ad, Tf0, nRf0, nullptr, colmask, lane, g, G, refill);
            trsm_rowblock<NB, false, false, FULL>(acc, nullptr, nullptr, ad, Tf1, nRf1, gp, colmask, lane, g, G, nohook);
        } else {
            trsm_rowblock<NB, false, false, FULL>(acc, nullptr, nullptr, ad, Tf1, nRf1, gp, colmask, lane, g, G, refill);
        }
        if (++stage == ApplyCfg<NB, TWO>::STAGES) { stage = 0; phase ^= 1u; }
    }
}

// A6 with two row-blocks per warp and iteration (trsm_rowblock_x2): half the B-fragment loads, two independent chains
// per warp.  Ring of 4 stages = two pairs: the pair of iteration i + 1 lands while pair i is in the registers.
#define APPLY2_WARPS 8
#define APPLY2_STAGES 4
template <int NB, bool TWO, bool FULL>
__global__ void __launch_bounds__(APPLY2_WARPS * 32, 1)
k_apply_mma2(const double* V, int64_t m, int n, int64_t ldv,             // Q == V allowed: no restrict on either
             const double* __restrict__ R0, const double* __restrict__ R1,
             double* Q, int64_t ldq, int land_ld)
{
    using Plan = SmemPlan<NB, APPLY2_WARPS, APPLY2_STAGES, 2, 0>;
    constexpr int LDL = Plan::LDL;
    constexpr int FD = TallCfg<NB>::FRAG_DOUBLES;
    extern __shared__ __align__(16) double smem[];
    double* Tf1 = smem;
    double* nRf1 = smem + NB * 64;
    double* Tf0 = smem + FD;
    double* nRf0 = smem + FD + NB * 64;
    double* scratch = smem + Plan::scratch;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Plan::bars);
    double* ring = smem + Plan::ring;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    static_assert(Plan::ring_doubles >= 64 * NB * NB, "ring too small to stage R");
    if (threadIdx.x < APPLY2_WARPS * APPLY2_STAGES) mbar_init(bars + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    build_tri_frags<NB>(R1, n, Tf1, nRf1, scratch, ring);
    if (TWO) build_tri_frags<NB>(R0, n, Tf0, nRf0, scratch, ring);
    for (int i = threadIdx.x; i < (int)Plan::ring_doubles; i += blockDim.x) ring[i] = 0.0;
    fence_proxy_async();
    __syncthreads();

    WarpRing<LDL> wr{ring + (size_t)warp * APPLY2_STAGES * 8 * LDL, bars + warp * APPLY2_STAGES, V, ldv, m, n, land_ld};
    const int64_t nrb = (m + 7) / 8;
    const int64_t gw = (int64_t)blockIdx.x * APPLY2_WARPS + warp;
    const int64_t stride = (int64_t)gridDim.x * APPLY2_WARPS;
#pragma unroll
    for (int s = 0; s < APPLY2_STAGES; ++s)
        if (gw + s * stride < nrb) wr.issue(s, gw + s * stride, lane);
    double accA[NB][2], accB[NB][2];
    const uint32_t colmask = col_mask<NB>(n, lane);
    const int64_t lane_off = (int64_t)(lane >> 2) * ldq + 2 * (lane & 3);
    int stage = 0;                                   // even: the pair uses stages (stage, stage + 1)
    uint32_t phase = 0;
    for (int64_t rblk = gw; rblk < nrb; rblk += 2 * stride) {
        const int64_t rblkB = rblk + stride;
        const bool hasB = rblkB < nrb;
        auto land = [&](int st, int64_t rb_idx, double (&acc)[NB][2]) {
            mbar_wait(wr.bar + st, phase);
            double* rb = wr.buf + st * 8 * LDL;
            const int valid = (int)((m - rb_idx * 8) < 8 ? (m - rb_idx * 8) : 8);
            if (valid < 8) {
                for (int e = lane; e < (8 - valid) * wr.ld; e += 32) rb[valid * wr.ld + e] = 0.0;
                __syncwarp();
            }
            load_acc<NB, LDL>(acc, rb, lane, wr.ld, colmask);
            return valid;
        };
        const int validA = land(stage, rblk, accA);
        int validB = 0;
        if (hasB) validB = land(stage + 1, rblkB, accB);
        else {
#pragma unroll
            for (int J = 0; J < NB; ++J) { accB[J][0] = 0.0; accB[J][1] = 0.0; }
        }
        auto refill = [&]() {
            const int64_t nextA = rblk + (int64_t)APPLY2_STAGES * stride, nextB = nextA + stride;
            if (nextA < nrb || nextB < nrb) {
                fence_proxy_async();
                __syncwarp();
                if (nextA < nrb) wr.issue(stage, nextA, lane);
                if (nextB < nrb) wr.issue(stage + 1, nextB, lane);
            }
        };
        auto nohook = []() {};
        double* gpA = ((lane >> 2) < validA) ? Q + rblk * 8 * ldq + lane_off : nullptr;
        double* gpB = (hasB && (lane >> 2) < validB) ? Q + rblkB * 8 * ldq + lane_off : nullptr;
        if (TWO) {
            trsm_rowblock_x2<NB, FULL>(accA, accB, Tf0, nRf0, nullptr, nullptr, colmask, lane, refill);
            trsm_rowblock_x2<NB, FULL>(accA, accB, Tf1, nRf1, gpA, gpB, colmask, lane, nohook);
        } else {
            trsm_rowblock_x2<NB, FULL>(accA, accB, Tf1, nRf1, gpA, gpB, colmask, lane, refill);
        }
        stage += 2;
        if (stage == APPLY2_STAGES) { stage = 0; phase ^= 1u; }
    }
}

// ------------------------------------------------------------------------------------------
// host dispatch
// ------------------------------------------------------------------------------------------
static bool fast_ok(const void* V, int n, int64_t ldv, const void* Q, int64_t ldq)
{
    if (n > 64 || (n & 1) || (ldv & 1)) return false;
    if (((uintptr_t)V & 15) != 0) return false;
    if (Q && (((uintptr_t)Q & 15) != 0 || (ldq & 1))) return false;
    return true;
}

#ifndef RQR_BLOCK_GRAM_MAX_NB
#define RQR_BLOCK_GRAM_MAX_NB 8
#endif
// BLOCK mode of the landing ring (rqr_mma.cuh WarpRing): ONE bulk copy per 8-row block instead of one per row, when the
// rows are contiguous (ldv == n).  Narrow rows are bound by the number of bulk copies, not by their bytes: measured
// (profiles/r2_summary.md section 9, 10^7 x 10..24 and 2^22 x 32..56) the plain Gram gains 10-30% at every n, A4 with R0
// 5-15% (not at 16 < n <= 24 when it also stores V1), the two-pass apply 5-20%, the in-place apply only for n <= 24 (it
// loses 12-15% for n >= 40).  kind: 1 = plain Gram (no R0), 2 = A4 with R0, 4 = A6.
#ifndef RQR_BLOCK_MODE
#define RQR_BLOCK_MODE 7
#endif
template <int NB>
static int landing_ld(int n, int64_t ldv, int kind, bool stores_v1_or_two_pass)
{
    bool block = ldv == n && (RQR_BLOCK_MODE & kind);
    if (kind == 1) block = block && NB <= RQR_BLOCK_GRAM_MAX_NB;
    if (kind == 2 && stores_v1_or_two_pass && NB == 3) block = false;
    if (kind == 4 && !stores_v1_or_two_pass && NB > 3) block = false;
    return block ? n : TallCfg<NB>::LDL;
}

static int grid_for(int64_t m, int warps)
{
    int64_t nrb = (m + 7) / 8;
    int64_t g = (nrb + warps - 1) / warps;
    return (int)(g < 148 ? (g < 1 ? 1 : g) : 148);
}

template <int NB>
static int launch_trsm_gram(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* V1,
                            int64_t ldq, double* part, int* nparts, cudaStream_t st)
{
    using Plan = SmemPlan<NB, GramWarps<NB>::value, GRAM_STAGES, 1, 2>;
    static_assert(Plan::bytes <= 227 * 1024, "A4 shared memory plan too large");
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_trsm_gram_mma<NB, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
        cudaFuncSetAttribute(k_trsm_gram_mma<NB, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
        cudaFuncSetAttribute(k_trsm_gram_mma<NB, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
    });
    const int grid = grid_for(m, GramWarps<NB>::value);
    *nparts = grid;
    const int lld = landing_ld<NB>(n, ldv, R0 ? 2 : 1, V1 != nullptr);
    if (R0 && n == 8 * NB) k_trsm_gram_mma<NB, true, true><<<grid, GramWarps<NB>::value * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, V1, ldq, part, lld);
    else if (R0)           k_trsm_gram_mma<NB, true, false><<<grid, GramWarps<NB>::value * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, V1, ldq, part, lld);
    else                   k_trsm_gram_mma<NB, false, false><<<grid, GramWarps<NB>::value * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, nullptr, ldq, part, lld);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// A/B switch of the 56 < n <= 64 kernel, compile time only (-DRQR_A4_PAIR=0 builds the single-warp kernel in)
#ifndef RQR_A4_PAIR
#define RQR_A4_PAIR 1
#endif

static int launch_trsm_gram_pair(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* V1,
                                 int64_t ldq, double* part, int* nparts, cudaStream_t st)
{
    static_assert(PairPlan::bytes <= 227 * 1024, "A4 pair shared memory plan too large");
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_trsm_gram_pair<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PairPlan::bytes);
        cudaFuncSetAttribute(k_trsm_gram_pair<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PairPlan::bytes);
    });
    const int64_t npair_blocks = ((m + 7) / 8 + 1) / 2;
    int64_t g = (npair_blocks + PAIR_WARPS / 2 - 1) / (PAIR_WARPS / 2);
    const int grid = (int)(g < 148 ? (g < 1 ? 1 : g) : 148);
    *nparts = grid;
    if (n == 64) k_trsm_gram_pair<true><<<grid, PAIR_WARPS * 32, PairPlan::bytes, st>>>(V, m, n, ldv, R0, V1, ldq, part);
    else         k_trsm_gram_pair<false><<<grid, PAIR_WARPS * 32, PairPlan::bytes, st>>>(V, m, n, ldv, R0, V1, ldq, part);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

int rqr_trsm_gram_mma(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* V1,
                      int64_t ldq, double* part, int* nparts, cudaStream_t st)
{
    if (!fast_ok(V, n, ldv, V1, ldq)) return RQR_TALL_NOT_HANDLED;
    if (!R0 && V1) return RQR_TALL_NOT_HANDLED;       // plain copy + Gram: generic kernel
    if (n <= 16) return launch_trsm_gram<2>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
    if (n <= 24) return launch_trsm_gram<3>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
    if (n <= 32) return launch_trsm_gram<4>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
    if (n <= 40) return launch_trsm_gram<5>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
    // column blocks of 8: n <= 16, 24, 32, 40, 48 run 2, 3, 4, 5, 6 blocks (NB (NB + 1) DMMA per 8 rows for the
    // substitution and as many for the Gram), above 48 the 8-block pair kernel
    if (n <= 48) return launch_trsm_gram<6>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
    if (n <= 56) return launch_trsm_gram<7>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
    if (RQR_A4_PAIR && R0) return launch_trsm_gram_pair(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
    return launch_trsm_gram<8>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
}

#ifndef RQR_APPLY_X2
#define RQR_APPLY_X2 1
#endif
template <int NB, bool TWO>
static int launch_apply2_mode(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                              double* Q, int64_t ldq, cudaStream_t st)
{
    using Plan = SmemPlan<NB, APPLY2_WARPS, APPLY2_STAGES, 2, 0>;
    static_assert(Plan::bytes <= 227 * 1024, "A6 (x2) shared memory plan too large");
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_apply_mma2<NB, TWO, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
        cudaFuncSetAttribute(k_apply_mma2<NB, TWO, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
    });
    const int grid = grid_for(m, 2 * APPLY2_WARPS);
    const int lld = landing_ld<NB>(n, ldv, 4, TWO);
    if (n == 8 * NB) k_apply_mma2<NB, TWO, true><<<grid, APPLY2_WARPS * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, R1, Q, ldq, lld);
    else             k_apply_mma2<NB, TWO, false><<<grid, APPLY2_WARPS * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, R1, Q, ldq, lld);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

template <int NB, bool TWO>
static int launch_apply_mode(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                             double* Q, int64_t ldq, cudaStream_t st)
{
    // two row-blocks per warp (k_apply_mma2): measured against the one-block kernel on the same box, in place: n = 32
    // 0.327 vs 0.340 ms (2^22 rows), n = 64 1.42 vs 1.46-1.48 ms inside the C3 factorization (equal stand-alone); slower
    // at n = 40 / 48 (0.548 vs 0.476 ms) and in the two-pass mode: only NB = 4 and NB = 8 in place take it
    if constexpr (RQR_APPLY_X2 && !TWO && (NB == 4 || NB == 8)) return launch_apply2_mode<NB, TWO>(V, m, n, ldv, R0, R1, Q, ldq, st);
    constexpr int W = ApplyCfg<NB, TWO>::WARPS;
    using Plan = SmemPlan<NB, W, ApplyCfg<NB, TWO>::STAGES, 2, 0>;
    static_assert(Plan::bytes <= 227 * 1024, "A6 shared memory plan too large");
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_apply_mma<NB, TWO, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
        cudaFuncSetAttribute(k_apply_mma<NB, TWO, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
    });
    const int grid = grid_for(m, W);
    const int lld = landing_ld<NB>(n, ldv, 4, TWO);
    if (n == 8 * NB) k_apply_mma<NB, TWO, true><<<grid, W * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, R1, Q, ldq, lld);
    else             k_apply_mma<NB, TWO, false><<<grid, W * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, R1, Q, ldq, lld);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

template <int NB>
static int launch_apply(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                        double* Q, int64_t ldq, cudaStream_t st)
{
    return R0 ? launch_apply_mode<NB, true>(V, m, n, ldv, R0, R1, Q, ldq, st)
              : launch_apply_mode<NB, false>(V, m, n, ldv, R0, R1, Q, ldq, st);
}

int rqr_apply_mma(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                  double* Q, int64_t ldq, cudaStream_t st)
{
    if (!fast_ok(V, n, ldv, Q, ldq)) return RQR_TALL_NOT_HANDLED;
    if (n <= 16) return launch_apply<2>(V, m, n, ldv, R0, R1, Q, ldq, st);
    if (n <= 24) return launch_apply<3>(V, m, n, ldv, R0, R1, Q, ldq, st);
    if (n <= 32) return launch_apply<4>(V, m, n, ldv, R0, R1, Q, ldq, st);
    if (n <= 40) return launch_apply<5>(V, m, n, ldv, R0, R1, Q, ldq, st);
    if (n <= 48) return launch_apply<6>(V, m, n, ldv, R0, R1, Q, ldq, st);
    if (n <= 56) return launch_apply<7>(V, m, n, ldv, R0, R1, Q, ldq, st);
    return launch_apply<8>(V, m, n, ldv, R0, R1, Q, ldq, st);
}
