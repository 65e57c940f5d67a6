// rqr_tall_mma.cu -- FP64 DMMA fast paths of A4 (rqr_trsm_gram) and A6 (rqr_apply), n <= 64.
//
// Design: one persistent CTA per SM, 8 warps, NO block-level
// synchronisation in the main loop.  Every warp is its own pipeline over 8-row blocks of V:
//   * a private ring of STAGES shared-memory row-blocks (8 rows x LD doubles, LD = n8 + 4 so
//     that all three fragment access patterns are bank-conflict free), filled by per-row
//     cp.async.bulk (TMA bulk copy, SASS UBLKCP) completing on the warp's own mbarriers;
//   * blocked forward substitution with 8x8 diagonal blocks (reading S7/H6):
//       X_J = acc_J T_J,  acc_J' -= X_J R[J,J']  (J' > J),  T_J = inv(R[J,J]) by substitution,
//     every product an mma.sync.m8n8k4.f64 (SASS DMMA); C->A fragment conversions go through
//     the warp's own row-block in shared memory (in place);
//   * the Gram update G += X^T X on the upper block triangle, 36 (n = 64) 8x8 accumulators
//     held in the warp's registers for the whole kernel; X^T as A and X as B are the SAME
//     register (lane l holds X[l%4][l/4] of a 4-row slab).
// The same trsm routine serves rqr_apply, so V1 re-formed there has the same bits (H1).
#include "rqr_common.cuh"
#include "rqr_tall.cuh"

#define MMA_WARPS 8
#define MMA_STAGES 4

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
//   Tf [J][h][lane]      = T_J[4h + lane%4][lane/4],     T_J = inv(R[J,J])   (B fragments)
//   nRf[p(J,J')][h][lane] = -R[8J + 4h + lane%4][8J' + lane/4],  J < J'
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

template <int NB>
__device__ void build_tri_frags(const double* __restrict__ R, int n, double* __restrict__ Tf,
                                double* __restrict__ nRf, double* __restrict__ scratch /* NB*64 */)
{
    const int tid = threadIdx.x;
    // T_J column c by back substitution: R_JJ t = e_c  (one thread per (J, c))
    for (int t = tid; t < NB * 8; t += blockDim.x) {
        const int J = t >> 3, c = t & 7;
        double tc[8];
#pragma unroll
        for (int i = 7; i >= 0; --i) {
            double s = (i == c) ? 1.0 : 0.0;
#pragma unroll
            for (int k = 7; k > i; --k) s = fma(-r_padded(R, n, 8 * J + i, 8 * J + k), tc[k], s);
            tc[i] = (i <= c) ? s / r_padded(R, n, 8 * J + i, 8 * J + i) : 0.0;
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) scratch[J * 64 + i * 8 + c] = tc[i];
    }
    __syncthreads();
    for (int t = tid; t < NB * 64; t += blockDim.x) {
        const int J = t >> 6, h = (t >> 5) & 1, lane = t & 31;
        Tf[t] = scratch[J * 64 + (4 * h + (lane & 3)) * 8 + (lane >> 2)];
    }
    for (int t = tid; t < TriFrags<NB>::NPAIR * 64; t += blockDim.x) {
        const int p = t >> 6, h = (t >> 5) & 1, lane = t & 31;
        // invert p -> (J, J')
        int J = 0, rem = p;
        while (rem >= NB - 1 - J) { rem -= NB - 1 - J; ++J; }
        const int Jp = J + 1 + rem;
        nRf[t] = -r_padded(R, n, 8 * J + 4 * h + (lane & 3), 8 * Jp + (lane >> 2));
    }
    __syncthreads();
}

// ------------------------------------------------------------------------------------------
// X = X R^-1 on one 8-row block held in shared memory (rb: 8 x LD doubles), in place, by the
// calling warp.  Optionally stores X to global (gout = row 0 of the block, guarded).
// ------------------------------------------------------------------------------------------
template <int NB, int LD>
__device__ __forceinline__ void trsm_rowblock(double* __restrict__ rb, const double* __restrict__ Tf,
                                              const double* __restrict__ nRf, double* __restrict__ gout,
                                              int64_t ldq, int rows_valid, int n, int lane)
{
    const int r = lane >> 2, q = lane & 3;
    double acc[NB][2];
#pragma unroll
    for (int J = 0; J < NB; ++J) {
        double2 v = *reinterpret_cast<const double2*>(rb + r * LD + 8 * J + 2 * q);
        acc[J][0] = v.x; acc[J][1] = v.y;
    }
#pragma unroll
    for (int J = 0; J < NB; ++J) {
        // C -> A fragments of acc_J through the row-block (in place)
        *reinterpret_cast<double2*>(rb + r * LD + 8 * J + 2 * q) = make_double2(acc[J][0], acc[J][1]);
        __syncwarp();
        double a0 = rb[r * LD + 8 * J + q], a1 = rb[r * LD + 8 * J + 4 + q];
        __syncwarp();
        double x0 = 0.0, x1 = 0.0;
        dmma(x0, x1, a0, Tf[J * 64 + lane]);
        dmma(x0, x1, a1, Tf[J * 64 + 32 + lane]);
        *reinterpret_cast<double2*>(rb + r * LD + 8 * J + 2 * q) = make_double2(x0, x1);
        if (gout != nullptr && r < rows_valid) {
            const int c = 8 * J + 2 * q;
            if (c + 1 < n) *reinterpret_cast<double2*>(gout + (int64_t)r * ldq + c) = make_double2(x0, x1);
            else if (c < n) gout[(int64_t)r * ldq + c] = x0;
        }
        if (J + 1 < NB) {
            __syncwarp();
            a0 = rb[r * LD + 8 * J + q]; a1 = rb[r * LD + 8 * J + 4 + q];
#pragma unroll
            for (int Jp = J + 1; Jp < NB; ++Jp) {
                const int p = TriFrags<NB>::pair(J, Jp);
                dmma(acc[Jp][0], acc[Jp][1], a0, nRf[p * 64 + lane]);
                dmma(acc[Jp][0], acc[Jp][1], a1, nRf[p * 64 + 32 + lane]);
            }
        }
    }
    __syncwarp();
}

// Per-warp ring of row-blocks fed by bulk async copies.
template <int LD>
struct WarpRing {
    double* buf;          // MMA_STAGES x 8 x LD doubles (this warp's)
    uint64_t* bar;        // MMA_STAGES mbarriers (this warp's)
    const double* V;
    int64_t ldv, m;
    int n;

    __device__ __forceinline__ void issue(int stage, int64_t rblk, int lane) const
    {
        // rows 8*rblk .. 8*rblk+7; lane i < 8 copies row i (8n bytes) into its padded slot
        const int64_t row = rblk * 8 + lane;
        const int valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
        if (lane == 0) mbar_expect_tx(bar + stage, (uint32_t)(valid * n * 8));
        __syncwarp();
        if (lane < valid) bulk_g2s(buf + (stage * 8 + lane) * LD, V + row * ldv, (uint32_t)(n * 8), bar + stage);
    }
};

template <int NB> struct TallCfg {
    static constexpr int LD = 8 * NB + 4;
    static constexpr int NBLK = NB * (NB + 1) / 2;
    static constexpr int FRAG_DOUBLES = TriFrags<NB>::DOUBLES;         // Tf + nRf
};

// shared-memory carve-up (doubles): [frag sets][scratch NB*64][bars as u64][ring]
template <int NB, int WARPS, int STAGES, int NSETS>
struct SmemPlan {
    static constexpr int LD = TallCfg<NB>::LD;
    static constexpr size_t frag = (size_t)NSETS * TallCfg<NB>::FRAG_DOUBLES;
    static constexpr size_t scratch = frag;
    static constexpr size_t bars = scratch + NB * 64;
    static constexpr size_t ring = bars + WARPS * STAGES;
    static constexpr size_t ring_doubles = (size_t)WARPS * STAGES * 8 * LD;
    static constexpr size_t red_doubles = (size_t)WARPS * TallCfg<NB>::NBLK * 64;
    static constexpr size_t total_doubles =
        (ring + ring_doubles) > red_doubles ? (ring + ring_doubles) : red_doubles;
    static constexpr size_t bytes = total_doubles * sizeof(double);
};

// ------------------------------------------------------------------------------------------
// A4: V1 = V R0^-1 (optional), store V1 (optional), partial Gram per CTA.
// ------------------------------------------------------------------------------------------
template <int NB, bool HAS_R>
__global__ void __launch_bounds__(MMA_WARPS * 32, 1)
k_trsm_gram_mma(const double* __restrict__ V, int64_t m, int n, int64_t ldv,
                const double* __restrict__ R0, double* __restrict__ V1, int64_t ldq,
                double* __restrict__ part)
{
    using Plan = SmemPlan<NB, MMA_WARPS, MMA_STAGES, 1>;
    constexpr int LD = Plan::LD;
    constexpr int NBLK = TallCfg<NB>::NBLK;
    extern __shared__ __align__(16) double smem[];
    double* Tf = smem;
    double* nRf = smem + NB * 64;
    double* scratch = smem + Plan::scratch;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Plan::bars);
    double* ring = smem + Plan::ring;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int r = lane >> 2, q = lane & 3;

    for (int i = threadIdx.x; i < (int)Plan::ring_doubles; i += blockDim.x) ring[i] = 0.0;
    if (threadIdx.x < MMA_WARPS * MMA_STAGES) mbar_init(bars + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
    __syncthreads();
    if (HAS_R) build_tri_frags<NB>(R0, n, Tf, nRf, scratch);

    WarpRing<LD> wr{ring + (size_t)warp * MMA_STAGES * 8 * LD, bars + warp * MMA_STAGES, V, ldv, m, n};
    const int64_t nrb = (m + 7) / 8;
    const int64_t gw = (int64_t)blockIdx.x * MMA_WARPS + warp;
    const int64_t stride = (int64_t)gridDim.x * MMA_WARPS;
#pragma unroll
    for (int s = 0; s < MMA_STAGES; ++s)
        if (gw + s * stride < nrb) wr.issue(s, gw + s * stride, lane);

    double G[NBLK][2];
#pragma unroll
    for (int b = 0; b < NBLK; ++b) { G[b][0] = 0.0; G[b][1] = 0.0; }

    int it = 0;
    for (int64_t rblk = gw; rblk < nrb; rblk += stride, ++it) {
        const int stage = it % MMA_STAGES;
        mbar_wait(wr.bar + stage, (uint32_t)((it / MMA_STAGES) & 1));
        double* rb = wr.buf + stage * 8 * LD;
        const int valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
        if (valid < 8) {
            for (int e = lane; e < (8 - valid) * LD; e += 32) rb[valid * LD + e] = 0.0;
            __syncwarp();
        }
        if (HAS_R)
            trsm_rowblock<NB, LD>(rb, Tf, nRf, V1 ? V1 + rblk * 8 * ldq : nullptr, ldq, valid, n, lane);
        // Gram: two 4-row slabs; lane holds X[4h + q][8a + r] = A fragment of X^T = B fragment of X
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            double g[NB];
#pragma unroll
            for (int a = 0; a < NB; ++a) g[a] = rb[(4 * h + q) * LD + 8 * a + r];
            int idx = 0;
#pragma unroll
            for (int a = 0; a < NB; ++a)
#pragma unroll
                for (int b = a; b < NB; ++b) { dmma(G[idx][0], G[idx][1], g[a], g[b]); ++idx; }
        }
        __syncwarp();
        const int64_t next = rblk + (int64_t)MMA_STAGES * stride;
        if (next < nrb) {
            fence_proxy_async();
            __syncwarp();
            wr.issue(stage, next, lane);
        }
    }
    // fixed-order reduction of the 8 warps' accumulators, then this CTA's partial (upper blocks)
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
        for (int w = 1; w < MMA_WARPS; ++w) s += red[((size_t)w * NBLK + b) * 64 + 2 * l + k];
        // block b -> (a, bb)
        int a = 0, rem = b;
        while (rem >= NB - a) { rem -= NB - a; ++a; }
        const int bb = a + rem;
        const int row = 8 * a + (l >> 2), col = 8 * bb + 2 * (l & 3) + k;
        if (row < n && col < n) P[row * n + col] = s;
    }
}

// ------------------------------------------------------------------------------------------
// A6: Q = (V R0^-1) R1^-1  (TWO) or Q = V R1^-1.
// ------------------------------------------------------------------------------------------
template <int NB, bool TWO>
__global__ void __launch_bounds__(MMA_WARPS * 32, 1)
k_apply_mma(const double* __restrict__ V, int64_t m, int n, int64_t ldv,
            const double* __restrict__ R0, const double* __restrict__ R1,
            double* __restrict__ Q, int64_t ldq)
{
    using Plan = SmemPlan<NB, MMA_WARPS, MMA_STAGES, 2>;
    constexpr int LD = Plan::LD;
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

    for (int i = threadIdx.x; i < (int)Plan::ring_doubles; i += blockDim.x) ring[i] = 0.0;
    if (threadIdx.x < MMA_WARPS * MMA_STAGES) mbar_init(bars + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
    __syncthreads();
    build_tri_frags<NB>(R1, n, Tf1, nRf1, scratch);
    if (TWO) build_tri_frags<NB>(R0, n, Tf0, nRf0, scratch);

    WarpRing<LD> wr{ring + (size_t)warp * MMA_STAGES * 8 * LD, bars + warp * MMA_STAGES, V, ldv, m, n};
    const int64_t nrb = (m + 7) / 8;
    const int64_t gw = (int64_t)blockIdx.x * MMA_WARPS + warp;
    const int64_t stride = (int64_t)gridDim.x * MMA_WARPS;
#pragma unroll
    for (int s = 0; s < MMA_STAGES; ++s)
        if (gw + s * stride < nrb) wr.issue(s, gw + s * stride, lane);
    int it = 0;
    for (int64_t rblk = gw; rblk < nrb; rblk += stride, ++it) {
        const int stage = it % MMA_STAGES;
        mbar_wait(wr.bar + stage, (uint32_t)((it / MMA_STAGES) & 1));
        double* rb = wr.buf + stage * 8 * LD;
        const int valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
        if (valid < 8) {
            for (int e = lane; e < (8 - valid) * LD; e += 32) rb[valid * LD + e] = 0.0;
            __syncwarp();
        }
        if (TWO) trsm_rowblock<NB, LD>(rb, Tf0, nRf0, nullptr, ldq, valid, n, lane);
        trsm_rowblock<NB, LD>(rb, Tf1, nRf1, Q + rblk * 8 * ldq, ldq, valid, n, lane);
        const int64_t next = rblk + (int64_t)MMA_STAGES * stride;
        if (next < nrb) {
            fence_proxy_async();
            __syncwarp();
            wr.issue(stage, next, lane);
        }
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

static int grid_for(int64_t m)
{
    int64_t nrb = (m + 7) / 8;
    int64_t g = (nrb + MMA_WARPS - 1) / MMA_WARPS;
    return (int)(g < 148 ? (g < 1 ? 1 : g) : 148);
}

template <int NB>
static int launch_trsm_gram(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* V1,
                            int64_t ldq, double* part, int* nparts, cudaStream_t st)
{
    using Plan = SmemPlan<NB, MMA_WARPS, MMA_STAGES, 1>;
    static bool attr = false;
    if (!attr) {
        cudaFuncSetAttribute(k_trsm_gram_mma<NB, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
        cudaFuncSetAttribute(k_trsm_gram_mma<NB, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
        attr = true;
    }
    const int grid = grid_for(m);
    *nparts = grid;
    if (R0) k_trsm_gram_mma<NB, true><<<grid, MMA_WARPS * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, V1, ldq, part);
    else    k_trsm_gram_mma<NB, false><<<grid, MMA_WARPS * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, nullptr, ldq, part);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

int rqr_trsm_gram_mma(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* V1,
                      int64_t ldq, double* part, int* nparts, cudaStream_t st)
{
    if (!fast_ok(V, n, ldv, V1, ldq)) return RQR_TALL_NOT_HANDLED;
    if (!R0 && V1) return RQR_TALL_NOT_HANDLED;       // plain copy + Gram: generic kernel
    if (n <= 16) return launch_trsm_gram<2>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
    if (n <= 32) return launch_trsm_gram<4>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
    return launch_trsm_gram<8>(V, m, n, ldv, R0, V1, ldq, part, nparts, st);
}

template <int NB>
static int launch_apply(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                        double* Q, int64_t ldq, cudaStream_t st)
{
    using Plan = SmemPlan<NB, MMA_WARPS, MMA_STAGES, 2>;
    static bool attr = false;
    if (!attr) {
        cudaFuncSetAttribute(k_apply_mma<NB, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
        cudaFuncSetAttribute(k_apply_mma<NB, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
        attr = true;
    }
    const int grid = grid_for(m);
    if (R0) k_apply_mma<NB, true><<<grid, MMA_WARPS * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, R1, Q, ldq);
    else    k_apply_mma<NB, false><<<grid, MMA_WARPS * 32, Plan::bytes, st>>>(V, m, n, ldv, R0, R1, Q, ldq);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

int rqr_apply_mma(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                  double* Q, int64_t ldq, cudaStream_t st)
{
    if (!fast_ok(V, n, ldv, Q, ldq)) return RQR_TALL_NOT_HANDLED;
    if (n <= 16) return launch_apply<2>(V, m, n, ldv, R0, R1, Q, ldq, st);
    if (n <= 32) return launch_apply<4>(V, m, n, ldv, R0, R1, Q, ldq, st);
    return launch_apply<8>(V, m, n, ldv, R0, R1, Q, ldq, st);
}
