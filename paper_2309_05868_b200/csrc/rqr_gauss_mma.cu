// rqr_gauss_mma.cu -- A2 for n >= 96 (and large products from n = 32): W = S2 W1 as a split-K FP64
// DMMA GEMM.  At n = 256 this step is 34 GFLOP over 0.8 GB (C4): FP64-bound, 8% of the path's flops.
// CTA (y = 64-row tile of S2, z = K chunk): 8 consumer warps, warp w owns rows 8w..8w+7 of the tile and
// all n columns (NBN accumulator blocks in registers); a producer warp stages 16-deep K slices of W1 (16 x n) with
// per-row bulk async copies into padded rows (stride n+4 doubles: the B-fragment reads are bank-conflict free), 4 stages,
// full/empty mbarriers; the A fragments (S2) come straight from global memory, one slice ahead in registers: every entry
// of S2 is used by exactly one warp.  Partials go to the caller's buffer and are reduced in fixed order by
// k_reduce_partials.
// RAD (N4): S2 is the dense Rademacher matrix of reading S21; nothing of S2 is read, every lane
// forms its A-fragment entries +-1/sqrt(s2) from the Philox words of its row (one call per 128 columns).
#include "rqr_mma.cuh"

#define GM_KB 16
#define GM_STAGES 4
#define GM_WARPS 8

__device__ __forceinline__ void gm_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_u32(bar)) : "memory");
}

template <int NBN>
struct GaussPlan {
    static constexpr int LDB = 8 * NBN + 4;
    static constexpr size_t b_doubles = (size_t)GM_KB * LDB;
    static constexpr size_t stage = b_doubles;          // only W1 is staged: every entry of S2 is used by ONE warp
    static constexpr size_t bars = GM_STAGES * stage;
    static constexpr size_t bytes = (bars + 2 * GM_STAGES) * sizeof(double);
};

template <int NBN, bool RAD>
__global__ void __launch_bounds__((GM_WARPS + 1) * 32, 1)
k_gauss_gemm_mma(const double* __restrict__ S2, const double* __restrict__ W1, int64_t s1, int n, int s2,
                 int64_t kchunk, double* __restrict__ part, uint64_t seed)
{
    using Plan = GaussPlan<NBN>;
    constexpr int LDB = Plan::LDB;
    extern __shared__ __align__(16) double smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + Plan::bars);
    uint64_t* empty = full + GM_STAGES;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < (int)Plan::bars; i += blockDim.x) smem[i] = 0.0;
    if (threadIdx.x < GM_STAGES) mbar_init(full + threadIdx.x, 1);
    else if (threadIdx.x < 2 * GM_STAGES) mbar_init(empty + (threadIdx.x - GM_STAGES), GM_WARPS);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
    __syncthreads();

    const int m0 = blockIdx.y * 64;
    const int64_t k0 = (int64_t)blockIdx.z * kchunk;
    const int64_t k1 = (k0 + kchunk < s1) ? k0 + kchunk : s1;
    const int nsteps = (int)((k1 - k0 + GM_KB - 1) / GM_KB);
    const int64_t lds2 = rqr_s2_ld(s1);                 // rows of S2 are padded with zeros to a multiple of 16

    if (warp == GM_WARPS) {
        int stage = 0;
        uint32_t ph = 0;
        for (int s = 0; s < nsteps; ++s) {
            const int64_t k = k0 + (int64_t)s * GM_KB;
            double* B = smem + (size_t)stage * Plan::stage;
            mbar_wait(empty + stage, ph ^ 1u);
            // the last slice may run past s1: S2's pad columns are zero, the matching rows of the B stage
            // keep finite data of an earlier slice (0 x finite = 0), so only the existing rows of W1 are copied
            const int rows_b = (int)((s1 - k) < GM_KB ? (s1 - k) : GM_KB);
            if (lane == 0) mbar_expect_tx(full + stage, (uint32_t)(rows_b * n * 8));
            __syncwarp();
            if (lane < rows_b) bulk_g2s(B + lane * LDB, W1 + (k + lane) * n, (uint32_t)(n * 8), full + stage);
            if (++stage == GM_STAGES) { stage = 0; ph ^= 1u; }
        }
        return;
    }
    const int r = lane >> 2, q = lane & 3;
    double acc[NBN][2];
#pragma unroll
    for (int b = 0; b < NBN; ++b) { acc[b][0] = 0.0; acc[b][1] = 0.0; }
    int stage = 0;
    uint32_t ph = 0;
    const uint64_t ng = (uint64_t)((s1 + 127) >> 7);
    const double inv = 1.0 / sqrt((double)s2);
    uint32_t o[4] = {0u, 0u, 0u, 0u};
    int64_t gcur = -1;
    // A fragments straight from global memory: lane (r, q) needs S2[m0 + 8 warp + r][k + 4 j + q], j < 4, of every
    // K slice -- one 32-byte sector per row and load, each entry of S2 read by exactly one lane of the grid, so
    // staging it in shared memory bought nothing and cost 64 bulk copies of 128 bytes per slice (measured: the
    // Rademacher form, which stages no A, ran the same product in 0.52 against 0.83 ms).  One slice ahead in registers.
    const int arow = m0 + 8 * warp + r;
    const double* Ag = RAD ? nullptr : S2 + (int64_t)(arow < s2 ? arow : 0) * lds2 + k0 + q;
    const bool aok = !RAD && arow < s2;
    double acur[GM_KB / 4], anext[GM_KB / 4];
#pragma unroll
    for (int j = 0; j < GM_KB / 4; ++j) { acur[j] = (aok && nsteps > 0) ? __ldg(Ag + 4 * j) : 0.0; anext[j] = 0.0; }
    for (int s = 0; s < nsteps; ++s) {
        const double* B = smem + (size_t)stage * Plan::stage + q * LDB + r;
        if (aok && s + 1 < nsteps) {
#pragma unroll
            for (int j = 0; j < GM_KB / 4; ++j) anext[j] = __ldg(Ag + (int64_t)(s + 1) * GM_KB + 4 * j);
        }
        uint32_t bits = 0;
        const int64_t kcol = k0 + (int64_t)s * GM_KB;
        if (RAD) {
            const int64_t g = kcol >> 7;
            if (g != gcur) {
                rqr_rademacher_bits(seed, (uint32_t)(m0 + 8 * warp + r), ng, (uint64_t)g, o);
                gcur = g;
            }
            const int b0 = (int)(kcol & 127);
            const uint32_t word = b0 < 64 ? (b0 < 32 ? o[0] : o[1]) : (b0 < 96 ? o[2] : o[3]);
            bits = word >> ((b0 & 31) + q);                    // bit 4 j: column kcol + 4 j + q
        }
        mbar_wait(full + stage, ph);
#pragma unroll
        for (int kk = 0; kk < GM_KB; kk += 4) {
            double a;
            if (RAD) a = (kcol + kk + q < s1) ? (((bits >> kk) & 1u) ? -inv : inv) : 0.0;
            else a = acur[kk / 4];
#pragma unroll
            for (int b = 0; b < NBN; ++b) dmma(acc[b][0], acc[b][1], a, B[kk * LDB + 8 * b]);
        }
        __syncwarp();
        if (lane == 0) gm_arrive(empty + stage);
        if (++stage == GM_STAGES) { stage = 0; ph ^= 1u; }
#pragma unroll
        for (int j = 0; j < GM_KB / 4; ++j) acur[j] = anext[j];
    }
    double* P = part + (int64_t)blockIdx.z * s2 * n;
    const int row = m0 + 8 * warp + r;
    if (row < s2) {
#pragma unroll
        for (int b = 0; b < NBN; ++b) {
            const int col = 8 * b + 2 * q;
            if (col < n) P[(int64_t)row * n + col] = acc[b][0];
            if (col + 1 < n) P[(int64_t)row * n + col + 1] = acc[b][1];
        }
    }
}

#ifndef RQR_GAUSS_MMA_MIN_STEPS
#define RQR_GAUSS_MMA_MIN_STEPS 8
#endif
template <int NBN, bool RAD>
static int launch_gauss_mma(const double* S2, const double* W1, int64_t s1, int n, int s2, double* part,
                            int64_t ks_cap, int* ks_out, cudaStream_t st, uint64_t seed)
{
    using Plan = GaussPlan<NBN>;
    static_assert(Plan::bytes <= 227 * 1024, "k_gauss_gemm_mma shared memory plan too large");
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_gauss_gemm_mma<NBN, RAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
    });
    const int tiles_m = (s2 + 63) / 64;
    const int64_t kblocks = (s1 + GM_KB - 1) / GM_KB;
    // Resident CTAs: one per SM at NBN >= 24 (141 / 174 KB of shared memory), two at NBN = 16 (108 KB).  The K split
    // that fills whole waves of those slots best, at most 296 CTAs, the larger split on a tie (C4: 8 row tiles x 18 =
    // 144 CTAs in one wave of 148 instead of 8 x 32 = 256 in 1.73 waves: 1.29 -> 1.14 ms).
    const int64_t slots = 148 * (Plan::bytes * 3 <= 227 * 1024 ? 3 : (Plan::bytes * 2 <= 227 * 1024 ? 2 : 1));
    int64_t kmax = 2 * slots / tiles_m;
    if (kmax > ks_cap) kmax = ks_cap;
    if (kmax > kblocks / RQR_GAUSS_MMA_MIN_STEPS) kmax = kblocks / RQR_GAUSS_MMA_MIN_STEPS;   // >= that many K slices per CTA
    if (kmax < 1) kmax = 1;
    int64_t ks = 1;
    double best = 0.0;
    for (int64_t k = 1; k <= kmax; ++k) {
        const int64_t ctas = tiles_m * k, waves = (ctas + slots - 1) / slots;
        const double eff = (double)ctas / (double)(waves * slots);
        if (eff >= best - 1e-12) { best = eff; ks = k; }
    }
    const int64_t kchunk = ((kblocks + ks - 1) / ks) * GM_KB;
    ks = (s1 + kchunk - 1) / kchunk;
    dim3 grid(1, tiles_m, (unsigned)ks);
    k_gauss_gemm_mma<NBN, RAD><<<grid, (GM_WARPS + 1) * 32, Plan::bytes, st>>>(S2, W1, s1, n, s2, kchunk, part, seed);
    RQR_LAUNCH_CHECK();
    *ks_out = (int)ks;
    return RQR_OK;
}

// returns RQR_TALL_NOT_HANDLED when the shape is left to the DFMA kernel; S2 == NULL: Rademacher S2 from `seed`.
// n >= 96: always.  32 <= n < 96: for s2 >= 128 rows and s2 s1 n >= 5e7: the paper-grid sketches (s2 = 600 ... 840 rows
// by s1 = 7 000 ... 67 000: 2-3x the DFMA kernel) and the BASELINE sketch at n = 64 (128 x 8192: 19.7 -> 14.5 us with at
// least 8 K slices per CTA, i.e. 64 partials instead of 148 for the reduction); smaller ones stay on the DFMA split-K
// kernel (same time on either: launch + reduction).
#ifndef RQR_GAUSS_MMA_MIN_WORK
#define RQR_GAUSS_MMA_MIN_WORK 5.0e7      // s2 * s1 * n
#endif
#ifndef RQR_GAUSS_MMA_MIN_S2
#define RQR_GAUSS_MMA_MIN_S2 128
#endif
template <bool RAD>
static int gauss_mma_dispatch(const double* S2, const double* W1, int64_t s1, int n, int s2, double* part,
                              int64_t ks_cap, int* ks_out, cudaStream_t st, uint64_t seed)
{
    if (n <= 64) return launch_gauss_mma<8, RAD>(S2, W1, s1, n, s2, part, ks_cap, ks_out, st, seed);
    if (n <= 80) return launch_gauss_mma<10, RAD>(S2, W1, s1, n, s2, part, ks_cap, ks_out, st, seed);
    if (n <= 96) return launch_gauss_mma<12, RAD>(S2, W1, s1, n, s2, part, ks_cap, ks_out, st, seed);
    if (n <= 112) return launch_gauss_mma<14, RAD>(S2, W1, s1, n, s2, part, ks_cap, ks_out, st, seed);
    if (n <= 128) return launch_gauss_mma<16, RAD>(S2, W1, s1, n, s2, part, ks_cap, ks_out, st, seed);
    if (n <= 192) return launch_gauss_mma<24, RAD>(S2, W1, s1, n, s2, part, ks_cap, ks_out, st, seed);
    return launch_gauss_mma<32, RAD>(S2, W1, s1, n, s2, part, ks_cap, ks_out, st, seed);
}

int rqr_gauss_gemm_mma(const double* S2, const double* W1, int64_t s1, int n, int s2, double* part,
                       int64_t ks_cap, int* ks_out, cudaStream_t st, uint64_t seed)
{
    if (n < 32 || n > 256 || (n & 1)) return RQR_TALL_NOT_HANDLED;
    if (n < 96 && ((double)s2 * (double)s1 * n < RQR_GAUSS_MMA_MIN_WORK || s2 < RQR_GAUSS_MMA_MIN_S2)) return RQR_TALL_NOT_HANDLED;
    if ((((uintptr_t)S2 | (uintptr_t)W1) & 15) != 0) return RQR_TALL_NOT_HANDLED;
    if (S2) return gauss_mma_dispatch<false>(S2, W1, s1, n, s2, part, ks_cap, ks_out, st, seed);
    return gauss_mma_dispatch<true>(S2, W1, s1, n, s2, part, ks_cap, ks_out, st, seed);
}
