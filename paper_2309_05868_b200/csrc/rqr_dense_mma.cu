// rqr_dense_mma.cu -- B'': the single dense Gaussian sketch W = S V on the FP64 tensor
// pipe.  S (s x m_total, N(0,1)/sqrt(s), Philox stream 3, reading S3) is never stored: every lane DRAWS the
// entries of its own A fragment in registers.
//
// One k-block = 8 rows of V.  For an 8-row tile of S (sketch rows sr0 .. sr0+7) and the k-block i0 .. i0+7, lane
// (r = lane / 4, k = lane % 4) draws ONE Box-Muller pair: the entries S[sr0 + r][i0 + 2k] and S[sr0 + r][i0 + 2k + 1]
// (adjacent entries of a row of S are the two outputs of one Philox counter whenever the first index is even).
// The 8 x 8 x 8 product is two mma.sync.m8n8k4.f64 with the contraction index permuted: piece 0 contracts over the
// even rows of the k-block (A = z_even, B = V[i0 + 2k][8j + c]), piece 1 over the odd rows -- so one draw per lane
// feeds 2 NBN DMMAs and S needs no shared memory at all.  V tiles (32 rows) are staged by bulk async copies
// (one per row), the B fragments of a k-block are shared by the RT row tiles of a warp.
//
// FP64 budget per 8 x 8 tile of S (n = 64): 16 DMMA = 256 cycles of the FP64 data path, and the draw itself
// (Philox on the integer pipe; log, sqrt, sincospi: ~80 FP64 instructions per pair) another ~160 cycles of the SAME
// data path (DFMA and DMMA share it).  The roof of this kernel is therefore
// 2 m n s / P64 + (s m / 2 pairs) / (pair rate), both measured (rqr_debug_dense_gauss_draw_only).
#include "rqr_mma.cuh"

#define DM_WARPS 8
#define DM_CHUNK 32          // rows of V per stage
#define DM_STAGES 3

template <int NBN> struct DensePlan {
    static constexpr int LD = 8 * NBN + 2;                 // row stride == 2 mod 8 doubles: the B-fragment reads of
                                                           // rows 2k (k = 0..3) x 4 consecutive columns hit 32 banks
    static constexpr size_t bar_doubles = 4;               // DM_STAGES <= 4 mbarriers, the ring stays 16-byte aligned
    static constexpr size_t tab_doubles = 2 * RQR_LOG_TAB_N;   // shared-memory copy of the logarithm table
    static constexpr size_t bytes = (bar_doubles + tab_doubles + (size_t)DM_STAGES * DM_CHUNK * LD) * sizeof(double);
};

// entries S[sr][i], S[sr][i + 1] of the dense sketch (unscaled z), i = global row index
__device__ __forceinline__ void dense_pair(uint64_t seed, uint64_t e, double& z0, double& z1, const RqrLogEntry* tab)
{
    if (!(e & 1)) {
        rqr_gauss_pair(seed, e >> 1, RQR_PHILOX_STREAM_DENSE, z0, z1, tab);
    } else {                                               // odd m_total / row0: the two entries straddle two pairs
        double a, b;
        rqr_gauss_pair(seed, e >> 1, RQR_PHILOX_STREAM_DENSE, a, z0, tab);
        rqr_gauss_pair(seed, (e + 1) >> 1, RQR_PHILOX_STREAM_DENSE, z1, b, tab);
    }
}

// DMMAs [D0, D1) of a k-block, in the order j (column block), t (row tile), piece (even / odd rows of the k-block).
// The B fragments of column block j + 1 are loaded when column block j starts (one block ahead of their use).
template <int NBN, int RT, int LD, int D0, int D1>
__device__ __forceinline__ void dense_dmmas(double (&acc)[RT][NBN][2], const double (&z0)[RT], const double (&z1)[RT],
                                            const double* __restrict__ b, double (&b0)[NBN], double (&b1)[NBN])
{
    static_for<D0, D1>([&](auto dc) {
        constexpr int d = decltype(dc)::value;
        constexpr int j = d / (2 * RT), t = (d / 2) % RT, piece = d % 2;
        if constexpr (d % (2 * RT) == 0 && j + 1 < NBN) { b0[j + 1] = b[8 * (j + 1)]; b1[j + 1] = b[LD + 8 * (j + 1)]; }
        if constexpr (piece == 0) dmma(acc[t][j][0], acc[t][j][1], z0[t], b0[j]);
        else                      dmma(acc[t][j][0], acc[t][j][1], z1[t], b1[j]);
    });
}

// grid = (P row-chunk walkers, ceil(s / (64 RT)) sketch-row groups); DRAW_ONLY: no V, no DMMA (generation rate).
// PIPE (m_total and row0 even: every lane's entry pair is one Box-Muller pair): software-pipelined main loop -- the
// 16 RT stages of the draws of k-block i + 1 alternate with the 2 NBN RT DMMAs of k-block i, so that a warp reaches
// its next DMMA about when the FP64 data path has finished the last one (16 cycles each) and never queues on it.
template <int NBN, int RT, bool DRAW_ONLY, bool PIPE>
__global__ void __launch_bounds__(DM_WARPS * 32, (RT * NBN <= 16) ? 2 : 1)
k_dense_gauss_mma(const double* __restrict__ V, int64_t m, int n, int64_t ldv, int64_t row0, int64_t m_total, int s,
                  uint64_t seed, double* __restrict__ part)
{
    using Plan = DensePlan<NBN>;
    constexpr int LD = Plan::LD;
    extern __shared__ __align__(16) double smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    RqrLogEntry* tab = reinterpret_cast<RqrLogEntry*>(smem + Plan::bar_doubles);
    double* ring = smem + Plan::bar_doubles + Plan::tab_doubles;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int r = lane >> 2, k = lane & 3;
    const int64_t nchunks = (m + DM_CHUNK - 1) / DM_CHUNK;

    for (int i = threadIdx.x; i < RQR_LOG_TAB_N; i += blockDim.x) tab[i] = d_rqr_log_tab[i];
    if (DRAW_ONLY) __syncthreads();
    if (!DRAW_ONLY) {
        if (threadIdx.x < DM_STAGES) mbar_init(bars + threadIdx.x, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        for (int i = threadIdx.x; i < DM_STAGES * DM_CHUNK * LD; i += blockDim.x) ring[i] = 0.0;   // pad columns stay 0
        fence_proxy_async();
        __syncthreads();
    }
    // warp 0 stages chunk `ch` into `stage`: lane i copies row i (8n bytes)
    auto issue = [&](int stage, int64_t ch) {
        const int64_t i0 = ch * DM_CHUNK;
        const int valid = (int)((m - i0) < DM_CHUNK ? (m - i0) : DM_CHUNK);
        if (lane == 0) mbar_expect_tx(bars + stage, (uint32_t)(valid * n * 8));
        __syncwarp();
        if (lane < valid) bulk_g2s(ring + ((size_t)stage * DM_CHUNK + lane) * LD, V + (i0 + lane) * ldv, (uint32_t)(n * 8), bars + stage);
    };
    if (!DRAW_ONLY && warp == 0) {
#pragma unroll
        for (int st = 0; st < DM_STAGES; ++st)
            if ((int64_t)blockIdx.x + (int64_t)st * gridDim.x < nchunks) issue(st, blockIdx.x + (int64_t)st * gridDim.x);
    }

    double acc[RT][NBN][2];
#pragma unroll
    for (int t = 0; t < RT; ++t)
#pragma unroll
        for (int j = 0; j < NBN; ++j) { acc[t][j][0] = 0.0; acc[t][j][1] = 0.0; }
    // this lane's sketch rows and their first entry index (row-major S: e = sr * m_total + global row)
    int sr[RT];
    uint64_t ebase[RT];
#pragma unroll
    for (int t = 0; t < RT; ++t) {
        sr[t] = blockIdx.y * (64 * RT) + 8 * (warp * RT + t) + r;
        // rows past s (a ragged last tile) draw row s - 1 again: their accumulators are never stored
        ebase[t] = (uint64_t)(sr[t] < s ? sr[t] : s - 1) * (uint64_t)m_total + (uint64_t)row0 + (uint64_t)(2 * k);
    }

    const bool tile_live = blockIdx.y * (64 * RT) + 8 * (warp * RT) < s;       // warp-uniform
    double z0[RT], z1[RT];
    RqrPairDraw dr[RT];
    if (PIPE && tile_live) {                                            // prologue: the draws of this CTA's first k-block
#pragma unroll
        for (int t = 0; t < RT; ++t) {
            dr[t].begin(seed, (ebase[t] + (uint64_t)blockIdx.x * DM_CHUNK) >> 1, RQR_PHILOX_STREAM_DENSE);
            rqr_pair_draw_run<0>(dr[t], tab);
            z0[t] = dr[t].z0; z1[t] = dr[t].z1;
        }
    }
    int stage = 0;
    uint32_t phase = 0;
    for (int64_t ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
        const int64_t i0 = ch * DM_CHUNK;
        const double* Vs = ring + (size_t)stage * DM_CHUNK * LD;
        if (!DRAW_ONLY) {
            mbar_wait(bars + stage, phase);
            const int valid = (int)((m - i0) < DM_CHUNK ? (m - i0) : DM_CHUNK);
            if (valid < DM_CHUNK) {                        // rows past the end hold an older chunk: zero them
                double* z = ring + ((size_t)stage * DM_CHUNK + valid) * LD;
                for (int e = threadIdx.x; e < (DM_CHUNK - valid) * LD; e += blockDim.x) z[e] = 0.0;
                __syncthreads();
            }
        }
#pragma unroll 1
        for (int kb = 0; kb < DM_CHUNK / 8; ++kb) {
            const double* b = Vs + (size_t)(8 * kb + 2 * k) * LD + r;     // rows 2k, 2k+1 of the k-block, column 8j + r
            if (!tile_live) {
                // this warp's row tiles all lie past s (s < 64 RT): nothing to draw, its accumulators are never stored
            } else if (PIPE) {
                // first row of the NEXT k-block of this CTA (past the end: drawn and never used)
                const int64_t inext = (kb + 1 < DM_CHUNK / 8) ? i0 + 8 * (kb + 1) : (ch + gridDim.x) * DM_CHUNK;
#pragma unroll
                for (int t = 0; t < RT; ++t) dr[t].begin(seed, (ebase[t] + (uint64_t)inext) >> 1, RQR_PHILOX_STREAM_DENSE);
                constexpr int NS = RqrPairDraw::NSTAGES * RT, ND = DRAW_ONLY ? 0 : 2 * NBN * RT;
                double b0[NBN], b1[NBN];
                if (!DRAW_ONLY) { b0[0] = b[0]; b1[0] = b[LD]; }
                static_for<0, NS>([&](auto Sc) {
                    constexpr int S = decltype(Sc)::value;
                    dr[S % RT].template stage<S / RT>(tab);         // the RT draws advance together: independent chains
                    if constexpr (!DRAW_ONLY)
                        dense_dmmas<NBN, RT, LD, (S * ND) / NS, ((S + 1) * ND) / NS>(acc, z0, z1, b, b0, b1);
                });
                if (DRAW_ONLY) {
#pragma unroll
                    for (int t = 0; t < RT; ++t) { acc[t][0][0] += z0[t]; acc[t][0][1] += z1[t]; }
                }
#pragma unroll
                for (int t = 0; t < RT; ++t) { z0[t] = dr[t].z0; z1[t] = dr[t].z1; }
            } else {
#pragma unroll
                for (int t = 0; t < RT; ++t) dense_pair(seed, ebase[t] + (uint64_t)(i0 + 8 * kb), z0[t], z1[t], tab);
                if (DRAW_ONLY) {
#pragma unroll
                    for (int t = 0; t < RT; ++t) { acc[t][0][0] += z0[t]; acc[t][0][1] += z1[t]; }
                } else {
#pragma unroll
                    for (int j = 0; j < NBN; ++j) {
                        const double c0 = b[8 * j], c1 = b[LD + 8 * j];
#pragma unroll
                        for (int t = 0; t < RT; ++t) {
                            dmma(acc[t][j][0], acc[t][j][1], z0[t], c0);
                            dmma(acc[t][j][0], acc[t][j][1], z1[t], c1);
                        }
                    }
                }
            }
        }
        if (!DRAW_ONLY) {
            __syncthreads();                               // every warp is done with this stage
            if (warp == 0) {
                const int64_t next = ch + (int64_t)DM_STAGES * gridDim.x;
                if (next < nchunks) {
                    fence_proxy_async();
                    issue(stage, next);
                }
            }
            if (++stage == DM_STAGES) { stage = 0; phase ^= 1u; }
        }
    }
    // this walker's partial of W: rows sr (C fragment: row r, columns 8j + 2k, 8j + 2k + 1), scaled by 1/sqrt(s) once
    const double d = sqrt((double)s);
#pragma unroll
    for (int t = 0; t < RT; ++t) {
        if (sr[t] < s) {
            double* P = part + ((int64_t)blockIdx.x * s + sr[t]) * n;
#pragma unroll
            for (int j = 0; j < NBN; ++j) {
                const int c = 8 * j + 2 * k;
                if (c + 1 < n) *reinterpret_cast<double2*>(P + c) = make_double2(acc[t][j][0] / d, acc[t][j][1] / d);
                else if (c < n) P[c] = acc[t][j][0] / d;
            }
        }
    }
}

template <int NBN, int RT, bool DRAW_ONLY, bool PIPE>
static int launch_dense_mma(const double* V, int64_t m, int n, int64_t ldv, int64_t row0, int64_t m_total, int s,
                            uint64_t seed, double* part, int64_t Pcap, int* P_out, cudaStream_t st)
{
    using Plan = DensePlan<NBN>;
    static_assert(Plan::bytes <= ((RT * NBN <= 16) ? 113 : 227) * 1024, "shared memory plan too large for the CTAs per SM");
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_dense_gauss_mma<NBN, RT, DRAW_ONLY, PIPE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
    });
    const int groups = (s + 64 * RT - 1) / (64 * RT);
    const int per_sm = (RT * NBN <= 16) ? 2 : 1;
    const int64_t nchunks = (m + DM_CHUNK - 1) / DM_CHUNK;
    int64_t P = (148 * per_sm) / groups;
    if (P > Pcap) P = Pcap;
    if (P > nchunks) P = nchunks;
    if (P < 1) P = 1;
    dim3 grid((unsigned)P, (unsigned)groups);
    k_dense_gauss_mma<NBN, RT, DRAW_ONLY, PIPE><<<grid, DM_WARPS * 32, Plan::bytes, st>>>(V, m, n, ldv, row0, m_total, s, seed, part);
    RQR_LAUNCH_CHECK();
    *P_out = (int)P;
    return RQR_OK;
}

// Returns RQR_TALL_NOT_HANDLED when the shape needs the generic kernel (odd n or ld, unaligned base).
int rqr_dense_gauss_mma(const double* V, int64_t m, int n, int64_t ldv, int64_t row0, int64_t m_total, int s,
                        uint64_t seed, double* part, int64_t Pcap, int* P_out, bool draw_only, cudaStream_t st)
{
    if ((n & 1) || (ldv & 1) || (((uintptr_t)V & 15) != 0)) return RQR_TALL_NOT_HANDLED;
    // every lane's two entries (i, i + 1 with i even) are one Box-Muller pair iff row0 and m_total are even
    const bool pipe = !((row0 | m_total) & 1);
#define DM_ARGS V, m, n, ldv, row0, m_total, s, seed, part, Pcap, P_out, st
#define DM_CASE(NBN, RT)                                                                             \
    do {                                                                                             \
        if (draw_only) return launch_dense_mma<NBN, RT, true, true>(DM_ARGS);                        \
        return pipe ? launch_dense_mma<NBN, RT, false, true>(DM_ARGS)                                \
                    : launch_dense_mma<NBN, RT, false, false>(DM_ARGS);                              \
    } while (0)
    if (n <= 16) { DM_CASE(2, 1); }
    if (n <= 32) { DM_CASE(4, 1); }
    if (n <= 64) { DM_CASE(8, 2); }
    if (n <= 128) { DM_CASE(16, 2); }
    DM_CASE(32, 1);
#undef DM_CASE
#undef DM_ARGS
}
