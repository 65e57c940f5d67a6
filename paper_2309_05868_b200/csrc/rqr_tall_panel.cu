// rqr_tall_panel.cu -- FP64 DMMA paths of A4 (rqr_trsm_gram) and A6 (rqr_apply) for 64 < n <= 256.
//
// For n >= 128 both halves of A4 are FP64-bound on B200 (n/8 and n/4 flop/byte against a ridge of
// 5.7), so fusing them saves nothing; and the Gram accumulator (n^2/2 doubles) no longer fits next
// to the substitution state in one SM's register file.  A4 is therefore two kernels:
//   k_trsm_panel  X = V R^-1 (row-wise blocked substitution, eq. (42)), stores X
//   k_syrk_fold   G = X^T X partials (Alg. 2 step 1)
// and A6 is k_trsm_panel in place.  ("large n".)
//
// k_trsm_panel: columns in panels of 64.  A warp owns an 8-row block; the whole block (NP panels
// x 8 C fragments) lives in registers.  For panel P:  x_P -= x_P' R[P',P] (P' < P; 128 independent
// DMMAs per pair), then the in-panel chain with R[P,P] (trsm_rowblock<8>, the routine of the
// n <= 64 kernels).  The B fragments of one (P',P) step are a 32 KB slot, prebuilt in global memory
// by k_build_panel_frags and streamed through a CTA-wide double buffer by a producer warp with
// bulk async copies (full/empty mbarriers); the 8 consumer warps use each slot once per row-block.
//
// k_syrk_fold: the upper block triangle of G (NB x NB blocks of 8 x 8, NB even) is folded into NB/2
// rows of NB+1 blocks -- fold f = {(f, b): b >= f} + {(NB-1-f, b): b >= NB-1-f} -- one fold per warp,
// perfectly balanced; all its operands are the column-block fragments f..NB-1 of a 4-row slab, loaded
// once per slab.  Accumulators stay in registers for the whole kernel.  NB = 32 needs two CTAs
// (blockIdx.y) to hold all folds: they walk the same row tiles, the second read hits L2.
#include "rqr_mma.cuh"

#define PANEL_WARPS 8        // consumer warps of k_syrk_fold; warp PANEL_WARPS is the producer
#ifndef PANEL_CW_WIDE
#define PANEL_CW_WIDE 15     // consumer warps of k_trsm_panel for NP = 2 (PanelPlan): 16 warps = 4 per sub-partition
#endif
#define PANEL_SLOT 4096      // doubles per fragment slot (32 KB)
#define PANEL_DIAG 2304      // doubles used by a diagonal slot: Tf (8*64) + nRf (28*64)
#define SYRK_TR 32           // rows per tile of k_syrk_fold

__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_u32(bar)) : "memory");
}

// slot order: for P = 0..NP-1: off(0,P), ..., off(P-1,P), diag(P)
__host__ __device__ __forceinline__ void panel_slot_decode(int s, int& Pp, int& P)
{
    P = 0;
    while (s > P) { s -= P + 1; ++P; }
    Pp = s;                                  // Pp == P: diagonal slot
}

// One CTA per slot.  off(P',P)[((J'*8+J)*2+s)*32+lane] = -R[64P'+8J'+2(lane%4)+s][64P+8J+lane/4];
// diag(P) = the Tf / nRf arrays of build_tri_frags for the 64x64 block R[P,P].  Padded with identity.
// last_nb = 2, 4, 6: the last panel is 16, 32, 48 columns wide (n <= 64 (NP-1) + 8 last_nb); its diagonal slot
// holds the NB = last_nb arrays (Tf NB*64, nRf NB(NB-1)/2*64 doubles), its off-diagonal slots are used for
// J < last_nb only.
__global__ void __launch_bounds__(256)
k_build_panel_frags(const double* __restrict__ R, int n, double* __restrict__ frags, int np, int last_nb)
{
    __shared__ double scratch[8 * 64];
    __shared__ double stage[64 * 64];
    int Pp, P;
    panel_slot_decode(blockIdx.x, Pp, P);
    double* out = frags + (size_t)blockIdx.x * PANEL_SLOT;
    if (Pp == P) {
        const int nb = (P == np - 1) ? last_nb : 8;
        if (nb == 2) build_tri_frags<2>(R, n, out, out + 128, scratch, stage, 64 * P);
        else if (nb == 4) build_tri_frags<4>(R, n, out, out + 256, scratch, stage, 64 * P);
        else if (nb == 6) build_tri_frags<6>(R, n, out, out + 384, scratch, stage, 64 * P);
        else build_tri_frags<8>(R, n, out, out + 512, scratch, stage, 64 * P);
    } else {
        for (int t = threadIdx.x; t < PANEL_SLOT; t += blockDim.x) {
            const int jj = t >> 6, h = (t >> 5) & 1, lane = t & 31;
            const int Jp = jj >> 3, J = jj & 7;
            out[t] = -r_padded(R, n, 64 * Pp + 8 * Jp + 2 * (lane & 3) + h, 64 * P + 8 * J + (lane >> 2));
        }
    }
}

template <int NP>
struct PanelPlan {
    // consumer warps of k_trsm_panel: 15 (+ the producer = 4 per SM sub-partition, 128 registers each; the kernel
    // needs 116) at NP = 2 (measured A/B in one process at 2^22 rows: n = 128 A6 2.283 ms with 11 warps, 2.522 with 13
    // -- an odd number of warps per sub-partition pair --, 2.207 with 15; n = 96 1.385 / 1.551 / 1.327), 8 above
    // (NP = 3: 2.46 vs 2.49 ms with 11; NP = 4: one 8 x 264-double landing block per warp is 17 KB)
    static constexpr int CW = (NP == 2) ? PANEL_CW_WIDE : 8;
    static constexpr int N8 = 64 * NP;
    static constexpr int LDL = N8 + LDL_PAD;
    static constexpr int STEPS = NP * (NP + 1) / 2;
    static constexpr int LSTAGES = (NP <= 2 && CW <= 8) ? 2 : 1;
    static constexpr int NBARS = 4 + CW * LSTAGES;       // full[2], empty[2], landing
    static constexpr size_t bars = 2 * PANEL_SLOT;                // doubles
    static constexpr size_t ring = bars + ((NBARS + 1) & ~1);
    static constexpr size_t ring_doubles = (size_t)CW * LSTAGES * 8 * LDL;
    static constexpr size_t bytes = (ring + ring_doubles) * sizeof(double);
};

// X = V R^-1 (npass = 1) or (V Ra^-1) Rb^-1 (npass = 2; fragment sets Ra then Rb), X -> Q.
// LASTNB = 2, 4, 6: the last panel has LASTNB column blocks (n <= 64 (NP-1) + 8 LASTNB): its DMMAs for
// J >= LASTNB are skipped.
template <int NP, bool FULL, int LASTNB>
__global__ void __launch_bounds__((PanelPlan<NP>::CW + 1) * 32, 1)
k_trsm_panel(const double* V, int64_t m, int n, int64_t ldv, const double* __restrict__ frags,
             int npass, double* Q, int64_t ldq)
{
    using Plan = PanelPlan<NP>;
    constexpr int LDL = Plan::LDL, STEPS = Plan::STEPS, LST = Plan::LSTAGES;
    extern __shared__ __align__(16) double smem[];
    double* Bbuf = smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Plan::bars);
    uint64_t* full = bars;
    uint64_t* empty = bars + 2;
    uint64_t* land = bars + 4;
    double* ring = smem + Plan::ring;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    for (int i = threadIdx.x; i < (int)Plan::ring_doubles; i += blockDim.x) ring[i] = 0.0;
    if (threadIdx.x < 2) mbar_init(full + threadIdx.x, 1);
    else if (threadIdx.x < 4) mbar_init(empty + (threadIdx.x - 2), Plan::CW);
    else if (threadIdx.x < Plan::NBARS) mbar_init(bars + threadIdx.x, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
    __syncthreads();

    const int64_t nrb = (m + 7) / 8;
    const int64_t ntiles = (nrb + Plan::CW - 1) / Plan::CW;

    if (warp == Plan::CW) {
        // producer: streams the fragment slots, in consumption order, for every tile of this CTA
        if (lane == 0) {
            int buf = 0;
            uint32_t ph = 0;
            for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x)
                for (int pass = 0; pass < npass; ++pass)
                    for (int s = 0; s < STEPS; ++s) {
                        int Pp, P;
                        panel_slot_decode(s, Pp, P);
                        const uint32_t bytes = (uint32_t)((Pp == P ? PANEL_DIAG : PANEL_SLOT) * sizeof(double));
                        mbar_wait(empty + buf, ph ^ 1u);
                        mbar_expect_tx(full + buf, bytes);
                        bulk_g2s(Bbuf + (size_t)buf * PANEL_SLOT,
                                 frags + ((size_t)pass * STEPS + s) * PANEL_SLOT, bytes, full + buf);
                        if (++buf == 2) { buf = 0; ph ^= 1u; }
                    }
        }
        return;
    }

    WarpRing<LDL> wr{ring + (size_t)warp * LST * 8 * LDL, land + warp * LST, V, ldv, m, n};
    const XsAddr<64> ad(lane);
    const int r = lane >> 2, q = lane & 3;
    const int64_t lane_off = (int64_t)r * ldq + 2 * q;
    uint32_t colmask[NP];
#pragma unroll
    for (int P = 0; P < NP; ++P) colmask[P] = col_mask<8>(n - 64 * P, lane);
#pragma unroll
    for (int s = 0; s < LST; ++s) {
        const int64_t t = blockIdx.x + (int64_t)s * gridDim.x;
        if (t < ntiles && t * Plan::CW + warp < nrb) wr.issue(s, t * Plan::CW + warp, lane);
    }

    double x[NP][8][2];
    double g[8];
    double G[36][2];        // unused by trsm_rowblock<.., GRAM = false>: optimised away
    int lstage = 0, buf = 0;
    uint32_t lphase = 0, fph = 0;
    auto nohook = []() {};
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t rblk = tile * Plan::CW + warp;
        const bool active = rblk < nrb;
        int valid = 0;
        if (active) {
            mbar_wait(wr.bar + lstage, lphase);
            double* rb = wr.buf + lstage * 8 * LDL;
            valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
            if (valid < 8) {
                for (int e = lane; e < (8 - valid) * LDL; e += 32) rb[valid * LDL + e] = 0.0;
                __syncwarp();
            }
#pragma unroll
            for (int P = 0; P < NP; ++P)
#pragma unroll
                for (int J = 0; J < 8; ++J) {
                    double2 v = *reinterpret_cast<const double2*>(rb + r * LDL + 64 * P + 8 * J + 2 * q);
                    x[P][J][0] = v.x; x[P][J][1] = v.y;
                }
            // the whole row-block is in registers: refill the stage for the tile LST rounds ahead
            const int64_t nt = tile + (int64_t)LST * gridDim.x;
            if (nt < ntiles && nt * Plan::CW + warp < nrb) {
                fence_proxy_async();
                __syncwarp();
                wr.issue(lstage, nt * Plan::CW + warp, lane);
            }
        } else {
#pragma unroll
            for (int P = 0; P < NP; ++P)
#pragma unroll
                for (int J = 0; J < 8; ++J) { x[P][J][0] = 0.0; x[P][J][1] = 0.0; }
        }
        if (++lstage == LST) { lstage = 0; lphase ^= 1u; }
        double* gp = (active && r < valid) ? Q + rblk * 8 * ldq + lane_off : nullptr;
        for (int pass = 0; pass < npass; ++pass) {
            double* gpp = (pass == npass - 1) ? gp : nullptr;
            static_for<0, NP>([&](auto Pc) {
                constexpr int P = decltype(Pc)::value;
                constexpr int NBP = (P == NP - 1) ? LASTNB : 8;        // column blocks of this panel
                static_for<0, P>([&](auto Ppc) {
                    constexpr int Pp = decltype(Ppc)::value;
                    mbar_wait(full + buf, fph);
                    const double* B = Bbuf + (size_t)buf * PANEL_SLOT + lane;
#pragma unroll
                    for (int Jp = 0; Jp < 8; ++Jp) {
#pragma unroll
                        for (int J = 0; J < NBP; ++J)
                            dmma(x[P][J][0], x[P][J][1], x[Pp][Jp][0], B[((Jp * 8 + J) * 2 + 0) * 32]);
#pragma unroll
                        for (int J = 0; J < NBP; ++J)
                            dmma(x[P][J][0], x[P][J][1], x[Pp][Jp][1], B[((Jp * 8 + J) * 2 + 1) * 32]);
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty + buf);
                    if (++buf == 2) { buf = 0; fph ^= 1u; }
                });
                mbar_wait(full + buf, fph);
                const double* B = Bbuf + (size_t)buf * PANEL_SLOT;
                if constexpr (NBP == 8) {
                    trsm_rowblock<8, false, false, FULL>(x[P], nullptr, nullptr, ad, B, B + 512,
                                                         gpp ? gpp + 64 * P : nullptr, colmask[P], lane, g, G, nohook);
                } else {
                    double gl[NBP];
                    double Gl[NBP * (NBP + 1) / 2][2];
                    const XsAddr<8 * NBP> adl(lane);
                    trsm_rowblock<NBP, false, false, FULL>(reinterpret_cast<double (&)[NBP][2]>(x[P]), nullptr, nullptr, adl,
                                                           B, B + 64 * NBP, gpp ? gpp + 64 * P : nullptr, colmask[P], lane,
                                                           gl, Gl, nohook);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + buf);
                if (++buf == 2) { buf = 0; fph ^= 1u; }
            });
        }
    }
}

// ------------------------------------------------------------------------------------------
// k_syrk_fold
// ------------------------------------------------------------------------------------------
template <int NB>
struct SyrkPlan {
    static constexpr int N8 = 8 * NB;
    static constexpr int LDS = N8 + 4;          // row stride = 8 words mod 32: Gram-fragment reads conflict free
    static constexpr int STAGES = (NB <= 16) ? 5 : (NB <= 24 ? 4 : 3);
    static constexpr size_t stage_doubles = (size_t)SYRK_TR * LDS;
    static constexpr size_t bars = STAGES * stage_doubles;
    static constexpr size_t bytes = (bars + 2 * STAGES) * sizeof(double);
};

// consumer warp owning fold F (compile time): walks the CTA's tiles, then writes its NB+1 blocks
template <int NB, int F>
__device__ __forceinline__ void syrk_fold_warp(const double* __restrict__ stages, uint64_t* full, uint64_t* empty,
                                               int64_t m, int64_t ntiles, int n, int lane,
                                               double* __restrict__ P, int accumulate)
{
    using Plan = SyrkPlan<NB>;
    constexpr int LDS = Plan::LDS, NF = NB - F, A2 = NB - 1 - 2 * F;
    const int r = lane >> 2, q = lane & 3;
    double G[NB + 1][2];
#pragma unroll
    for (int b = 0; b <= NB; ++b) { G[b][0] = 0.0; G[b][1] = 0.0; }
    int stage = 0;
    uint32_t ph = 0;
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int64_t left = m - tile * SYRK_TR;
        const int valid = (int)(left < SYRK_TR ? left : SYRK_TR);
        mbar_wait(full + stage, ph);
        const double* base = stages + (size_t)stage * Plan::stage_doubles + q * LDS + r + 8 * F;
        const int nslab = (valid + 3) >> 2;
#pragma unroll 1
        for (int h = 0; h < nslab; ++h) {
            const bool ok = 4 * h + q < valid;       // rows past the end of V hold stale data
            double fr[NF];
#pragma unroll
            for (int j = 0; j < NF; ++j) fr[j] = ok ? base[(size_t)h * 4 * LDS + 8 * j] : 0.0;
#pragma unroll
            for (int j = 0; j < NF; ++j) dmma(G[j][0], G[j][1], fr[0], fr[j]);
#pragma unroll
            for (int k = 0; k <= F; ++k) dmma(G[NF + k][0], G[NF + k][1], fr[A2], fr[A2 + k]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + stage);
        if (++stage == Plan::STAGES) { stage = 0; ph ^= 1u; }
    }
#pragma unroll
    for (int b = 0; b <= NB; ++b) {
        const int a_blk = b < NF ? F : NB - 1 - F;
        const int b_blk = b < NF ? F + b : NB - 1 - F + (b - NF);
        const int row = 8 * a_blk + r, col = 8 * b_blk + 2 * q;
        // accumulate: this launch covers a later chunk of rows and adds to the partial of the first one
        // (two-level summation: no register accumulator sums more than one chunk; only this lane touches dst)
        if (row < n && col < n) P[(size_t)row * n + col] = accumulate ? P[(size_t)row * n + col] + G[b][0] : G[b][0];
        if (row < n && col + 1 < n)
            P[(size_t)row * n + col + 1] = accumulate ? P[(size_t)row * n + col + 1] + G[b][1] : G[b][1];
    }
}

template <int NB, int F>
__device__ __forceinline__ void syrk_dispatch(int f, const double* stages, uint64_t* full, uint64_t* empty,
                                              int64_t m, int64_t ntiles, int n, int lane, double* P, int accumulate)
{
    if constexpr (F < NB / 2) {
        if (f == F) syrk_fold_warp<NB, F>(stages, full, empty, m, ntiles, n, lane, P, accumulate);
        else syrk_dispatch<NB, F + 1>(f, stages, full, empty, m, ntiles, n, lane, P, accumulate);
    }
}

// grid = (row walkers, ceil(NB/2 / 8)); part[blockIdx.x] receives this walker's partial (upper blocks)
template <int NB>
__global__ void __launch_bounds__((PANEL_WARPS + 1) * 32, 1)
k_syrk_fold(const double* __restrict__ X, int64_t m, int n, int64_t ldx, double* __restrict__ part, int accumulate)
{
    using Plan = SyrkPlan<NB>;
    extern __shared__ __align__(16) double smem[];
    double* stages = smem;
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + Plan::bars);
    uint64_t* empty = full + Plan::STAGES;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < (int)Plan::bars; i += blockDim.x) stages[i] = 0.0;
    if (threadIdx.x < Plan::STAGES) mbar_init(full + threadIdx.x, 1);
    else if (threadIdx.x < 2 * Plan::STAGES) mbar_init(empty + (threadIdx.x - Plan::STAGES), PANEL_WARPS);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
    __syncthreads();
    const int64_t ntiles = (m + SYRK_TR - 1) / SYRK_TR;

    if (warp == PANEL_WARPS) {
        int stage = 0;
        uint32_t ph = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const int64_t row0 = tile * SYRK_TR;
            const int valid = (int)((m - row0) < SYRK_TR ? (m - row0) : SYRK_TR);
            mbar_wait(empty + stage, ph ^ 1u);
            if (lane == 0) mbar_expect_tx(full + stage, (uint32_t)(valid * n * 8));
            __syncwarp();
            if (lane < valid)
                bulk_g2s(stages + (size_t)stage * Plan::stage_doubles + (size_t)lane * Plan::LDS,
                         X + (row0 + lane) * ldx, (uint32_t)(n * 8), full + stage);
            if (++stage == Plan::STAGES) { stage = 0; ph ^= 1u; }
        }
        return;
    }
    // folds are split evenly over the gridDim.y CTAs of a walker (NB = 20: 5 + 5, not 8 + 2)
    const int fpp = (NB / 2 + (int)gridDim.y - 1) / (int)gridDim.y;
    const int f = blockIdx.y * fpp + warp;
    double* P = part + (size_t)blockIdx.x * n * n;
    if (warp < fpp && f < NB / 2) {
        syrk_dispatch<NB, 0>(f, stages, full, empty, m, ntiles, n, lane, P, accumulate);
    } else {
        // no fold for this warp (NB/2 not a multiple of 8): keep the empty-barrier protocol alive
        int stage = 0;
        uint32_t ph = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            mbar_wait(full + stage, ph);
            if (lane == 0) mbar_arrive(empty + stage);
            if (++stage == Plan::STAGES) { stage = 0; ph ^= 1u; }
        }
    }
}

// ------------------------------------------------------------------------------------------
// host dispatch
// ------------------------------------------------------------------------------------------
static bool panel_ok(const void* V, int n, int64_t ldv, const void* Q, int64_t ldq)
{
    if (n <= 64 || n > 256 || (n & 1) || (ldv & 1)) return false;
    if (((uintptr_t)V & 15) != 0) return false;
    if (Q && (((uintptr_t)Q & 15) != 0 || (ldq & 1))) return false;
    return true;
}

template <int NP, int LASTNB>
static int launch_panel_w(const double* V, int64_t m, int n, int64_t ldv, const double* frags, int npass,
                          double* Q, int64_t ldq, cudaStream_t st)
{
    using Plan = PanelPlan<NP>;
    static_assert(Plan::bytes <= 227 * 1024, "k_trsm_panel shared memory plan too large");
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_trsm_panel<NP, true, LASTNB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
        cudaFuncSetAttribute(k_trsm_panel<NP, false, LASTNB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
    });
    const int64_t ntiles = ((m + 7) / 8 + Plan::CW - 1) / Plan::CW;
    const int grid = (int)(ntiles < 148 ? ntiles : 148);
    const int threads = (Plan::CW + 1) * 32;
    if (n == 64 * (NP - 1) + 8 * LASTNB)
        k_trsm_panel<NP, true, LASTNB><<<grid, threads, Plan::bytes, st>>>(V, m, n, ldv, frags, npass, Q, ldq);
    else
        k_trsm_panel<NP, false, LASTNB><<<grid, threads, Plan::bytes, st>>>(V, m, n, ldv, frags, npass, Q, ldq);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// column blocks of the last panel, in steps of 16 columns (the syrk folds need an even number of blocks)
static int panel_last_nb(int n, int NP)
{
    const int rem = n - 64 * (NP - 1);
    return rem <= 16 ? 2 : rem <= 32 ? 4 : rem <= 48 ? 6 : 8;
}

template <int NP>
static int launch_panel(const double* V, int64_t m, int n, int64_t ldv, const double* frags, int npass,
                        double* Q, int64_t ldq, cudaStream_t st)
{
    switch (panel_last_nb(n, NP)) {
        case 2: return launch_panel_w<NP, 2>(V, m, n, ldv, frags, npass, Q, ldq, st);
        case 4: return launch_panel_w<NP, 4>(V, m, n, ldv, frags, npass, Q, ldq, st);
        case 6: return launch_panel_w<NP, 6>(V, m, n, ldv, frags, npass, Q, ldq, st);
        default: return launch_panel_w<NP, 8>(V, m, n, ldv, frags, npass, Q, ldq, st);
    }
}

template <int NB>
static int launch_syrk(const double* X, int64_t m, int n, int64_t ldx, double* part, int* nparts, int accumulate,
                       cudaStream_t st)
{
    using Plan = SyrkPlan<NB>;
    static_assert(Plan::bytes <= 227 * 1024, "k_syrk_fold shared memory plan too large");
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_syrk_fold<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Plan::bytes);
    });
    constexpr int PARTS = (NB / 2 + PANEL_WARPS - 1) / PANEL_WARPS;
    const int64_t ntiles = (m + SYRK_TR - 1) / SYRK_TR;
    int walkers = 148 / PARTS;
    if (ntiles < walkers) walkers = (int)ntiles;
    *nparts = walkers;
    dim3 grid(walkers, PARTS);
    k_syrk_fold<NB><<<grid, (PANEL_WARPS + 1) * 32, Plan::bytes, st>>>(X, m, n, ldx, part, accumulate);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

static int build_frags(const double* R, int n, int NP, double* frags, cudaStream_t st)
{
    k_build_panel_frags<<<NP * (NP + 1) / 2, 256, 0, st>>>(R, n, frags, NP, panel_last_nb(n, NP));
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// The syrk runs per chunk of SYRK_CHUNK_ROWS rows; the first chunk writes the partial set, the later ones add to
// it (two-level summation: a register accumulator sums at most SYRK_CHUNK_ROWS / (4 walkers) products).
#define SYRK_CHUNK_ROWS ((int64_t)1 << 21)
template <int NB>
static int launch_syrk_chunks(const double* X, int64_t m, int n, int64_t ldx, double* part, int* nparts, cudaStream_t st)
{
    int np0 = 0;
    for (int64_t r0 = 0; r0 < m; r0 += SYRK_CHUNK_ROWS) {
        const int64_t mc = (m - r0) < SYRK_CHUNK_ROWS ? (m - r0) : SYRK_CHUNK_ROWS;
        int np = 0;
        int rc = launch_syrk<NB>(X + r0 * ldx, mc, n, ldx, part, &np, r0 > 0, st);
        if (rc != RQR_OK) return rc;
        if (r0 == 0) np0 = np;                 // the first chunk is the largest: it defines every partial
    }
    *nparts = np0;
    return RQR_OK;
}

int rqr_trsm_gram_panel(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* V1,
                        int64_t ldq, double* part, int* nparts, double* frags, int64_t chunk_rows, cudaStream_t st)
{
    (void)chunk_rows;
    if (!panel_ok(V, n, ldv, V1, ldq)) return RQR_TALL_NOT_HANDLED;
    if (R0 && !V1) return -7;                       // n > 64: V1 must be stored (see include/rqr.h, hazard H1)
    if (!R0 && V1) return RQR_TALL_NOT_HANDLED;     // plain copy + Gram: generic kernel
    const int NP = (n + 63) / 64;
    const double* X = V;
    int64_t ldx = ldv;
    if (R0) {
        int rc = build_frags(R0, n, NP, frags, st);
        if (rc != RQR_OK) return rc;
        rc = NP == 2 ? launch_panel<2>(V, m, n, ldv, frags, 1, V1, ldq, st)
           : NP == 3 ? launch_panel<3>(V, m, n, ldv, frags, 1, V1, ldq, st)
                     : launch_panel<4>(V, m, n, ldv, frags, 1, V1, ldq, st);
        if (rc != RQR_OK) return rc;
        X = V1;
        ldx = ldq;
    }
    switch (8 * (NP - 1) + panel_last_nb(n, NP)) {        // column blocks: 10, 12, ..., 32
        case 10: return launch_syrk_chunks<10>(X, m, n, ldx, part, nparts, st);
        case 14: return launch_syrk_chunks<14>(X, m, n, ldx, part, nparts, st);
        case 18: return launch_syrk_chunks<18>(X, m, n, ldx, part, nparts, st);
        case 22: return launch_syrk_chunks<22>(X, m, n, ldx, part, nparts, st);
        case 26: return launch_syrk_chunks<26>(X, m, n, ldx, part, nparts, st);
        case 30: return launch_syrk_chunks<30>(X, m, n, ldx, part, nparts, st);
        case 12: return launch_syrk_chunks<12>(X, m, n, ldx, part, nparts, st);
        case 16: return launch_syrk_chunks<16>(X, m, n, ldx, part, nparts, st);
        case 20: return launch_syrk_chunks<20>(X, m, n, ldx, part, nparts, st);
        case 24: return launch_syrk_chunks<24>(X, m, n, ldx, part, nparts, st);
        case 28: return launch_syrk_chunks<28>(X, m, n, ldx, part, nparts, st);
        default: return launch_syrk_chunks<32>(X, m, n, ldx, part, nparts, st);
    }
}

int rqr_apply_panel(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                    double* Q, int64_t ldq, double* frags, cudaStream_t st)
{
    if (!panel_ok(V, n, ldv, Q, ldq)) return RQR_TALL_NOT_HANDLED;
    const int NP = (n + 63) / 64;
    const int steps = NP * (NP + 1) / 2;
    int npass = 1, rc;
    if (R0) {
        rc = build_frags(R0, n, NP, frags, st);
        if (rc != RQR_OK) return rc;
        npass = 2;
    }
    rc = build_frags(R1, n, NP, frags + (size_t)(npass - 1) * steps * PANEL_SLOT, st);
    if (rc != RQR_OK) return rc;
    return NP == 2 ? launch_panel<2>(V, m, n, ldv, frags, npass, Q, ldq, st)
         : NP == 3 ? launch_panel<3>(V, m, n, ldv, frags, npass, Q, ldq, st)
                   : launch_panel<4>(V, m, n, ldv, frags, npass, Q, ldq, st);
}
