// rqr_common.cuh -- shared device helpers of librqr (CUDA path only; the CPU oracle shares
// nothing with this file).  sm_100a.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <atomic>
#include "../../include/rqr.h"
#include "rqr_gauss.cuh"

#define RQR_MAX_N 256
#define RQR_MAX_S2 1024
#define RQR_MAX_GRAM_PARTIALS 304        // >= 2 CTAs per SM on 148 SMs (one chunk of rows)
#define RQR_GRAM_CHUNK_ROWS ((int64_t)1 << 23)   // A4 accumulates at most this many rows per partial set
#define RQR_GAUSS_PARTIAL_ROWS 32768     // ksplit * s2 <= this (3 resident CTAs per SM at s2 = 767 ... 842: 37 ... 31 splits)
#define RQR_PANEL_FRAG_BYTES (2 * 10 * 4096 * sizeof(double))   // rqr_tall_panel.cu

#define RQR_PHILOX_STREAM_COUNT 0u
#define RQR_PHILOX_STREAM_S2 1u
#define RQR_PHILOX_STREAM_DENSE 3u
#define RQR_PHILOX_STREAM_RADEMACHER 4u

#define RQR_LAUNCH_CHECK()                                   \
    do {                                                     \
        if (cudaGetLastError() != cudaSuccess) return RQR_ERR_LAUNCH; \
    } while (0)

// Kernel attributes (dynamic shared memory opt-in, non-portable cluster size) are per device: the opt-in runs once
// per DEVICE, keyed by cudaGetDevice, with an atomic flag per device (two threads racing on a first call both set
// the same attribute: idempotent).  A device index outside the table sets the attributes on every call.
#define RQR_MAX_DEVICES 64
struct RqrOncePerDevice {
    std::atomic<unsigned char> done[RQR_MAX_DEVICES];
    int device() const
    {
        int d = -1;
        return (cudaGetDevice(&d) == cudaSuccess && d >= 0 && d < RQR_MAX_DEVICES) ? d : -1;
    }
};
#define RQR_ONCE_PER_DEVICE(...)                                                          \
    do {                                                                                  \
        static RqrOncePerDevice once__;                                                   \
        const int dev__ = once__.device();                                                \
        if (dev__ < 0 || !once__.done[dev__].load(std::memory_order_acquire)) {           \
            __VA_ARGS__                                                                   \
            if (dev__ >= 0) once__.done[dev__].store(1, std::memory_order_release);       \
        }                                                                                 \
    } while (0)

static inline size_t rqr_align256(size_t x) { return (x + 255) & ~(size_t)255; }
// Gram partials the workspace holds: the A4 kernels are launched per chunk of RQR_GRAM_CHUNK_ROWS rows, each
// chunk with its own partial set, so that no register accumulator sums more than ~600 row-blocks before the
// fixed-order tree (rounding error of a long chain on an input whose first rows carry most of the mass).
// 160 MB budget: 1216 partials for n <= 128, 305 at n = 256.
static inline int rqr_gram_partial_cap(int n)
{
    const int64_t by_budget = ((int64_t)160 << 20) / ((int64_t)n * n * 8);
    const int64_t cap = by_budget < 1216 ? by_budget : 1216;
    return (int)(cap < RQR_MAX_GRAM_PARTIALS ? RQR_MAX_GRAM_PARTIALS : cap);
}
// leading dimension of S2 in the workspace: s1 rounded up to 16 doubles, pad columns zero, so that every
// row is 128-byte aligned for the bulk copies of the DMMA GEMM whatever s1 is (paper grid: odd s1)
__host__ __device__ static inline int64_t rqr_s2_ld(int64_t s1) { return (s1 + 15) & ~(int64_t)15; }

// A0 radix sort (rqr_sketch.cu): rows per tile and words of its digit-count scratch ((bins + 1) x tiles + bins)
#define RQR_SORT_MAX_BINS 256
static inline int64_t rqr_sort_tile_rows(int64_t m)
{
    // about eight tiles per SM (two resident CTAs, four rounds), a multiple of 1024 rows, 1024 .. 8192
    int64_t t = ((m + 1183) / 1184 + 1023) / 1024 * 1024;
    return t < 1024 ? 1024 : (t > 8192 ? 8192 : t);
}
static inline size_t rqr_sort_hist_words(int64_t m)
{
    const int64_t T = rqr_sort_tile_rows(m), C = (m + T - 1) / T;
    return (size_t)RQR_SORT_MAX_BINS * (size_t)C + RQR_SORT_MAX_BINS;
}

// ---------------------------------------------------------------------------------------
// Workspace layout.  Offsets of a region depend only on
// arguments every user of that region has.
//   [0,256)            header: counters / flags used inside single calls
//   A  tall scratch    f(n)      Gram partials, small matrices of the one-shot drivers, panel
//                                fragment slots of the n > 64 kernels (2 sets x 10 x 32 KB)
//   B  bucket offsets  f(s1)     (s1+1) u32 offsets, s1 u32 cursors
//   C  S2 slot         f(s1)     sized for s2 = RQR_MAX_S2; empty with RQR_S2_RADEMACHER
//   D  gauss partials  f(n)
//   E  sorted rows     f(m)      m u32 (row | sign<<31)
//   W  one-shot W      (s2max x n), in the n-only part (before B)
//   F  one-shot W1     (s1 x n)
//   G  A0 sort scratch f(m)      m u32 (second row list of the radix sort) + per-tile digit counts
// ---------------------------------------------------------------------------------------
struct RqrLayout {
    size_t hdr, A, A_small, A_frags, B_off, B_cur, C, D, E, F_W1, F_W, G_sort, total;
};

// no_S2: the Rademacher S2 of N4 is generated on the fly, region C is empty
static inline RqrLayout rqr_layout(int64_t m, int n, int64_t s1, bool no_S2 = false)
{
    RqrLayout L;
    size_t nn = (size_t)n * n * sizeof(double);
    L.hdr = 0;
    L.A = 256;
    L.A_small = L.A + rqr_align256((size_t)rqr_gram_partial_cap(n) * nn);
    L.A_frags = L.A_small + rqr_align256(16 * nn);
    // W (s2 x n) of the one-shot drivers sits in the n-only part: rqr_gauss_randcholqr and rqr_cholqr2 do not
    // know s1, and nothing they write may land on the prepared sketch state (regions B, C, E)
    L.F_W = L.A_frags + RQR_PANEL_FRAG_BYTES;
    L.B_off = L.F_W + rqr_align256((size_t)RQR_MAX_S2 * n * sizeof(double));
    L.B_cur = L.B_off + rqr_align256((size_t)(s1 + 1) * 4);
    L.C = L.B_cur + rqr_align256((size_t)s1 * 4);
    L.D = L.C + (no_S2 ? 0 : rqr_align256((size_t)RQR_MAX_S2 * (size_t)rqr_s2_ld(s1) * sizeof(double)));
    L.E = L.D + rqr_align256((size_t)RQR_GAUSS_PARTIAL_ROWS * n * sizeof(double));
    L.F_W1 = L.E + rqr_align256((size_t)m * 4);
    // G: scratch of the A0 radix sort (rqr_sketch_prepare only): the second row list of the ping-pong and the
    // per-tile digit counts
    L.G_sort = L.F_W1 + rqr_align256((size_t)s1 * n * sizeof(double));
    L.total = L.G_sort + rqr_align256((size_t)m * 4) + rqr_align256(rqr_sort_hist_words(m) * 4);
    return L;
}

// small matrices inside A_small (each n*n doubles)
enum { RQR_SM_R0 = 0, RQR_SM_R1 = 1, RQR_SM_G = 2, RQR_SM_RA = 3, RQR_SM_RB = 4, RQR_SM_RC = 5 };

// ---------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11).  Specification: DESIGN.md reading S1.
// key = (seed lo, seed hi); counter = (idx lo, idx hi, stream, 0).
// ---------------------------------------------------------------------------------------
__host__ __device__ __forceinline__ void rqr_philox(uint64_t seed, uint64_t idx, uint32_t stream,
                                                    uint32_t out[4])
{
    uint32_t c0 = (uint32_t)idx, c1 = (uint32_t)(idx >> 32), c2 = stream, c3 = 0u;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        rqr_philox_round(c0, c1, c2, c3, k0, k1);       // rqr_gauss.cuh
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Rademacher S2 (N4; reading S21): the 128 sign bits of row r, columns [128 g, 128 g + 128)
__device__ __forceinline__ void rqr_rademacher_bits(uint64_t seed, uint32_t r, uint64_t ng, uint64_t g, uint32_t out[4])
{
    rqr_philox(seed, (uint64_t)r * ng + g, RQR_PHILOX_STREAM_RADEMACHER, out);
}

// CountSketch bucket and sign of GLOBAL row index i (reading S1/S2).
__device__ __forceinline__ void rqr_hash_sign(uint64_t seed, uint64_t i, uint32_t s1,
                                              uint32_t& bucket, uint32_t& neg)
{
    uint32_t o[4];
    rqr_philox(seed, i, RQR_PHILOX_STREAM_COUNT, o);
    bucket = __umulhi(o[0], s1);     // (uint64(o0) * s1) >> 32
    neg = o[1] & 1u;
}

// Box-Muller pair q of a stream (reading S3): returns z_even, z_odd (standard normal).  Branch-free staged routine
// of rqr_gauss.cuh; `tab` = its logarithm table (the copy in global memory, or a shared-memory copy in hot loops).
__device__ __forceinline__ void rqr_gauss_pair(uint64_t seed, uint64_t q, uint32_t stream,
                                               double& z0, double& z1, const RqrLogEntry* tab = d_rqr_log_tab)
{
    RqrPairDraw d;
    d.begin(seed, q, stream);
    rqr_pair_draw_run<0>(d, tab);
    z0 = d.z0;
    z1 = d.z1;
}

__device__ __forceinline__ double rqr_gauss_entry(uint64_t seed, uint64_t e, uint32_t stream)
{
    double z0, z1;
    rqr_gauss_pair(seed, e >> 1, stream, z0, z1);
    return (e & 1) ? z1 : z0;
}

// first-failure-wins numerical status
__device__ __forceinline__ void rqr_set_info(int* d_info, int code)
{
    if (d_info) atomicCAS(d_info, 0, code);
}
