// rqr_sketch.cu -- A0 sketch generation, A1 CountSketch, A2 Gaussian sketch GEMM, and the
// single dense Gaussian sketch comparator.  See include/rqr.h for the contracts and DESIGN.md
// for the kernel designs.  sm_100a.
#include "rqr_common.cuh"
#include "rqr_tall.cuh"
#include "rqr_mma.cuh"

int rqr_dense_gauss_mma(const double* V, int64_t m, int n, int64_t ldv, int64_t row0, int64_t m_total, int s,
                        uint64_t seed, double* part, int64_t Pcap, int* P_out, bool draw_only, cudaStream_t st);
int rqr_gauss_gemm_mma(const double* S2, const double* W1, int64_t s1, int n, int s2, double* part,
                       int64_t ks_cap, int* ks_out, cudaStream_t st, uint64_t seed);

// =========================================================================================
// A0: sketch generation (off the paper's clock)
// =========================================================================================

// S2[e] = z(e) / sqrt(s2), one Box-Muller pair per thread (entries 2q, 2q+1).
__global__ void k_gen_S2(uint64_t seed, int s2, int64_t s1, int64_t ld, int64_t total, double* __restrict__ S2)
{
    const double d = sqrt((double)s2);
    int64_t npairs = (total + 1) >> 1;
    for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < npairs;
         q += (int64_t)gridDim.x * blockDim.x) {
        double z0, z1;
        rqr_gauss_pair(seed, (uint64_t)q, RQR_PHILOX_STREAM_S2, z0, z1);
        int64_t e = 2 * q;                      // logical entry e = r * s1 + c lives at r * ld + c
        S2[(e / s1) * ld + e % s1] = z0 / d;
        if (e + 1 < total) S2[((e + 1) / s1) * ld + (e + 1) % s1] = z1 / d;
    }
}

// -----------------------------------------------------------------------------------------------------------------
// Bucket-sorted row list = STABLE sort of the rows by bucket, as an LSD radix sort on the bucket id with digits of
// `bits` <= 8 bits.  A pass is three launches -- digit counts per tile of T consecutive positions, an exclusive scan of
// the counts of every digit over the tiles, a stable scatter -- and every step has a fixed order, so the list is the same
// bits run to run (W1 is then bit-reproducible) and equals numpy's stable argsort of the oracle's buckets
// (tests/test_gpu_steps.py::test_sorted_row_list_is_the_stable_sort).  The bucket of an entry is recomputed from its
// row index (Philox) in every pass: the only arrays are the two m-word row lists of the ping-pong.
// Replaces round 1's histogram / cursor fill with global atomics + a bitonic sort per bucket (0.88 ms at 2^23 rows).
// -----------------------------------------------------------------------------------------------------------------
#define SORT_THREADS 512
#define SORT_WARPS (SORT_THREADS / 32)

// entry (row | sign << 31) at position pos of the pass input (in == NULL: the identity list) and its digit
__device__ __forceinline__ void sort_load(const uint32_t* __restrict__ in, int64_t pos, uint64_t seed, int64_t row0,
                                          uint32_t s1, int shift, uint32_t mask, uint32_t& entry, uint32_t& digit)
{
    uint32_t row = in ? (in[pos] & 0x7fffffffu) : (uint32_t)pos;
    uint32_t b, neg;
    rqr_hash_sign(seed, (uint64_t)(row0 + row), s1, b, neg);
    entry = in ? in[pos] : (row | (neg << 31));
    digit = (b >> shift) & mask;
}

// counts[d * C + tile] = number of positions of the tile whose digit is d
__global__ void __launch_bounds__(SORT_THREADS)
k_sort_count(uint64_t seed, int64_t row0, int64_t m, uint32_t s1, const uint32_t* __restrict__ in, int shift, int bits,
             int T, int C, uint32_t* __restrict__ counts)
{
    __shared__ uint32_t h[RQR_SORT_MAX_BINS];
    const int bins = 1 << bits;
    for (int d = threadIdx.x; d < bins; d += SORT_THREADS) h[d] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * T;
    for (int i = threadIdx.x; i < T && base + i < m; i += SORT_THREADS) {
        uint32_t e, d;
        sort_load(in, base + i, seed, row0, s1, shift, (uint32_t)bins - 1, e, d);
        atomicAdd(&h[d], 1u);
    }
    __syncthreads();
    for (int d = threadIdx.x; d < bins; d += SORT_THREADS) counts[(size_t)d * C + blockIdx.x] = h[d];
}

// one CTA per digit: exclusive scan of counts[d][0..C) in place, total[d] = the digit's count
__global__ void __launch_bounds__(1024)
k_sort_scan_tiles(uint32_t* __restrict__ counts, int C, uint32_t* __restrict__ total)
{
    __shared__ uint32_t warp_tot[32];
    __shared__ uint32_t carry;
    uint32_t* c = counts + (size_t)blockIdx.x * C;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < C; base += 1024) {
        const int idx = base + tid;
        const uint32_t v = idx < C ? c[idx] : 0u;
        uint32_t x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_tot[wid] = x;
        __syncthreads();
        if (wid == 0) {
            uint32_t t = warp_tot[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t y = __shfl_up_sync(0xffffffffu, t, o);
                if (lane >= o) t += y;
            }
            warp_tot[lane] = t;
        }
        __syncthreads();
        if (idx < C) c[idx] = carry + (wid ? warp_tot[wid - 1] : 0u) + x - v;
        __syncthreads();
        if (tid == 0) carry += warp_tot[31];
        __syncthreads();
    }
    if (tid == 0) total[blockIdx.x] = carry;
}

// stable scatter of one tile: out[digit_base[d] + tile_off[d][tile] + rank within the tile] = entry.
// Thread t owns the K = T / 256 consecutive positions [t K, (t + 1) K) of the tile and a private column cnt[d][t] of
// 16-bit counters: it counts its digits, the counters of every digit are scanned over the threads (thread order =
// position order), and a second walk over the same positions hands out the ranks in order.  No atomics and no vote /
// match instructions (a match.any version spent 85% of its time in MATCH: ~28 distinct digits per warp).
#define SCATTER_THREADS 256
__global__ void __launch_bounds__(SCATTER_THREADS)
k_sort_scatter(uint64_t seed, int64_t row0, int64_t m, uint32_t s1, const uint32_t* __restrict__ in,
               uint32_t* __restrict__ out, int shift, int bits, int T, int C, const uint32_t* __restrict__ tile_off,
               const uint32_t* __restrict__ total)
{
    extern __shared__ uint32_t sm_sort[];
    constexpr int NT = SCATTER_THREADS;
    const int bins = 1 << bits, K = T / NT, KP = K + 2;             // K % 4 == 0: KP / 2 odd, conflict-free walks
    uint32_t* ent = sm_sort;                                        // NT x (K + 1): odd row stride, conflict-free
    uint32_t* dbase = ent + NT * (K + 1);                           // bins (<= 256)
    uint16_t* dig = reinterpret_cast<uint16_t*>(dbase + bins);      // NT x KP
    uint16_t* cnt = dig + (size_t)NT * KP;                          // bins x NT
    __shared__ uint32_t warp_tot[NT / 32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int64_t base = (int64_t)blockIdx.x * T;
    for (int i = tid; i < T; i += NT) {                             // coalesced: position i -> owner i / K, slot i % K
        uint32_t e = 0, d = 0xFFFFu;
        if (base + i < m) sort_load(in, base + i, seed, row0, s1, shift, (uint32_t)bins - 1, e, d);
        ent[(i / K) * (K + 1) + (i % K)] = e;
        dig[(i / K) * KP + (i % K)] = (uint16_t)d;
    }
    for (int i = tid; i < bins * NT / 2; i += NT) reinterpret_cast<uint32_t*>(cnt)[i] = 0u;
    {   // dbase = exclusive scan of total[0..bins), bins <= 256 = one element per thread
        const uint32_t v = tid < bins ? total[tid] : 0u;
        uint32_t x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_tot[wid] = x;
        __syncthreads();
        uint32_t before = 0;
        for (int w = 0; w < wid; ++w) before += warp_tot[w];
        // first output position of this tile's run of digit d: the digit's base + the earlier tiles' counts
        if (tid < bins) dbase[tid] = before + x - v + tile_off[(size_t)tid * C + blockIdx.x];
    }
    __syncthreads();
    const uint16_t* mydig = dig + (size_t)tid * KP;
    for (int j = 0; j < K; ++j) {
        const uint32_t d = mydig[j];
        if (d != 0xFFFFu) cnt[d * NT + tid] += 1;
    }
    __syncthreads();
    for (int d = wid; d < bins; d += NT / 32) {                     // per digit: exclusive scan over the 256 threads
        uint16_t* row = cnt + (size_t)d * NT;
        uint32_t v[8], sum = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) { v[q] = row[lane * 8 + q]; sum += v[q]; }
        uint32_t x = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        uint32_t run = x - sum;
#pragma unroll
        for (int q = 0; q < 8; ++q) { row[lane * 8 + q] = (uint16_t)run; run += v[q]; }
    }
    __syncthreads();
    for (int j = 0; j < K; ++j) {
        const uint32_t d = mydig[j];
        if (d == 0xFFFFu) continue;
        const uint32_t rank = cnt[d * NT + tid];
        cnt[d * NT + tid] = (uint16_t)(rank + 1);
        out[dbase[d] + rank] = ent[tid * (K + 1) + j];
    }
}

// off[b] = first position of the sorted list whose bucket is >= b (b = 0 .. s1): bucket boundaries of the list.
// One thread per boundary, a binary search over the sorted list (the bucket of a probed entry is recomputed from its
// row index): s1 + 1 searches of log2(m) dependent probes instead of a pass over all m entries with a Philox call
// each (C3: 65 -> ~20 us).
__global__ void __launch_bounds__(256)
k_bucket_bounds(uint64_t seed, int64_t row0, int64_t m, uint32_t s1, const uint32_t* __restrict__ entries,
                uint32_t* __restrict__ off)
{
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b > (int64_t)s1) return;
    int64_t lo = 0, hi = m;                       // first position in [0, m] whose bucket is >= b
    if (b == 0) hi = 0;
    if (b == (int64_t)s1) lo = m;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        uint32_t bk, neg;
        rqr_hash_sign(seed, (uint64_t)(row0 + (__ldg(entries + mid) & 0x7fffffffu)), s1, bk, neg);
        if ((int64_t)bk >= b) hi = mid; else lo = mid + 1;
    }
    off[b] = (uint32_t)lo;
}

static int launch_prepare_S2(int64_t s1, int s2, uint64_t seed, double* S2, cudaStream_t st)
{
    int64_t total = (int64_t)s2 * s1;
    int64_t npairs = (total + 1) / 2;
    int blocks = (int)((npairs + 255) / 256 < 148 * 16 ? (npairs + 255) / 256 : 148 * 16);
    if (blocks < 1) blocks = 1;
    const int64_t ld = rqr_s2_ld(s1);
    if (ld != s1 && cudaMemsetAsync(S2, 0, (size_t)s2 * ld * sizeof(double), st) != cudaSuccess) return RQR_ERR_LAUNCH;
    k_gen_S2<<<blocks, 256, 0, st>>>(seed, s2, s1, ld, total, S2);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// `scratch`: m words (second row list) followed by the digit-count words (rqr_sort_hist_words)
static int launch_prepare_sorted(int64_t m, int64_t row0, int64_t s1, uint64_t seed, uint32_t* off,
                                 uint32_t* entries, uint32_t* scratch, cudaStream_t st)
{
    int key_bits = 0;
    while (((int64_t)1 << key_bits) < s1) ++key_bits;
    const int passes = key_bits <= 8 ? 1 : (key_bits + 7) / 8;     // digits of at most 8 bits (k_sort_scatter's table)
    int bits = (key_bits + passes - 1) / passes;
    if (bits < 1) bits = 1;
    const int bins = 1 << bits;
    const int T = (int)rqr_sort_tile_rows(m);
    const int C = (int)((m + T - 1) / T);
    uint32_t* other = scratch;
    uint32_t* counts = scratch + (((size_t)m + 63) & ~(size_t)63);
    uint32_t* total = counts + (size_t)RQR_SORT_MAX_BINS * C;
    const int K = T / SCATTER_THREADS;
    const size_t smem = (size_t)SCATTER_THREADS * (K + 1) * 4 + (size_t)bins * 4 + (size_t)SCATTER_THREADS * (K + 2) * 2 + (size_t)bins * SCATTER_THREADS * 2;
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_sort_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    });
    // the last pass must land in `entries`: an odd number of passes starts by writing `entries`
    const uint32_t* in = nullptr;
    uint32_t* out = (passes & 1) ? entries : other;
    for (int p = 0; p < passes; ++p) {
        const int shift = p * bits;
        k_sort_count<<<C, SORT_THREADS, 0, st>>>(seed, row0, m, (uint32_t)s1, in, shift, bits, T, C, counts);
        RQR_LAUNCH_CHECK();
        k_sort_scan_tiles<<<bins, 1024, 0, st>>>(counts, C, total);
        RQR_LAUNCH_CHECK();
        k_sort_scatter<<<C, SCATTER_THREADS, smem, st>>>(seed, row0, m, (uint32_t)s1, in, out, shift, bits, T, C, counts, total);
        RQR_LAUNCH_CHECK();
        in = out;
        out = (out == entries) ? other : entries;
    }
    k_bucket_bounds<<<(int)((s1 + 1 + 255) / 256), 256, 0, st>>>(seed, row0, m, (uint32_t)s1, entries, off);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

extern "C" int rqr_sketch_prepare(int64_t m, int n, int64_t row0, int64_t s1, int s2,
                                  uint64_t seed, int variant, void* work, void* stream)
{
    if (m < 1 || m >= ((int64_t)1 << 31)) return -1;
    if (n < 2 || n > RQR_MAX_N) return -2;
    if (row0 < 0) return -3;
    if (s1 < 1 || s1 >= ((int64_t)1 << 31)) return -4;
    if (s2 < 1 || s2 > RQR_MAX_S2 || s2 > s1) return -5;
    const bool rademacher = (variant & RQR_S2_RADEMACHER) != 0;
    variant &= ~RQR_S2_RADEMACHER;
    if (variant != RQR_VARIANT_SORTED && variant != RQR_VARIANT_SCATTER && variant != RQR_VARIANT_STREAM) return -7;
    if (!work) return -8;
    cudaStream_t st = (cudaStream_t)stream;
    RqrLayout L = rqr_layout(m, n, s1, rademacher);
    char* w = (char*)work;
    int rc = rademacher ? RQR_OK : launch_prepare_S2(s1, s2, seed, (double*)(w + L.C), st);
    if (rc != RQR_OK) return rc;
    if (variant == RQR_VARIANT_SORTED)
        rc = launch_prepare_sorted(m, row0, s1, seed, (uint32_t*)(w + L.B_off), (uint32_t*)(w + L.E),
                                   (uint32_t*)(w + L.G_sort), st);
    return rc;
}

// =========================================================================================
// A1: CountSketch  W1[h(i),:] += sigma(i) V[i,:]   (PAPER.md:236, :240; S1 unscaled, :341)
// =========================================================================================

// SORTED / gather variant.  One CTA per bucket (grid-stride).  The CTA's threads form
// R row-slots x LPR lanes-per-row; lane c of slot r owns VEC consecutive columns and sums the
// bucket's rows r, r+R, r+2R, ... (4 loads in flight per thread), then the R slot sums are
// added in slot order through shared memory.  Fixed mapping => bit-reproducible W1.
// HBM-bound: every row of V is read exactly once, 8n contiguous bytes.
#ifndef RQR_GATHER_PREFETCH_MAX_N
#define RQR_GATHER_PREFETCH_MAX_N 40
#endif
template <int VEC, bool PREFETCH>
__global__ void __launch_bounds__(256, 8)
k_countsketch_gather(const double* __restrict__ V, int64_t ldv, int n,
                     const uint32_t* __restrict__ off, const uint32_t* __restrict__ entries,
                     uint32_t s1, double* __restrict__ W1, uint32_t split)
{
    // split > 1 (fewer buckets than resident CTAs): work item w = bucket b, segment j of its row list; the
    // segment sums go to W1[j][b][:] (a scratch of split partial sketches) and are added in order j = 0, 1, ...
    // by k_reduce_partials.
    extern __shared__ double red[];                 // R * n doubles
    const int lpr = (n + VEC - 1) / VEC;            // lanes per row
    const int R = max(1, 256 / lpr);
    const int slot = threadIdx.x / lpr;
    const int col = (threadIdx.x % lpr) * VEC;
    const bool active = slot < R && col < n;
    for (uint32_t w = blockIdx.x; w < s1 * split; w += gridDim.x) {
        const uint32_t b = w / split, j = w - b * split;
        const uint32_t beg0 = off[b], len = off[b + 1] - beg0;
        const uint32_t beg = beg0 + (uint32_t)((uint64_t)len * j / split);
        const uint32_t end = beg0 + (uint32_t)((uint64_t)len * (j + 1) / split);
        double a0 = 0.0, a1 = 0.0;
        if (active) {
            uint32_t k = beg + slot;
            // 4 rows in flight; PREFETCH: the row-list entries of the NEXT four are loaded while these are in flight
            uint32_t e[4] = {0u, 0u, 0u, 0u}, en[4] = {0u, 0u, 0u, 0u};
            if (PREFETCH && k + 3u * R < end) {
#pragma unroll
                for (int u = 0; u < 4; ++u) e[u] = entries[k + u * R];
            }
            for (; k + 3u * R < end; k += 4u * R) {
                double x[4][2];
                if (!PREFETCH) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) e[u] = entries[k + u * R];
                }
                const bool more = PREFETCH && k + 7u * R < end;
                if (more) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) en[u] = entries[k + (4 + u) * R];
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const double* p = V + (int64_t)(e[u] & 0x7fffffffu) * ldv + col;
                    if (VEC == 2) {
                        double2 t = __ldg(reinterpret_cast<const double2*>(p));
                        x[u][0] = t.x; x[u][1] = t.y;
                    } else {
                        x[u][0] = __ldg(p); x[u][1] = 0.0;
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (e[u] >> 31) { a0 -= x[u][0]; a1 -= x[u][1]; }
                    else            { a0 += x[u][0]; a1 += x[u][1]; }
                }
                if (PREFETCH) {
#pragma unroll
                    for (int u = 0; u < 4; ++u) e[u] = en[u];
                }
            }
            for (; k < end; k += R) {
                uint32_t e = entries[k];
                const double* p = V + (int64_t)(e & 0x7fffffffu) * ldv + col;
                double x0, x1 = 0.0;
                if (VEC == 2) { double2 t = __ldg(reinterpret_cast<const double2*>(p)); x0 = t.x; x1 = t.y; }
                else x0 = __ldg(p);
                if (e >> 31) { a0 -= x0; a1 -= x1; } else { a0 += x0; a1 += x1; }
            }
            red[slot * n + col] = a0;
            if (VEC == 2) red[slot * n + col + 1] = a1;
        }
        __syncthreads();
        for (int c = threadIdx.x; c < n; c += blockDim.x) {
            double s = red[c];
            for (int r = 1; r < R; ++r) s += red[r * n + c];
            W1[((int64_t)j * s1 + b) * n + c] = s;
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256) k_reduce_partials(const double* __restrict__ part, int nparts, int64_t elems, double* __restrict__ out);

// SCATTER variant: stream V in row order, hash on the fly, red.global.add.f64 into W1 (which
// lives in L2).  Order of the atomics is not fixed => last bits vary run to run.
__global__ void __launch_bounds__(256)
k_countsketch_scatter(const double* __restrict__ V, int64_t m, int64_t ldv, int n, int64_t row0,
                      uint64_t seed, uint32_t s1, double* __restrict__ W1)
{
    const int lpr = n < 32 ? n : 32;                // lanes cooperating on one row
    const int rows_per_warp = 32 / lpr;
    const int lane = threadIdx.x & 31;
    const int sub = lane / lpr, c0 = lane % lpr;
    const int64_t warp_global = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t i = warp_global * rows_per_warp + sub; i < m; i += nwarps * rows_per_warp) {
        if (sub >= rows_per_warp) continue;
        uint32_t b, neg;
        rqr_hash_sign(seed, (uint64_t)(row0 + i), s1, b, neg);
        const double* src = V + i * ldv;
        double* dst = W1 + (int64_t)b * n;
        for (int c = c0; c < n; c += lpr) {
            double x = __ldg(src + c);
            atomicAdd(dst + c, neg ? -x : x);
        }
    }
}

// STREAM variant: no stored S1.  Every warp is its own pipeline over 8-row blocks of V (rows in order: a sequential
// HBM stream): bulk async copy into a private ring, bucket and sign of the 8 rows from Philox (lanes 0..7), sign flip in
// shared memory, then ONE bulk reduction per row, cp.reduce.async.bulk.global.shared::cta.add.f64 (SASS UBLKRED):
// the L2 adds 8n contiguous bytes to row h(i) of W1 -- n/4 32-byte sectors per request instead of n element-wise
// atomics issued by the LSU.  W1 must be zero on entry.
#define CS_MAX_STAGES 8
#define CS_MAX_WARPS 16
template <bool CONTIG>
__global__ void __launch_bounds__(CS_MAX_WARPS * 32, 1)
k_countsketch_stream(const double* __restrict__ V, int64_t m, int64_t ldv, int n, int64_t row0, uint64_t seed,
                     uint32_t s1, double* __restrict__ W1, int warps, int stages)
{
    extern __shared__ __align__(16) double smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);                         // warps x stages
    double* ring = smem + ((warps * stages + 1) & ~1);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (warp >= warps) return;
    if (lane < stages) mbar_init(bars + warp * stages + lane, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncwarp();
    uint64_t* bar = bars + warp * stages;
    double* buf = ring + (size_t)warp * stages * 8 * n;
    const int64_t nrb = (m + 7) / 8;
    const int64_t gw = (int64_t)blockIdx.x * warps + warp;
    const int64_t stride = (int64_t)gridDim.x * warps;
    auto issue = [&](int stage, int64_t rblk) {
        const int valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
        if (lane == 0) mbar_expect_tx(bar + stage, (uint32_t)(valid * n * 8));
        __syncwarp();
        if (CONTIG) {
            if (lane == 0) bulk_g2s(buf + (size_t)stage * 8 * n, V + rblk * 8 * ldv, (uint32_t)(valid * n * 8), bar + stage);
        } else if (lane < valid) {
            bulk_g2s(buf + ((size_t)stage * 8 + lane) * n, V + (rblk * 8 + lane) * ldv, (uint32_t)(n * 8), bar + stage);
        }
    };
    // stages of the ring at iteration i: block i (in use), block i - 1 (its reductions may still read it) and the
    // blocks i + 1 .. i + stages - 2 in flight
    for (int s = 0; s < stages - 2; ++s)
        if (gw + s * stride < nrb) issue(s, gw + s * stride);
    int stage = 0, it = 0;
    uint32_t phase = 0;
    for (int64_t rblk = gw; rblk < nrb; rblk += stride, ++it) {
        // refill the stage consumed two iterations ago: its bulk reductions have READ shared memory once every lane
        // has at most its newest group pending; row-block i + stages - 2 goes into it
        asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
        __syncwarp();
        {
            const int64_t next = rblk + (int64_t)(stages - 2) * stride;
            const int ps = stage >= 2 ? stage - 2 : stage + stages - 2;
            if (next < nrb) issue(ps, next);
        }
        const int valid = (int)((m - rblk * 8) < 8 ? (m - rblk * 8) : 8);
        uint32_t b = 0, neg = 0;
        if (lane < valid) rqr_hash_sign(seed, (uint64_t)(row0 + rblk * 8 + lane), s1, b, neg);
        const uint32_t negmask = __ballot_sync(0xffffffffu, neg != 0);
        mbar_wait(bar + stage, phase);
        double* rb = buf + (size_t)stage * 8 * n;
        for (uint32_t msk = negmask; msk; msk &= msk - 1) {                   // rows with sigma = -1
            double* row = rb + (size_t)(__ffs(msk) - 1) * n;
            for (int c = 2 * lane; c < n; c += 64) {
                double2 v = *reinterpret_cast<double2*>(row + c);
                *reinterpret_cast<double2*>(row + c) = make_double2(-v.x, -v.y);
            }
        }
        fence_proxy_async();
        __syncwarp();
        if (lane < valid) {
            asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], %2;"
                         :: "l"(W1 + (size_t)b * n), "r"(smem_u32(rb + (size_t)lane * n)), "r"((uint32_t)(n * 8)) : "memory");
        }
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        if (++stage == stages) { stage = 0; phase ^= 1u; }
    }
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

static int launch_countsketch_stream(const double* V, int64_t m, int n, int64_t ldv, int64_t row0, int64_t s1,
                                     uint64_t seed, double* W1, cudaStream_t st)
{
    if ((n & 1) || (ldv & 1) || (((uintptr_t)V | (uintptr_t)W1) & 15)) return RQR_TALL_NOT_HANDLED;
    // The per-warp loop is latency-bound (copy in, hash, flip, reduce out): what counts is row-blocks in flight per SM.
    // Ring = warps x stages x 8 rows x n doubles within 192 KB, as many warps as leave >= 5 stages (3 in flight):
    // n <= 38: 16 warps, n <= 76: 8 (n = 64: 8 x 6), n <= 153: 4, above: 4 x 3.
    int warps = CS_MAX_WARPS;
    while (warps > 4 && (size_t)warps * 5 * 64 * n > 192 * 1024) warps >>= 1;
    int stages = (int)((192 * 1024) / ((size_t)warps * 64 * n));
    if (stages > CS_MAX_STAGES) stages = CS_MAX_STAGES;
    if (stages < 3) stages = 3;
    while (warps > 1 && (size_t)warps * stages * 64 * n > 200 * 1024) warps >>= 1;
    const size_t smem = (size_t)(((warps * stages + 1) & ~1) + (size_t)warps * stages * 8 * n) * sizeof(double);
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_countsketch_stream<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        cudaFuncSetAttribute(k_countsketch_stream<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    });
    const int64_t nrb = (m + 7) / 8;
    int64_t g = (nrb + warps - 1) / warps;
    const int grid = (int)(g < 148 ? (g < 1 ? 1 : g) : 148);
    if (ldv == n) k_countsketch_stream<true><<<grid, CS_MAX_WARPS * 32, smem, st>>>(V, m, ldv, n, row0, seed, (uint32_t)s1, W1, warps, stages);
    else          k_countsketch_stream<false><<<grid, CS_MAX_WARPS * 32, smem, st>>>(V, m, ldv, n, row0, seed, (uint32_t)s1, W1, warps, stages);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// TILE form of the stream variant, for a sketch that fits SHARED MEMORY (s1 n doubles <= 224 KB) with n <= 20.
// Every CTA streams its rows in order with plain coalesced loads (lane = two columns of one row, 32 / LPR rows per
// warp step, the next 32 rows already in flight), draws bucket and sign of 32 rows at a time from Philox (lane = row,
// the codes travel by shuffle) and adds every row to its bucket row of the tile with shared-memory atomics
// (ATOMS.CAST.SPIN); the tile is flushed ONCE per CTA by bulk reductions (UBLKRED).  north_star: "scatter-adds rows
// through shared-memory bucket tiles".  W1 must be zero on entry.
// Measured: 3.5-3.8 TB/s at n = 16 / 20 and 2.8 at n = 10 against 1.7 / 2.1 / 1.0 of the per-row bulk
// reductions; the shared-memory CAS loop binds it (the same kernel with a plain, racy += runs at 5.0 / 4.2 TB/s), and
// column slices for wider sketches (n = 32: 4 slices of 8 columns) ran at 2.1-2.7 TB/s even without atomics: not built.
#define CST_THREADS 512
#define CST_MAX_TILE_BYTES (224 * 1024)
#define CST_MAX_LPR 10
template <int LPR>
__global__ void __launch_bounds__(CST_THREADS, 1)
k_countsketch_tile(const double* __restrict__ V, int64_t m, int64_t ldv, int n, int64_t row0, uint64_t seed,
                   uint32_t s1, double* __restrict__ W1, int bulk_flush)
{
    extern __shared__ __align__(16) double tile[];                 // s1 x n
    constexpr int RPS = 32 / LPR;                                  // rows per warp step
    constexpr int NSTEP = (32 + RPS - 1) / RPS;
    constexpr int NW = CST_THREADS / 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tile_elems = (int)s1 * n;
    for (int e = threadIdx.x; e < tile_elems; e += CST_THREADS) tile[e] = 0.0;
    __syncthreads();
    const int g = lane / LPR, j = lane - g * LPR;                  // row of the step, lane inside the row
    const bool has0 = g < RPS && j < n, has1 = g < RPS && (j + LPR) < n;
    const int64_t ngroups = (m + 31) / 32, gstride = (int64_t)gridDim.x * NW;
    double x0[NSTEP], x1[NSTEP], y0[NSTEP], y1[NSTEP];             // this group's rows / the next group's, in flight
    auto load = [&](int64_t grp, double (&a0)[NSTEP], double (&a1)[NSTEP]) {
        const int64_t i0 = grp * 32;
#pragma unroll
        for (int s = 0; s < NSTEP; ++s) {
            const int r = s * RPS + g;
            const bool ok = grp < ngroups && r < 32 && (i0 + r) < m;
            const double* src = V + (i0 + r) * ldv + j;
            a0[s] = (ok && has0) ? __ldcs(src) : 0.0;
            a1[s] = (ok && has1) ? __ldcs(src + LPR) : 0.0;
        }
    };
    int64_t grp = (int64_t)blockIdx.x * NW + warp;
    load(grp, x0, x1);
    for (; grp < ngroups; grp += gstride) {
        const int64_t i0 = grp * 32;
        load(grp + gstride, y0, y1);
        uint32_t b = 0, neg = 0;
        if (i0 + lane < m) rqr_hash_sign(seed, (uint64_t)(row0 + i0 + lane), s1, b, neg);
        const uint32_t code = b | (neg << 31);
#pragma unroll
        for (int s = 0; s < NSTEP; ++s) {
            const int r = s * RPS + g;
            const uint32_t cr = __shfl_sync(0xffffffffu, code, r & 31);
            const bool ok = r < 32 && (i0 + r) < m;
            double* p = tile + (size_t)(cr & 0x7fffffffu) * n + j;
            const bool ng = (cr >> 31) != 0;
            if (ok && has0) atomicAdd(p, ng ? -x0[s] : x0[s]);
            if (ok && has1) atomicAdd(p + LPR, ng ? -x1[s] : x1[s]);
        }
#pragma unroll
        for (int s = 0; s < NSTEP; ++s) { x0[s] = y0[s]; x1[s] = y1[s]; }
    }
    __syncthreads();
    if (bulk_flush) {                                              // the tile IS the sketch: 4 KB pieces
        fence_proxy_async();
        __syncthreads();
        const uint32_t total = (uint32_t)tile_elems * 8u, piece = 4096u;
        for (uint32_t off = threadIdx.x * piece; off < total; off += CST_THREADS * piece) {
            const uint32_t bytes = (total - off) < piece ? (total - off) : piece;
            asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], %2;"
                         :: "l"((char*)W1 + off), "r"(smem_u32(tile) + off), "r"(bytes) : "memory");
        }
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    } else {                                                       // odd s1 n or unaligned W1: element-wise red
        for (int e = threadIdx.x; e < tile_elems; e += CST_THREADS) {
            const double v = tile[e];
            if (v != 0.0) atomicAdd(W1 + e, v);
        }
    }
}

template <int LPR>
static int launch_countsketch_tile_lpr(const double* V, int64_t m, int n, int64_t ldv, int64_t row0, int64_t s1,
                                       uint64_t seed, double* W1, cudaStream_t st)
{
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_countsketch_tile<LPR>, cudaFuncAttributeMaxDynamicSharedMemorySize, CST_MAX_TILE_BYTES);
    });
    const size_t smem = (size_t)s1 * n * sizeof(double);
    const int64_t ngroups = (m + 31) / 32, want = (ngroups + CST_THREADS / 32 - 1) / (CST_THREADS / 32);
    const int grid = (int)(want < 148 ? (want < 1 ? 1 : want) : 148);
    const int bulk = (((s1 * n) % 2 == 0) && (((uintptr_t)W1 & 15) == 0)) ? 1 : 0;
    k_countsketch_tile<LPR><<<grid, CST_THREADS, smem, st>>>(V, m, ldv, n, row0, seed, (uint32_t)s1, W1, bulk);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

static int launch_countsketch_tile(const double* V, int64_t m, int n, int64_t ldv, int64_t row0, int64_t s1,
                                   uint64_t seed, double* W1, cudaStream_t st)
{
    const int lpr = (n + 1) / 2;
    if (lpr > CST_MAX_LPR || (size_t)s1 * n * sizeof(double) > CST_MAX_TILE_BYTES) return RQR_TALL_NOT_HANDLED;
#define RQR_CST_CASE(L) case L: return launch_countsketch_tile_lpr<L>(V, m, n, ldv, row0, s1, seed, W1, st);
    switch (lpr) {
        RQR_CST_CASE(1) RQR_CST_CASE(2) RQR_CST_CASE(3) RQR_CST_CASE(4) RQR_CST_CASE(5) RQR_CST_CASE(6) RQR_CST_CASE(7)
        RQR_CST_CASE(8) RQR_CST_CASE(9) RQR_CST_CASE(10)
    default: break;
    }
#undef RQR_CST_CASE
    return RQR_TALL_NOT_HANDLED;
}

extern "C" int rqr_countsketch(const double* V, int64_t m, int n, int64_t ldv, int64_t row0,
                               int64_t s1, uint64_t seed, double* W1, void* work, int variant,
                               int flags, void* stream)
{
    if (!V) return -1;
    if (m < 1 || m >= ((int64_t)1 << 31)) return -2;
    if (n < 2 || n > RQR_MAX_N) return -3;
    if (ldv < n) return -4;
    if (row0 < 0) return -5;
    if (s1 < 1 || s1 >= ((int64_t)1 << 31)) return -6;
    if (!W1) return -8;
    const bool rademacher = (variant & RQR_S2_RADEMACHER) != 0;      // only moves region E of the workspace
    variant &= ~RQR_S2_RADEMACHER;
    if (variant != RQR_VARIANT_SORTED && variant != RQR_VARIANT_SCATTER && variant != RQR_VARIANT_STREAM) return -10;
    cudaStream_t st = (cudaStream_t)stream;
    if (variant == RQR_VARIANT_STREAM) {
        if (cudaMemsetAsync(W1, 0, (size_t)s1 * n * sizeof(double), st) != cudaSuccess)
            return RQR_ERR_LAUNCH;
        int rc = launch_countsketch_tile(V, m, n, ldv, row0, s1, seed, W1, st);      // the sketch fits shared memory
        if (rc != RQR_TALL_NOT_HANDLED) return rc;
        rc = launch_countsketch_stream(V, m, n, ldv, row0, s1, seed, W1, st);
        if (rc != RQR_TALL_NOT_HANDLED) return rc;
        variant = RQR_VARIANT_SCATTER;              // odd n / ld or unaligned bases: per-element atomics (W1 is zeroed)
    }
    if (variant == RQR_VARIANT_SCATTER) {
        if (cudaMemsetAsync(W1, 0, (size_t)s1 * n * sizeof(double), st) != cudaSuccess)
            return RQR_ERR_LAUNCH;
        int64_t want = (m + 7) / 8;
        int blocks = (int)(want < 148 * 8 ? want : 148 * 8);
        if (blocks < 1) blocks = 1;
        k_countsketch_scatter<<<blocks, 256, 0, st>>>(V, m, ldv, n, row0, seed, (uint32_t)s1, W1);
        RQR_LAUNCH_CHECK();
        return RQR_OK;
    }
    if (!work) return -9;
    RqrLayout L = rqr_layout(m, n, s1, rademacher);
    char* w = (char*)work;
    uint32_t* off = (uint32_t*)(w + L.B_off);
    uint32_t* ent = (uint32_t*)(w + L.E);
    if (!(flags & RQR_FLAG_PREPARED)) {
        int rc = launch_prepare_sorted(m, row0, s1, seed, off, ent, (uint32_t*)(w + L.G_sort), st);
        if (rc != RQR_OK) return rc;
    }
    const bool vec2 = (n % 2 == 0) && (ldv % 2 == 0) && (((uintptr_t)V & 15) == 0);
    const int lpr = vec2 ? n / 2 : n;
    const int R = 256 / lpr > 1 ? 256 / lpr : 1;
    size_t smem = (size_t)R * n * sizeof(double);
    // One CTA walks one bucket at a time and 148 x 8 CTAs are resident: with fewer buckets than half of that the grid
    // is underfilled (s1 = 200: 17% of the CTA slots).  Every bucket's row list is then split into `split` segments,
    // the smallest count that fills the last round of CTAs to >= 95%; the segment sums go to `split` partial sketches
    // in region A of the workspace (free during A1) and are added in a fixed order.  With s1 >= 592 the pass is bound
    // by DRAM, not by CTA slots (measured at s1 = 2048: 5.36 TB/s with or without a split), and is left alone.
    int64_t split = 1;
    if (s1 * 2 <= 148 * 8) {
        const double slots = 148.0 * 8.0;
        const int64_t fit = (int64_t)rqr_gram_partial_cap(n) * n / s1;          // region A holds cap n^2 doubles
        const int64_t rows = m / (s1 * 4 * R);                                  // >= 4 R rows per segment
        int64_t best = 1;
        double best_eff = 0.0;
        for (int64_t sp = 1; sp <= 64 && sp <= fit && (sp == 1 || sp <= rows); ++sp) {
            const double waves = (double)(s1 * sp) / slots;
            const double eff = waves / ceil(waves);
            if (eff > best_eff + 1e-9) { best_eff = eff; best = sp; }
            if (eff >= 0.95) break;
        }
        split = best;
    }
    double* dst = split > 1 ? (double*)(w + L.A) : W1;
    const int64_t items = s1 * split;
    int blocks = (int)(items < 148 * 8 ? items : 148 * 8);
    // PREFETCH: the next four row-list entries are loaded while four rows are in flight (the entry load and the row load
    // it feeds are two dependent memory latencies).  Measured A/B in one process, both forms at 8 resident CTAs per SM
    // (__launch_bounds__(256, 8): 32 registers either way): it pays for even n <= 40 without a bucket split (2^22 x 32
    // 193 -> 184 us, 2^25 x 32 1457 -> 1361, 10^7 x 20 309 -> 292) and loses for odd n (scalar loads: 173 -> 238 us
    // at n = 33), with split buckets and from n = 48 up.
    const bool pf = vec2 && n <= RQR_GATHER_PREFETCH_MAX_N && split == 1;
    if (vec2 && pf)  k_countsketch_gather<2, true><<<blocks, 256, smem, st>>>(V, ldv, n, off, ent, (uint32_t)s1, dst, (uint32_t)split);
    else if (vec2)   k_countsketch_gather<2, false><<<blocks, 256, smem, st>>>(V, ldv, n, off, ent, (uint32_t)s1, dst, (uint32_t)split);
    else             k_countsketch_gather<1, false><<<blocks, 256, smem, st>>>(V, ldv, n, off, ent, (uint32_t)s1, dst, (uint32_t)split);
    RQR_LAUNCH_CHECK();
    if (split > 1) {
        const int64_t elems = s1 * n;
        k_reduce_partials<<<(int)((elems + 63) / 64), 256, 0, st>>>(dst, (int)split, elems, W1);
        RQR_LAUNCH_CHECK();
    }
    return RQR_OK;
}

// =========================================================================================
// A2: Gaussian sketch  W = S2 W1, split-K GEMM + fixed-order reduction
// =========================================================================================
#define GS_BM 64
#define GS_BN 64
#define GS_BK 16

// partial[ks] (s2 x n) = S2[:, k0:k1] * W1[k0:k1, :].  64x64 tile per CTA, 4x4 per thread.
__global__ void __launch_bounds__(256)
k_gauss_gemm_splitk(const double* __restrict__ S2, const double* __restrict__ W1, int64_t s1,
                    int n, int s2, int64_t kchunk, double* __restrict__ part)
{
    const int64_t lds2 = rqr_s2_ld(s1);
    __shared__ double As[GS_BK][GS_BM + 1];
    __shared__ double Bs[GS_BK][GS_BN];
    const int tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;       // 16 x 16 threads
    const int row_base = blockIdx.y * GS_BM, col_base = blockIdx.x * GS_BN;
    const int64_t k0 = (int64_t)blockIdx.z * kchunk;
    const int64_t k1 = k0 + kchunk < s1 ? k0 + kchunk : s1;
    double acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
    for (int64_t kk = k0; kk < k1; kk += GS_BK) {
        // A tile: 64 rows x 16 k  (1024 elements, 4 per thread), k fastest in global
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            int idx = tid + t * 256;
            int r = idx >> 4, k = idx & 15;
            int gr = row_base + r; int64_t gk = kk + k;
            As[k][r] = (gr < s2 && gk < k1) ? S2[(int64_t)gr * lds2 + gk] : 0.0;
        }
        // B tile: 16 k x 64 cols
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            int idx = tid + t * 256;
            int k = idx >> 6, c = idx & 63;
            int gc = col_base + c; int64_t gk = kk + k;
            Bs[k][c] = (gc < n && gk < k1) ? W1[gk * n + gc] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < GS_BK; ++k) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = As[k][ty + 16 * i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = Bs[k][tx + 16 * j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
    double* P = part + (int64_t)blockIdx.z * s2 * n;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        int gr = row_base + ty + 16 * i;
        if (gr >= s2) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int gc = col_base + tx + 16 * j;
            if (gc < n) P[(int64_t)gr * n + gc] = acc[i][j];
        }
    }
}

// N4: the same split-K product with S2 a dense Rademacher matrix generated on the fly (entries +-1/sqrt(s2),
// PAPER.md:947; reading S21): no S2 in memory, the A tile comes from 16 bits of the row's Philox words.
__global__ void __launch_bounds__(256)
k_rademacher_gemm_splitk(uint64_t seed, const double* __restrict__ W1, int64_t s1, int n, int s2,
                         int64_t kchunk, double* __restrict__ part)
{
    __shared__ double As[GS_BK][GS_BM + 1];
    __shared__ double Bs[GS_BK][GS_BN];
    const int tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;
    const int row_base = blockIdx.y * GS_BM, col_base = blockIdx.x * GS_BN;
    const int64_t k0 = (int64_t)blockIdx.z * kchunk;              // a multiple of GS_BK = 16
    const int64_t k1 = k0 + kchunk < s1 ? k0 + kchunk : s1;
    const uint64_t ng = (uint64_t)((s1 + 127) >> 7);
    const double inv = 1.0 / sqrt((double)s2);
    uint32_t o0 = 0, o1 = 0, o2 = 0, o3 = 0;
    int64_t gcur = -1;
    double acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
    for (int64_t kk = k0; kk < k1; kk += GS_BK) {
        if (tid < GS_BM) {                                        // one thread per row of the tile
            const int gr = row_base + tid;
            const int64_t g = kk >> 7;
            if (g != gcur) {
                uint32_t o[4];
                rqr_rademacher_bits(seed, (uint32_t)gr, ng, (uint64_t)g, o);
                o0 = o[0]; o1 = o[1]; o2 = o[2]; o3 = o[3];
                gcur = g;
            }
            const int b0 = (int)(kk & 127);
            const uint32_t word = b0 < 64 ? (b0 < 32 ? o0 : o1) : (b0 < 96 ? o2 : o3);
            const uint32_t bits = word >> (b0 & 31);
#pragma unroll
            for (int k = 0; k < GS_BK; ++k)
                As[k][tid] = (gr < s2 && kk + k < k1) ? (((bits >> k) & 1u) ? -inv : inv) : 0.0;
        }
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            int idx = tid + t * 256;
            int k = idx >> 6, c = idx & 63;
            int gc = col_base + c; int64_t gk = kk + k;
            Bs[k][c] = (gc < n && gk < k1) ? W1[gk * n + gc] : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < GS_BK; ++k) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = As[k][ty + 16 * i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = Bs[k][tx + 16 * j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
    double* P = part + (int64_t)blockIdx.z * s2 * n;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        int gr = row_base + ty + 16 * i;
        if (gr >= s2) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            int gc = col_base + tx + 16 * j;
            if (gc < n) P[(int64_t)gr * n + gc] = acc[i][j];
        }
    }
}

// out[e] = sum_p part[p][e].  Fixed order: 4 interleaved groups of partials (p = g, g+4, ...; 8
// loads in flight per thread), then the groups in order 0..3 through shared memory.
__global__ void __launch_bounds__(256)
k_reduce_partials(const double* __restrict__ part, int nparts, int64_t elems, double* __restrict__ out)
{
    __shared__ double sg[4][64];
    const int64_t e = (int64_t)blockIdx.x * 64 + (threadIdx.x & 63);
    const int g = threadIdx.x >> 6;
    double s = 0.0;
    if (e < elems) {
        const double* src = part + e;
        int p = g;
        for (; p + 28 < nparts; p += 32) {
            double x[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) x[u] = __ldcg(src + (int64_t)(p + 4 * u) * elems);
#pragma unroll
            for (int u = 0; u < 8; ++u) s += x[u];
        }
        for (; p < nparts; p += 4) s += __ldcg(src + (int64_t)p * elems);
    }
    sg[g][threadIdx.x & 63] = s;
    __syncthreads();
    if (g == 0 && e < elems) {
        const int l = threadIdx.x;
        out[e] = ((sg[0][l] + sg[1][l]) + sg[2][l]) + sg[3][l];
    }
}

extern "C" const double* rqr_workspace_S2(void* work, int n, int64_t s1)
{
    RqrLayout L = rqr_layout(1, n, s1);
    return (const double*)((char*)work + L.C);
}

extern "C" int rqr_workspace_rows(void* work, int64_t m, int n, int64_t s1, int variant, const uint32_t** offsets,
                                  const uint32_t** entries)
{
    if (!work) return -1;
    if (m < 1 || n < 2 || n > RQR_MAX_N || s1 < 1) return -2;
    RqrLayout L = rqr_layout(m, n, s1, (variant & RQR_S2_RADEMACHER) != 0);
    if (offsets) *offsets = (const uint32_t*)((char*)work + L.B_off);
    if (entries) *entries = (const uint32_t*)((char*)work + L.E);
    return RQR_OK;
}

extern "C" int rqr_gauss_sketch(const double* W1, int64_t s1, int n, int s2, uint64_t seed,
                                double* W, void* work, int flags, void* stream)
{
    if (!W1) return -1;
    if (s1 < 1 || s1 >= ((int64_t)1 << 31)) return -2;
    if (n < 2 || n > RQR_MAX_N) return -3;
    if (s2 < 1 || s2 > RQR_MAX_S2 || s2 > s1) return -4;
    if (!W) return -6;
    if (!work) return -7;
    cudaStream_t st = (cudaStream_t)stream;
    const bool rademacher = (flags & RQR_S2_RADEMACHER) != 0;
    RqrLayout L = rqr_layout(1, n, s1, rademacher);
    char* w = (char*)work;
    double* S2 = (double*)(w + L.C);
    double* part = (double*)(w + L.D);
    if (!rademacher && !(flags & RQR_FLAG_PREPARED)) {
        int rc = launch_prepare_S2(s1, s2, seed, S2, st);
        if (rc != RQR_OK) return rc;
    }
    int64_t ks_cap = RQR_GAUSS_PARTIAL_ROWS / s2;
    int64_t elems = (int64_t)s2 * n;
    {
        int ks_mma = 0;                           // n >= 96: FP64 DMMA GEMM (rqr_gauss_mma.cu)
        int rc = rqr_gauss_gemm_mma(rademacher ? nullptr : S2, W1, s1, n, s2, part, ks_cap, &ks_mma, st, seed);
        if (rc == RQR_OK) {
            k_reduce_partials<<<(int)((elems + 63) / 64), 256, 0, st>>>(part, ks_mma, elems, W);
            RQR_LAUNCH_CHECK();
            return RQR_OK;
        }
        if (rc != RQR_TALL_NOT_HANDLED) return rc;
    }
    int tiles_m = (s2 + GS_BM - 1) / GS_BM, tiles_n = (n + GS_BN - 1) / GS_BN;
    int64_t ks = 296 / (tiles_m * tiles_n);
    if (ks > ks_cap) ks = ks_cap;
    int64_t kblocks = (s1 + GS_BK - 1) / GS_BK;
    if (ks > kblocks) ks = kblocks;
    if (ks < 1) ks = 1;
    int64_t kchunk = ((kblocks + ks - 1) / ks) * GS_BK;
    ks = (s1 + kchunk - 1) / kchunk;
    dim3 grid(tiles_n, tiles_m, (unsigned)ks);
    if (rademacher) k_rademacher_gemm_splitk<<<grid, 256, 0, st>>>(seed, W1, s1, n, s2, kchunk, part);
    else k_gauss_gemm_splitk<<<grid, 256, 0, st>>>(S2, W1, s1, n, s2, kchunk, part);
    RQR_LAUNCH_CHECK();
    k_reduce_partials<<<(int)((elems + 63) / 64), 256, 0, st>>>(part, (int)ks, elems, W);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// =========================================================================================
// Single dense Gaussian sketch  W = S V,  S (s x m_total) = N(0,1)/sqrt(s) generated on the
// fly from Philox stream 3.  Comparator only.
// grid = (P persistent row-chunk walkers, ceil(s/32) sketch-row tiles).
// =========================================================================================
#define DG_ROWS 32
// NJ = column slots per thread (columns cq + 8 j, j < NJ: n <= 8 NJ), RT = sketch rows per thread (rows
// r + 32 k, k < RT: a tile of 32 RT sketch rows), so that one shared-memory load of V feeds RT fma.
// The Gaussians of a tile are drawn as Box-Muller PAIRS (entries 2q, 2q + 1 of the row-major S are the two
// outputs of Philox counter q): adjacent V rows share one evaluation whenever the first entry index is even.
template <int NJ, int RT>
__global__ void __launch_bounds__(256, NJ * RT <= 16 ? 3 : 2)
k_dense_gauss_sketch(const double* __restrict__ V, int64_t m, int n, int64_t ldv, int64_t row0,
                     int64_t m_total, int s, uint64_t seed, double* __restrict__ part)
{
    extern __shared__ double sm[];
    constexpr int TR = 32 * RT;              // sketch rows per tile
    constexpr int LDV = 8 * NJ;              // padded row of the V tile (pad columns are zero)
    double* St = sm;                         // [TR][33]
    double* Vt = sm + TR * 33;               // [32][LDV]
    const int tid = threadIdx.x;
    const int r = tid >> 3, cq = tid & 7;
    const double d = sqrt((double)s);
    double acc[RT][NJ];
#pragma unroll
    for (int k = 0; k < RT; ++k)
#pragma unroll
        for (int j = 0; j < NJ; ++j) acc[k][j] = 0.0;
    const int64_t nchunks = (m + DG_ROWS - 1) / DG_ROWS;
    for (int64_t ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
        const int64_t i0 = ch * DG_ROWS;
        for (int t = tid; t < TR * 16; t += 256) {
            const int rr = t >> 4, ii = 2 * (t & 15);
            const int sr = blockIdx.y * TR + rr;
            double v0 = 0.0, v1 = 0.0;
            if (sr < s && i0 + ii < m) {
                const uint64_t e = (uint64_t)sr * (uint64_t)m_total + (uint64_t)(row0 + i0 + ii);
                const bool second = i0 + ii + 1 < m;
                if (!(e & 1)) {
                    rqr_gauss_pair(seed, e >> 1, RQR_PHILOX_STREAM_DENSE, v0, v1);
                    if (!second) v1 = 0.0;
                } else {
                    v0 = rqr_gauss_entry(seed, e, RQR_PHILOX_STREAM_DENSE);
                    if (second) v1 = rqr_gauss_entry(seed, e + 1, RQR_PHILOX_STREAM_DENSE);
                }
            }
            St[rr * 33 + ii] = v0;
            St[rr * 33 + ii + 1] = v1;
        }
        for (int t = tid; t < 32 * LDV; t += 256) {
            const int ii = t / LDV, c = t - ii * LDV;
            Vt[t] = (c < n && i0 + ii < m) ? V[(i0 + ii) * ldv + c] : 0.0;
        }
        __syncthreads();
#pragma unroll 4
        for (int ii = 0; ii < 32; ++ii) {
            double a[RT];
#pragma unroll
            for (int k = 0; k < RT; ++k) a[k] = St[(r + 32 * k) * 33 + ii];
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const double v = Vt[ii * LDV + cq + 8 * j];
#pragma unroll
                for (int k = 0; k < RT; ++k) acc[k][j] = fma(a[k], v, acc[k][j]);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int k = 0; k < RT; ++k) {
        const int srow = blockIdx.y * TR + r + 32 * k;
        if (srow < s) {
            double* P = part + ((int64_t)blockIdx.x * s + srow) * n;
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int c = cq + 8 * j;
                if (c < n) P[c] = acc[k][j] / d;       // the 1/sqrt(s) of S, applied once per partial sum
            }
        }
    }
}

template <int NJ, int RT>
static int launch_dense_gauss(const double* V, int64_t m, int n, int64_t ldv, int64_t row0, int64_t m_total, int s,
                              uint64_t seed, double* part, int* P_out, cudaStream_t st)
{
    const int stiles = (s + 32 * RT - 1) / (32 * RT);
    const int64_t nchunks = (m + DG_ROWS - 1) / DG_ROWS;
    int64_t P = (148 * 4) / stiles;
    const int64_t Pcap = ((int64_t)rqr_gram_partial_cap(n) * n) / s;     // region A holds cap n^2 doubles
    if (P > Pcap) P = Pcap;
    if (P > nchunks) P = nchunks;
    if (P < 1) P = 1;
    const size_t smem = (size_t)(32 * RT * 33 + 32 * 8 * NJ) * sizeof(double);
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_dense_gauss_sketch<NJ, RT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
    });
    dim3 grid((unsigned)P, stiles);
    k_dense_gauss_sketch<NJ, RT><<<grid, 256, smem, st>>>(V, m, n, ldv, row0, m_total, s, seed, part);
    *P_out = (int)P;
    return RQR_OK;
}

extern "C" int rqr_dense_gauss_sketch(const double* V, int64_t m, int n, int64_t ldv, int64_t row0,
                                      int64_t m_total, int s, uint64_t seed, double* W, void* work,
                                      void* stream)
{
    if (!V) return -1;
    if (m < 1) return -2;
    if (n < 2 || n > RQR_MAX_N) return -3;
    if (ldv < n) return -4;
    if (row0 < 0 || row0 + m > m_total) return -5;
    if (s < 1 || s > RQR_MAX_S2) return -7;
    if (!W) return -9;
    if (!work) return -10;
    cudaStream_t st = (cudaStream_t)stream;
    double* part = (double*)((char*)work + 256);      // region A
    int P = 1;
    const int64_t elems = (int64_t)s * n;
    {
        // FP64 tensor-pipe kernel (rqr_dense_mma.cu): even n and ld, 16-byte aligned V
        const int64_t Pcap = ((int64_t)rqr_gram_partial_cap(n) * n) / s;
        int rc = rqr_dense_gauss_mma(V, m, n, ldv, row0, m_total, s, seed, part, Pcap, &P, false, st);
        if (rc == RQR_OK) {
            k_reduce_partials<<<(int)((elems + 63) / 64), 256, 0, st>>>(part, P, elems, W);
            RQR_LAUNCH_CHECK();
            return RQR_OK;
        }
        if (rc != RQR_TALL_NOT_HANDLED) return rc;
    }
    if (n <= 16) launch_dense_gauss<2, 4>(V, m, n, ldv, row0, m_total, s, seed, part, &P, st);
    else if (n <= 32) launch_dense_gauss<4, 4>(V, m, n, ldv, row0, m_total, s, seed, part, &P, st);
    else if (n <= 64) launch_dense_gauss<8, 4>(V, m, n, ldv, row0, m_total, s, seed, part, &P, st);
    else if (n <= 128) launch_dense_gauss<16, 2>(V, m, n, ldv, row0, m_total, s, seed, part, &P, st);
    else launch_dense_gauss<32, 1>(V, m, n, ldv, row0, m_total, s, seed, part, &P, st);
    RQR_LAUNCH_CHECK();
    k_reduce_partials<<<(int)((elems + 63) / 64), 256, 0, st>>>(part, P, elems, W);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// Measurement hook: the DRAW of the s x m Gaussians of rqr_dense_gauss_sketch alone (same launch shape, same
// per-lane Box-Muller pairs, no V traffic and no products): the generation bound of B''.  `work` as above.
extern "C" int rqr_debug_dense_gauss_draw_only(int64_t m, int n, int s, uint64_t seed, void* work, void* stream)
{
    if (m < 1) return -1;
    if (n < 2 || n > RQR_MAX_N || (n & 1)) return -2;
    if (s < 1 || s > RQR_MAX_S2) return -3;
    if (!work) return -5;
    double* part = (double*)((char*)work + 256);
    int P = 1;
    const int64_t Pcap = ((int64_t)rqr_gram_partial_cap(n) * n) / s;
    return rqr_dense_gauss_mma((const double*)work, m, n, n, 0, m, s, seed, part, Pcap, &P, true, (cudaStream_t)stream);
}

// =========================================================================================
// Inspection helpers for the parity tests
// =========================================================================================
__global__ void k_debug_hash_sign(uint64_t seed, int64_t row0, int64_t count, uint32_t s1,
                                  uint32_t* __restrict__ bucket, int8_t* __restrict__ sign)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count;
         i += (int64_t)gridDim.x * blockDim.x) {
        uint32_t b, neg;
        rqr_hash_sign(seed, (uint64_t)(row0 + i), s1, b, neg);
        bucket[i] = b;
        sign[i] = neg ? (int8_t)-1 : (int8_t)1;
    }
}

__global__ void k_debug_gauss(uint64_t seed, uint32_t stream_id, uint64_t first, int64_t count,
                              double* __restrict__ z)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count;
         i += (int64_t)gridDim.x * blockDim.x)
        z[i] = rqr_gauss_entry(seed, first + (uint64_t)i, stream_id);
}

extern "C" int rqr_debug_hash_sign(uint64_t seed, int64_t row0, int64_t count, int64_t s1,
                                   uint32_t* bucket, int8_t* sign, void* stream)
{
    if (count < 1) return -3;
    if (s1 < 1 || s1 >= ((int64_t)1 << 31)) return -4;
    if (!bucket) return -5;
    if (!sign) return -6;
    int blocks = (int)((count + 255) / 256 < 4096 ? (count + 255) / 256 : 4096);
    k_debug_hash_sign<<<blocks, 256, 0, (cudaStream_t)stream>>>(seed, row0, count, (uint32_t)s1, bucket, sign);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

__global__ void k_debug_rademacher(uint64_t seed, int64_t s1, int row, int64_t c0, int64_t count, int8_t* sign)
{
    const uint64_t ng = (uint64_t)((s1 + 127) >> 7);
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t c = c0 + i;
        uint32_t o[4];
        rqr_rademacher_bits(seed, (uint32_t)row, ng, (uint64_t)(c >> 7), o);
        const int b = (int)(c & 127);
        const uint32_t word = b < 64 ? (b < 32 ? o[0] : o[1]) : (b < 96 ? o[2] : o[3]);
        sign[i] = ((word >> (b & 31)) & 1u) ? (int8_t)-1 : (int8_t)1;
    }
}

extern "C" int rqr_debug_rademacher(uint64_t seed, int64_t s1, int row, int64_t c0, int64_t count, int8_t* sign,
                                    void* stream)
{
    if (s1 < 1 || s1 >= ((int64_t)1 << 31)) return -2;
    if (row < 0 || row >= RQR_MAX_S2) return -3;
    if (c0 < 0 || count < 1 || c0 + count > s1) return -4;
    if (!sign) return -6;
    int blocks = (int)((count + 255) / 256 < 4096 ? (count + 255) / 256 : 4096);
    k_debug_rademacher<<<blocks, 256, 0, (cudaStream_t)stream>>>(seed, s1, row, c0, count, sign);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

extern "C" int rqr_debug_gauss(uint64_t seed, uint32_t stream_id, uint64_t first, int64_t count,
                               double* z, void* stream)
{
    if (count < 1) return -4;
    if (!z) return -5;
    int blocks = (int)((count + 255) / 256 < 4096 ? (count + 255) / 256 : 4096);
    k_debug_gauss<<<blocks, 256, 0, (cudaStream_t)stream>>>(seed, stream_id, first, count, z);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}
