// rqr_tall.cu -- the m-sized passes: A4 fused V R0^-1 + Gram (rqr_trsm_gram) and A6 triangular
// apply (rqr_apply).  This file holds the GENERIC kernels (any 2 <= n <= 256, any ld); the
// DMMA fast paths live in rqr_tall_mma.cu and are dispatched from here.
#include "rqr_common.cuh"
#include "rqr_tall.cuh"

#define GEN_TR 64      // rows per tile in the generic kernels

// One row of X = V R^-1 by forward substitution (eq. (42)), in place in a
// shared-memory row.  Explicit fma so that every kernel that calls it rounds identically (H1).
__device__ __forceinline__ void row_trsm_inplace(double* __restrict__ x, const double* __restrict__ R,
                                                 int n)
{
    for (int j = 0; j < n; ++j) {
        double acc = x[j];
        for (int k = 0; k < j; ++k) acc = fma(-x[k], __ldg(R + k * n + j), acc);
        x[j] = acc / __ldg(R + j * n + j);
    }
}

// Generic A4: per 64-row tile: load, optional row-wise substitution, optional store of V1, then
// this CTA's partial Gram (upper triangle) accumulated in its own slice of `part`.
__global__ void __launch_bounds__(256)
k_trsm_gram_generic(const double* V, int64_t m, int n, int64_t ldv,      // V1 == V allowed: no restrict on either
                    const double* __restrict__ R0, double* V1, int64_t ldq,
                    double* __restrict__ part)
{
    extern __shared__ double Xs[];                // GEN_TR x (n+1)
    const int ld = n + 1;
    const int tid = threadIdx.x;
    double* P = part + (int64_t)blockIdx.x * n * n;
    for (int e = tid; e < n * n; e += 256) P[e] = 0.0;
    const int64_t ntiles = (m + GEN_TR - 1) / GEN_TR;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t i0 = t * GEN_TR;
        const int rows = (int)((m - i0) < GEN_TR ? (m - i0) : GEN_TR);
        __syncthreads();
        for (int e = tid; e < GEN_TR * n; e += 256) {
            int r = e / n, c = e - r * n;
            Xs[r * ld + c] = (r < rows) ? V[(i0 + r) * ldv + c] : 0.0;
        }
        __syncthreads();
        if (R0 && tid < rows) row_trsm_inplace(Xs + tid * ld, R0, n);
        __syncthreads();
        if (V1) {
            for (int e = tid; e < rows * n; e += 256) {
                int r = e / n, c = e - r * n;
                V1[(i0 + r) * ldq + c] = Xs[r * ld + c];
            }
        }
        for (int e = tid; e < n * n; e += 256) {
            int a = e / n, b = e - a * n;
            if (b < a) continue;
            double s = 0.0;
            for (int r = 0; r < GEN_TR; ++r) s = fma(Xs[r * ld + a], Xs[r * ld + b], s);
            P[e] += s;
        }
    }
}

// G[a][b] = G[b][a] = sum_p part[p][a][b] (a <= b).  Fixed order: 4 interleaved groups of partials
// (p = g, g+4, ...; 8 loads in flight per thread), then the groups in order 0..3 through shared
// memory.  One CTA per 64 consecutive entries of a row: latency-bound, so wide and shallow.
__global__ void __launch_bounds__(256)
k_gram_reduce(const double* __restrict__ part, int nparts, int n, double* __restrict__ G)
{
    __shared__ double sg[4][64];
    const int a = blockIdx.y, b = blockIdx.x * 64 + (threadIdx.x & 63), g = threadIdx.x >> 6;
    double s = 0.0;
    if (b < n && b >= a) {
        const double* src = part + (int64_t)a * n + b;
        const int64_t nn = (int64_t)n * n;
        int p = g;
        for (; p + 28 < nparts; p += 32) {
            double x[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) x[u] = __ldcg(src + (int64_t)(p + 4 * u) * nn);
#pragma unroll
            for (int u = 0; u < 8; ++u) s += x[u];
        }
        for (; p < nparts; p += 4) s += __ldcg(src + (int64_t)p * nn);
    }
    sg[g][threadIdx.x & 63] = s;
    __syncthreads();
    if (g == 0 && b < n && b >= a) {
        const int l = threadIdx.x;
        const double t = ((sg[0][l] + sg[1][l]) + sg[2][l]) + sg[3][l];
        G[(int64_t)a * n + b] = t;
        G[(int64_t)b * n + a] = t;
    }
}

// Generic A6: Q = (V R0^-1) R1^-1 row by row; R0 == NULL: Q = V R1^-1.
__global__ void __launch_bounds__(256)
k_apply_generic(const double* V, int64_t m, int n, int64_t ldv,          // Q == V allowed: no restrict on either
                const double* __restrict__ R0, const double* __restrict__ R1,
                double* Q, int64_t ldq)
{
    extern __shared__ double Xs[];
    const int ld = n + 1;
    const int tid = threadIdx.x;
    const int64_t ntiles = (m + GEN_TR - 1) / GEN_TR;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t i0 = t * GEN_TR;
        const int rows = (int)((m - i0) < GEN_TR ? (m - i0) : GEN_TR);
        __syncthreads();
        for (int e = tid; e < rows * n; e += 256) {
            int r = e / n, c = e - r * n;
            Xs[r * ld + c] = V[(i0 + r) * ldv + c];
        }
        __syncthreads();
        if (tid < rows) {
            if (R0) row_trsm_inplace(Xs + tid * ld, R0, n);
            row_trsm_inplace(Xs + tid * ld, R1, n);
        }
        __syncthreads();
        for (int e = tid; e < rows * n; e += 256) {
            int r = e / n, c = e - r * n;
            Q[(i0 + r) * ldq + c] = Xs[r * ld + c];
        }
    }
}

static int generic_grid(int64_t m)
{
    int64_t ntiles = (m + GEN_TR - 1) / GEN_TR;
    int64_t g = ntiles < RQR_MAX_GRAM_PARTIALS ? ntiles : RQR_MAX_GRAM_PARTIALS;
    return (int)(g < 1 ? 1 : g);
}

static void generic_attrs()
{
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_trsm_gram_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
        cudaFuncSetAttribute(k_apply_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
    });
}

static int trsm_gram_impl(const double* V, int64_t m, int n, int64_t ldv, const double* R0,
                          double* G, double* V1, int64_t ldq, void* work, void* stream, bool force_generic)
{
    if (!V) return -1;
    if (m < 1 || m >= ((int64_t)1 << 31)) return -2;
    if (n < 2 || n > RQR_MAX_N) return -3;
    if (ldv < n) return -4;
    if (!G) return -6;
    if (V1 && ldq < n) return -8;
    if (!work) return -9;
    cudaStream_t st = (cudaStream_t)stream;
    double* part = (double*)((char*)work + 256);        // region A
    int nparts = 0;
    double* frags = (double*)((char*)work + rqr_layout(1, n, 1).A_frags);
    // rows are processed in chunks, one partial set per chunk (rqr_gram_partial_cap): bounded accumulation chains
    const int cap = rqr_gram_partial_cap(n);
    int64_t chunk = RQR_GRAM_CHUNK_ROWS;
    while ((m + chunk - 1) / chunk * 148 > cap) chunk *= 2;
    int rc = RQR_TALL_NOT_HANDLED;
    if (!force_generic) {
        for (int64_t r0 = 0; r0 < m; r0 += chunk) {
            const int64_t mc = (m - r0) < chunk ? (m - r0) : chunk;
            int np = 0;
            rc = rqr_trsm_gram_mma(V + r0 * ldv, mc, n, ldv, R0, V1 ? V1 + r0 * ldq : nullptr, ldq,
                                   part + (size_t)nparts * n * n, &np, st);
            if (rc != RQR_OK) break;
            nparts += np;
        }
        if (rc == RQR_TALL_NOT_HANDLED) {
            nparts = 0;
            rc = rqr_trsm_gram_panel(V, m, n, ldv, R0, V1, ldq, part, &nparts, frags, chunk, st);
        }
    }
    if (rc == RQR_TALL_NOT_HANDLED) {
        generic_attrs();
        nparts = generic_grid(m);
        size_t smem = (size_t)GEN_TR * (n + 1) * sizeof(double);
        k_trsm_gram_generic<<<nparts, 256, smem, st>>>(V, m, n, ldv, R0, V1, ldq, part);
        RQR_LAUNCH_CHECK();
    } else if (rc != RQR_OK) return rc;
    dim3 rgrid((n + 63) / 64, n);
    k_gram_reduce<<<rgrid, 256, 0, st>>>(part, nparts, n, G);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

extern "C" int rqr_trsm_gram(const double* V, int64_t m, int n, int64_t ldv, const double* R0,
                             double* G, double* V1, int64_t ldq, void* work, void* stream)
{
    return trsm_gram_impl(V, m, n, ldv, R0, G, V1, ldq, work, stream, false);
}
extern "C" int rqr_debug_trsm_gram_generic(const double* V, int64_t m, int n, int64_t ldv, const double* R0,
                                           double* G, double* V1, int64_t ldq, void* work, void* stream)
{
    return trsm_gram_impl(V, m, n, ldv, R0, G, V1, ldq, work, stream, true);
}

static int apply_impl(const double* V, int64_t m, int n, int64_t ldv, const double* R0,
                      const double* R1, double* Q, int64_t ldq, void* work, void* stream, bool force_generic)
{
    if (!V) return -1;
    if (m < 1 || m >= ((int64_t)1 << 31)) return -2;
    if (n < 2 || n > RQR_MAX_N) return -3;
    if (ldv < n) return -4;
    if (!R1) return -6;
    if (!Q) return -7;
    if (ldq < n) return -8;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = force_generic ? RQR_TALL_NOT_HANDLED : rqr_apply_mma(V, m, n, ldv, R0, R1, Q, ldq, st);
    if (rc == RQR_TALL_NOT_HANDLED && !force_generic && n > 64) {
        if (!work) return -9;
        rc = rqr_apply_panel(V, m, n, ldv, R0, R1, Q, ldq,
                             (double*)((char*)work + rqr_layout(1, n, 1).A_frags), st);
    }
    if (rc == RQR_TALL_NOT_HANDLED) {
        generic_attrs();
        size_t smem = (size_t)GEN_TR * (n + 1) * sizeof(double);
        int64_t ntiles = (m + GEN_TR - 1) / GEN_TR;
        int grid = (int)(ntiles < 148 * 8 ? ntiles : 148 * 8);
        k_apply_generic<<<grid, 256, smem, st>>>(V, m, n, ldv, R0, R1, Q, ldq);
        RQR_LAUNCH_CHECK();
        return RQR_OK;
    }
    return rc;
}

extern "C" int rqr_apply(const double* V, int64_t m, int n, int64_t ldv, const double* R0,
                         const double* R1, double* Q, int64_t ldq, void* work, void* stream)
{
    return apply_impl(V, m, n, ldv, R0, R1, Q, ldq, work, stream, false);
}
extern "C" int rqr_debug_apply_generic(const double* V, int64_t m, int n, int64_t ldv, const double* R0,
                                       const double* R1, double* Q, int64_t ldq, void* work, void* stream)
{
    return apply_impl(V, m, n, ldv, R0, R1, Q, ldq, work, stream, true);
}

// ---------------------------------------------------------------------------------------
// rqr_trsm_gram_noalloc: A4 with the Gram partials in a file-scope device array instead of the caller's workspace
// (include/rqr.h).  One array per device that loads the library, shared by every call: calls that overlap on the
// GPU race on it.  Nothing in it must start at zero: CTA p overwrites partial p before k_gram_reduce reads it.
// ---------------------------------------------------------------------------------------
static __device__ __align__(256) double d_noalloc_gram_part[(size_t)RQR_NOALLOC_MAX_PARTIALS * RQR_NOALLOC_MAX_N * RQR_NOALLOC_MAX_N];

// Device address of the array on the CURRENT device.  In host code `d_noalloc_gram_part` is only a stand-in for the
// symbol, not an address a kernel may use; cudaGetSymbolAddress resolves it per device.  Looked up once per device.
static double* noalloc_gram_part()
{
    static std::atomic<double*> addr[RQR_MAX_DEVICES];
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    const bool keep = dev >= 0 && dev < RQR_MAX_DEVICES;
    if (keep) {
        double* p = addr[dev].load(std::memory_order_acquire);
        if (p) return p;
    }
    double* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, d_noalloc_gram_part) != cudaSuccess || !p) {
        cudaGetLastError();
        return nullptr;
    }
    if (keep) addr[dev].store(p, std::memory_order_release);
    return p;
}

extern "C" int rqr_trsm_gram_noalloc(const double* V, int64_t m, int n, int64_t ldv, const double* R0,
                                     double* G, double* V1, int64_t ldq, void* stream)
{
    if (!V) return -1;
    if (m < 1) return -2;
    if (n < 2) return -3;
    if (n > RQR_NOALLOC_MAX_N || m > RQR_NOALLOC_MAX_M) return RQR_ERR_SCRATCH_LIMIT;
    if (ldv < n) return -4;
    if (!G) return -6;
    if (V1 && ldq < n) return -8;
    double* part = noalloc_gram_part();
    if (!part) return RQR_ERR_LAUNCH;
    cudaStream_t st = (cudaStream_t)stream;
    int nparts = 0;
    // n <= 64 and one chunk of rows: the DMMA kernels run at most 148 CTAs, one partial each
    int rc = rqr_trsm_gram_mma(V, m, n, ldv, R0, V1, ldq, part, &nparts, st);
    if (rc == RQR_TALL_NOT_HANDLED) {
        generic_attrs();
        nparts = generic_grid(m);
        if (nparts > RQR_NOALLOC_MAX_PARTIALS) nparts = RQR_NOALLOC_MAX_PARTIALS;
        size_t smem = (size_t)GEN_TR * (n + 1) * sizeof(double);
        k_trsm_gram_generic<<<nparts, 256, smem, st>>>(V, m, n, ldv, R0, V1, ldq, part);
        RQR_LAUNCH_CHECK();
    } else if (rc != RQR_OK) return rc;
    dim3 rgrid((n + 63) / 64, n);
    k_gram_reduce<<<rgrid, 256, 0, st>>>(part, nparts, n, G);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}
