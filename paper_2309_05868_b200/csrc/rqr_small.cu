// rqr_small.cu -- the latency-bound n x n / s2 x n steps: A3 Householder R factor, A5 Cholesky,
// A7 triangular product.  Single-CTA kernels ("does not parallelize well").
#include "rqr_common.cuh"

__device__ __forceinline__ double warp_sum(double x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;      // identical in every lane (butterfly)
}

// =========================================================================================
// A3: R0 = R factor of the Householder QR of W (s2 x n), diag > 0   (Alg. 1 step 2)
// Register-resident version: 32 warps; warp w owns columns w + 32 q (q < CPW), lane l owns rows
// l + 32 p (p < RPL).  One __syncthreads per Householder step; the reflector v travels through
// a double-buffered shared vector.
// =========================================================================================
template <int RPL, int CPW>
__global__ void __launch_bounds__(1024, 1)
k_geqrf_reg(const double* __restrict__ W, int s2, int n, double* __restrict__ R0, int* d_info)
{
    __shared__ double vbuf[2][32 * RPL];
    __shared__ double beta_s[2];
    __shared__ unsigned char flip[32 * CPW];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double a[CPW][RPL];
#pragma unroll
    for (int q = 0; q < CPW; ++q)
#pragma unroll
        for (int p = 0; p < RPL; ++p) {
            int c = w + 32 * q, i = lane + 32 * p;
            a[q][p] = (c < n && i < s2) ? W[(int64_t)i * n + c] : 0.0;
        }
    for (int j = 0; j < n; ++j) {
        const int wo = j & 31, qo = j >> 5, lj = j & 31, pj = j >> 5;
        if (w == wo) {
            // owner: build the reflector of column j from rows >= j
            double tail2 = 0.0, x1 = 0.0;
#pragma unroll
            for (int q = 0; q < CPW; ++q) if (q == qo) {
#pragma unroll
                for (int p = 0; p < RPL; ++p) {
                    int i = lane + 32 * p;
                    if (i > j) tail2 += a[q][p] * a[q][p];
                    if (i == j) x1 = a[q][p];
                }
            }
            tail2 = warp_sum(tail2);
            x1 = __shfl_sync(0xffffffffu, x1, lj);
            const double nrm = sqrt(tail2 + x1 * x1);
            const double sgn = (x1 < 0.0) ? -1.0 : 1.0;
            const double vj = x1 + sgn * nrm;
            const double vtv = tail2 + vj * vj;
            const double beta = (vtv > 0.0) ? 2.0 / vtv : 0.0;
            if (lane == 0) {
                beta_s[j & 1] = beta;
                flip[j] = (sgn > 0.0);            // diagonal becomes -sgn*nrm
                if (!(nrm > 0.0) || !(nrm < 1.0e308)) rqr_set_info(d_info, RQR_INFO_SINGULAR + j + 1);
            }
#pragma unroll
            for (int q = 0; q < CPW; ++q) if (q == qo) {
#pragma unroll
                for (int p = 0; p < RPL; ++p) {
                    int i = lane + 32 * p;
                    double v = (i > j) ? a[q][p] : ((i == j) ? vj : 0.0);
                    vbuf[j & 1][i] = v;
                    if (i == j) a[q][p] = -sgn * nrm;     // H x = -sgn ||x|| e1
                    else if (i > j) a[q][p] = 0.0;
                }
            }
        }
        __syncthreads();
        double v[RPL];
#pragma unroll
        for (int p = 0; p < RPL; ++p) v[p] = vbuf[j & 1][lane + 32 * p];
        const double beta = beta_s[j & 1];
        double dot[CPW];
#pragma unroll
        for (int q = 0; q < CPW; ++q) {
            double s = 0.0;
#pragma unroll
            for (int p = 0; p < RPL; ++p) s = fma(v[p], a[q][p], s);
            dot[q] = s;
        }
#pragma unroll
        for (int q = 0; q < CPW; ++q) dot[q] = warp_sum(dot[q]);
#pragma unroll
        for (int q = 0; q < CPW; ++q) {
            int c = w + 32 * q;
            if (c > j && c < n) {
                const double ws = beta * dot[q];
#pragma unroll
                for (int p = 0; p < RPL; ++p) a[q][p] = fma(-ws, v[p], a[q][p]);
            }
        }
        (void)pj;
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < CPW; ++q)
#pragma unroll
        for (int p = 0; p < RPL; ++p) {
            int c = w + 32 * q, i = lane + 32 * p;
            if (c < n && i < n) {
                double r = (c >= i) ? a[q][p] : 0.0;
                if (c >= i && flip[i]) r = -r;
                R0[(int64_t)i * n + c] = r;
            }
        }
}

// Generic fallback, any 2 <= n <= 256, s2 <= 512: W stays in global memory (L2-resident) and is
// destroyed.  1024 threads = 4 row groups x 256 columns.
__global__ void __launch_bounds__(1024, 1)
k_geqrf_gmem(double* __restrict__ W, int s2, int n, double* __restrict__ R0, int* d_info)
{
    __shared__ double v[RQR_MAX_S2];
    __shared__ double pd[4][RQR_MAX_N];
    __shared__ double red[32];
    __shared__ double beta_s, diag_s;
    __shared__ unsigned char flip[RQR_MAX_N];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int g = tid >> 8, cc = tid & 255;
    for (int j = 0; j < n; ++j) {
        // reflector of column j
        double t2 = 0.0;
        for (int i = j + 1 + tid; i < s2; i += 1024) { double x = W[(int64_t)i * n + j]; t2 += x * x; }
        t2 = warp_sum(t2);
        if (lane == 0) red[wid] = t2;
        __syncthreads();
        if (wid == 0) {
            double s = warp_sum(red[lane]);
            if (lane == 0) {
                const double x1 = W[(int64_t)j * n + j];
                const double nrm = sqrt(s + x1 * x1);
                const double sgn = (x1 < 0.0) ? -1.0 : 1.0;
                const double vj = x1 + sgn * nrm;
                const double vtv = s + vj * vj;
                beta_s = (vtv > 0.0) ? 2.0 / vtv : 0.0;
                diag_s = -sgn * nrm;
                v[j] = vj;
                flip[j] = (sgn > 0.0);
                if (!(nrm > 0.0) || !(nrm < 1.0e308)) rqr_set_info(d_info, RQR_INFO_SINGULAR + j + 1);
            }
        }
        for (int i = j + 1 + tid; i < s2; i += 1024) v[i] = W[(int64_t)i * n + j];
        __syncthreads();
        // w_c = beta * v^T W[j:, c] for c > j
        const int c = j + 1 + cc;
        double s = 0.0;
        if (c < n) for (int i = j + g; i < s2; i += 4) s = fma(v[i], W[(int64_t)i * n + c], s);
        pd[g][cc] = s;
        __syncthreads();
        if (c < n) {
            const double ws = beta_s * (((pd[0][cc] + pd[1][cc]) + pd[2][cc]) + pd[3][cc]);
            for (int i = j + g; i < s2; i += 4) W[(int64_t)i * n + c] = fma(-ws, v[i], W[(int64_t)i * n + c]);
        }
        if (tid == 0) W[(int64_t)j * n + j] = diag_s;
        __syncthreads();
    }
    for (int e = tid; e < n * n; e += 1024) {
        int i = e / n, c = e - i * n;
        double r = (c >= i) ? W[(int64_t)i * n + c] : 0.0;
        if (c >= i && flip[i]) r = -r;
        R0[e] = r;
    }
}

extern "C" int rqr_small_geqrf(double* W, int s2, int n, double* R0, int* d_info, void* stream)
{
    if (!W) return -1;
    if (s2 < 1 || s2 > RQR_MAX_S2) return -2;
    if (n < 2 || n > RQR_MAX_N || n > s2) return -3;
    if (!R0) return -4;
    cudaStream_t st = (cudaStream_t)stream;
    const int rpl = (s2 + 31) / 32, cpw = (n + 31) / 32;
#define GEQRF_CASE(R, C)                                                              \
    if (rpl <= R && cpw <= C) {                                                       \
        k_geqrf_reg<R, C><<<1, 1024, 0, st>>>(W, s2, n, R0, d_info);                   \
        RQR_LAUNCH_CHECK();                                                           \
        return RQR_OK;                                                                \
    }
    GEQRF_CASE(1, 1) GEQRF_CASE(2, 1) GEQRF_CASE(4, 1) GEQRF_CASE(4, 2) GEQRF_CASE(8, 2)
    GEQRF_CASE(16, 1)
#undef GEQRF_CASE
    k_geqrf_gmem<<<1, 1024, 0, st>>>(W, s2, n, R0, d_info);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// =========================================================================================
// A5: upper Cholesky factor  G + shift I = R1^T R1   (Alg. 2 step 2)
// Right-looking, one CTA.  `A` is the working n x n array: shared memory when it fits
// (n <= 160), else the output buffer R1 in global memory.
// =========================================================================================
template <bool SMEM>
__global__ void __launch_bounds__(1024, 1)
k_chol(const double* __restrict__ G, int n, double shift_h, const double* __restrict__ d_shift,
       double* __restrict__ R1, int* d_info)
{
    const double shift = shift_h + (d_shift ? *d_shift : 0.0);
    extern __shared__ double sA[];
    __shared__ double dinv_s;
    __shared__ int fail_s;
    double* A = SMEM ? sA : R1;
    const int tid = threadIdx.x;
    for (int e = tid; e < n * n; e += 1024) {
        int i = e / n, c = e - i * n;
        A[e] = G[e] + ((i == c) ? shift : 0.0);
    }
    if (tid == 0) fail_s = 0;
    __syncthreads();
    for (int j = 0; j < n; ++j) {
        if (tid == 0) {
            const double d = A[j * n + j];
            if (!(d > 0.0) || !(d < 1.0e308)) { fail_s = j + 1; dinv_s = 0.0; }
            else { const double r = sqrt(d); A[j * n + j] = r; dinv_s = r; }
        }
        __syncthreads();
        if (fail_s) break;
        const double rjj = dinv_s;
        for (int c = j + 1 + tid; c < n; c += 1024) A[j * n + c] = A[j * n + c] / rjj;
        __syncthreads();
        // trailing update of the upper triangle: A[a][b] -= R[j][a] R[j][b], j < a <= b
        const int t = n - j - 1;
        for (int e = tid; e < t * t; e += 1024) {
            int a = e / t, b = e - a * t;
            if (b >= a) {
                a += j + 1; b += j + 1;
                A[a * n + b] = fma(-A[j * n + a], A[j * n + b], A[a * n + b]);
            }
        }
        __syncthreads();
    }
    if (fail_s) {
        if (tid == 0) rqr_set_info(d_info, RQR_INFO_NOT_SPD + fail_s);
    }
    __syncthreads();
    for (int e = tid; e < n * n; e += 1024) {
        int i = e / n, c = e - i * n;
        R1[e] = (c >= i) ? A[e] : 0.0;
    }
}

int rqr_chol_dev(const double* G, int n, double shift, const double* d_shift, double* R1,
                 int* d_info, cudaStream_t st);

extern "C" int rqr_chol(const double* G, int n, double shift, double* R1, int* d_info, void* stream)
{
    return rqr_chol_dev(G, n, shift, nullptr, R1, d_info, (cudaStream_t)stream);
}

// shift = 11 (m n + n (n+1)) 2^-53 tr(G)   (shifted CholeskyQR3, reading S9)
__global__ void k_scholqr3_shift(const double* __restrict__ G, int n, double m, double* out)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double tr = 0.0;
        for (int j = 0; j < n; ++j) tr += G[j * n + j];
        *out = 11.0 * (m * n + (double)n * (n + 1)) * 0x1p-53 * tr;
    }
}

int rqr_scholqr3_shift(const double* G, int n, int64_t m, double* d_out, cudaStream_t st)
{
    k_scholqr3_shift<<<1, 32, 0, st>>>(G, n, (double)m, d_out);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

int rqr_chol_dev(const double* G, int n, double shift, const double* d_shift, double* R1,
                 int* d_info, cudaStream_t st)
{
    if (!G) return -1;
    if (n < 2 || n > RQR_MAX_N) return -2;
    if (!R1) return -4;
    if (G == R1) return -4;
    size_t bytes = (size_t)n * n * sizeof(double);
    if (bytes <= 200 * 1024) {
        static bool attr_set = false;
        if (!attr_set) {
            cudaFuncSetAttribute(k_chol<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
            attr_set = true;
        }
        k_chol<true><<<1, 1024, bytes, st>>>(G, n, shift, d_shift, R1, d_info);
    } else {
        k_chol<false><<<1, 1024, 0, st>>>(G, n, shift, d_shift, R1, d_info);
    }
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// =========================================================================================
// A7: R = R1 R0, upper x upper   (Alg. 3 step 3)
// =========================================================================================
__global__ void k_triu_mul(const double* __restrict__ R1, const double* __restrict__ R0, int n,
                           double* __restrict__ R)
{
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n * n; e += gridDim.x * blockDim.x) {
        int a = e / n, c = e - a * n;
        double acc = 0.0;
        for (int k = a; k <= c; ++k) acc = fma(R1[a * n + k], R0[k * n + c], acc);
        R[e] = (c >= a) ? acc : 0.0;
    }
}

extern "C" int rqr_triu_mul(const double* R1, const double* R0, int n, double* R, void* stream)
{
    if (!R1) return -1;
    if (!R0) return -2;
    if (n < 2 || n > RQR_MAX_N) return -3;
    if (!R || R == R1 || R == R0) return -4;
    int blocks = (n * n + 255) / 256;
    if (blocks > 148) blocks = 148;
    k_triu_mul<<<blocks, 256, 0, (cudaStream_t)stream>>>(R1, R0, n, R);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}
