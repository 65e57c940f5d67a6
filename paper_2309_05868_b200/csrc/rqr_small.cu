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

// Small-shape version (s2 <= 128, n <= 64: the n = 64 configs).  A Householder step is a chain of
// dependent latencies executed by ONE warp, so the kernel is written for few instructions per step
// (measured on B200: DFMA 8.7 cycles dependent, double shuffle-add round 41, sqrt 95, 1/x 77):
//   * 8 warps; lane = 8 g + t: column c = 8 w + 4 qq + g (qq = 0, 1), rows i = t + 8 p (p < 16): a dot
//     product is 16 local fma and a 3-round shuffle reduction inside the 8-lane group;
//   * finished entries LEAVE the register tile: after step j row j (final R0[j][j+1:]) is written to
//     global memory and zeroed, the pivot column is zeroed.  The tile then only holds rows > j of
//     columns > j, so norms, dot products and updates need no row or column predicates;
//   * beta = 2 / v^T v = 1 / (nrm |v_j|) is formed by every thread in the shadow of its dot product.
__device__ __forceinline__ double group8_sum(double x)
{
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// A/B switch of the single-factorization kernel, compile time only (-DRQR_GEQRF_G8X=0: eight columns per warp)
#ifndef RQR_GEQRF_G8X
#define RQR_GEQRF_G8X 1
#endif

// timing hooks of a working experiment (compiled out unless RQR_G8_TRACE is defined by the including file)
#ifndef RQR_G8_MARK
#define RQR_G8_MARK(k)
#endif

// One Householder step of k_geqrf_g8 with the row-slot index of the pivot, P = j / 8, known at
// compile time: slots p < P hold finished (zeroed) rows and are skipped, the pivot element is
// col[P] of lane t == j % 8 without a select.  QQ = column quads per warp: QQ = 2 (8 warps, warp w holds columns
// 8 w + 4 qq + g, owner of column j is w == P) or QQ = 1 (16 warps, columns 4 w + g, owner w == j / 4): the same
// arithmetic column by column (bit-identical results), half the instructions per warp and step on the chain.
template <int P, int QQ>
__device__ __forceinline__ void geqrf_g8_step(double (&a)[QQ][16], int j, int n, int w, int lane,
                                              double (*vbuf)[128], double* den_s, double* sgn_s,
                                              double* __restrict__ R0, int* d_info)
{
    const int g = lane >> 3, t = lane & 7, tj = j & 7;
    RQR_G8_MARK(0);
    if (w == (QQ == 2 ? P : (j >> 2))) {                   // warp-uniform: the warp that owns column j
        auto reflect = [&](double (&col)[16]) {
            double s0 = 0.0, s1 = 0.0;
#pragma unroll
            for (int p = P; p < 16; p += 2) {
                s0 = fma(col[p], col[p], s0);
                if (p + 1 < 16) s1 = fma(col[p + 1], col[p + 1], s1);
            }
            const double ss = group8_sum(s0 + s1);                                   // ||a[j:, j]||^2
            const double x1 = __shfl_sync(0xffffffffu, col[P], (lane & 24) | tj);    // a[j][j]
            const double nrm = sqrt(ss);
            const double sgn = (x1 < 0.0) ? -1.0 : 1.0;
            const double vj = x1 + sgn * nrm;
            if (g == (j & 3)) {
#pragma unroll
                for (int p = P; p < 16; ++p) vbuf[j & 1][t + 8 * p] = col[p];        // rows < j are zero
                if (t == tj) vbuf[j & 1][j] = vj;
                if (t == 0) {
                    den_s[j & 1] = nrm * fabs(vj);                                   // v^T v / 2
                    sgn_s[j & 1] = sgn;
                    R0[(int64_t)j * n + j] = nrm;               // -sgn*nrm, row negated when sgn > 0 (S4)
                    if (!(nrm > 0.0) || !(nrm < 1.0e308)) rqr_set_info(d_info, RQR_INFO_SINGULAR + j + 1);
                }
#pragma unroll
                for (int p = P; p < 16; ++p) col[p] = 0.0;                           // column j is done
            }
        };
        if (QQ == 2 && ((j >> 2) & 1)) reflect(a[QQ - 1]); else reflect(a[0]);
    }
    RQR_G8_MARK(1);
    __syncthreads();
    RQR_G8_MARK(2);
    if (4 * QQ * w + 4 * QQ - 1 <= j) return;        // warp-uniform: every column of this warp is finished (all zero);
                                                     // it only keeps the barriers
    double v[16];
#pragma unroll
    for (int p = P; p < 16; ++p) v[p] = vbuf[j & 1][t + 8 * p];
    const double den = den_s[j & 1], sg = sgn_s[j & 1];
    const double beta = (den > 0.0) ? 1.0 / den : 0.0;
    double dot[QQ];
#pragma unroll
    for (int qq = 0; qq < QQ; ++qq) {
        double s0 = 0.0, s1 = 0.0;
#pragma unroll
        for (int p = P; p < 16; p += 2) {
            s0 = fma(v[p], a[qq][p], s0);
            if (p + 1 < 16) s1 = fma(v[p + 1], a[qq][p + 1], s1);
        }
        dot[qq] = s0 + s1;
    }
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
#pragma unroll
        for (int qq = 0; qq < QQ; ++qq) dot[qq] += __shfl_xor_sync(0xffffffffu, dot[qq], o);
    }
    RQR_G8_MARK(3);
#pragma unroll
    for (int qq = 0; qq < QQ; ++qq) {
        const double ws = beta * dot[qq];            // finished and padding columns are all zero: ws = 0
#pragma unroll
        for (int p = P; p < 16; ++p) a[qq][p] = fma(-ws, v[p], a[qq][p]);
    }
    if (t == tj) {                                   // row j is final: move it out of the tile
#pragma unroll
        for (int qq = 0; qq < QQ; ++qq) {
            const int c = 4 * QQ * w + 4 * qq + g;
            const double val = a[qq][P];
            a[qq][P] = 0.0;
            if (c > j && c < n) R0[(int64_t)j * n + c] = (sg > 0.0) ? -val : val;
        }
    }
    RQR_G8_MARK(4);
}

template <int P, int QQ>
__device__ __forceinline__ void geqrf_g8_steps(double (&a)[QQ][16], int n, int w, int lane, double (*vbuf)[128],
                                               double* den_s, double* sgn_s, double* __restrict__ R0, int* d_info)
{
    if constexpr (P < 8) {
        const int jend = (8 * P + 8 < n) ? 8 * P + 8 : n;
        for (int j = 8 * P; j < jend; ++j) geqrf_g8_step<P, QQ>(a, j, n, w, lane, vbuf, den_s, sgn_s, R0, d_info);
        if (8 * P + 8 < n) geqrf_g8_steps<P + 1, QQ>(a, n, w, lane, vbuf, den_s, sgn_s, R0, d_info);
    }
}

template <int QQ>
__device__ __forceinline__ void geqrf_g8_body(const double* __restrict__ W, int s2, int n, double* __restrict__ R0,
                                              int* d_info)
{
    __shared__ double vbuf[2][128];
    __shared__ double den_s[2], sgn_s[2];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int g = lane >> 3, t = lane & 7;
    double a[QQ][16];
#pragma unroll
    for (int qq = 0; qq < QQ; ++qq)
#pragma unroll
        for (int p = 0; p < 16; ++p) {
            const int c = 4 * QQ * w + 4 * qq + g, i = t + 8 * p;
            a[qq][p] = (c < n && i < s2) ? W[(int64_t)i * n + c] : 0.0;
        }
    for (int e = threadIdx.x; e < n * n; e += blockDim.x) {      // exact zeros below the diagonal
        const int i = e / n, c = e - i * n;
        if (c < i) R0[e] = 0.0;
    }
    geqrf_g8_steps<0, QQ>(a, n, w, lane, vbuf, den_s, sgn_s, R0, d_info);
}

__global__ void __launch_bounds__(256, 1)
k_geqrf_g8(const double* __restrict__ W, int s2, int n, double* __restrict__ R0, int* d_info)
{
    geqrf_g8_body<2>(W, s2, n, R0, d_info);
}

// four columns per warp (QQ = 1), ceil(n / 4) <= 8 warps: the single factorization of A3 at n <= 32
__global__ void __launch_bounds__(256, 1)
k_geqrf_g8x(const double* __restrict__ W, int s2, int n, double* __restrict__ R0, int* d_info)
{
    geqrf_g8_body<1>(W, s2, n, R0, d_info);
}

// One level of a TSQR tree: block b = rows [b rows/nb, (b+1) rows/nb) of A (at most 128 each), its R
// factor goes to Rout + b n^2.  A rank-deficient BLOCK is not an error of the tree: d_info is NULL
// except at the root.
__global__ void __launch_bounds__(256, 1)
k_geqrf_g8_batched(const double* __restrict__ A, int64_t rows, int nb, int n, double* __restrict__ Rout)
{
    const int64_t r0 = (int64_t)blockIdx.x * rows / nb, r1 = (int64_t)(blockIdx.x + 1) * rows / nb;
    geqrf_g8_body<2>(A + r0 * n, (int)(r1 - r0), n, Rout + (int64_t)blockIdx.x * n * n, nullptr);
}

// R factor of the Householder QR of a TALL matrix A (rows x n, n <= 64, any rows >= n) by a TSQR tree of
// k_geqrf_g8 blocks: level by level, blocks of at most 128 rows are reduced to their n x n R factors, which are
// stacked and reduced again.  R (diag > 0) is unique, so the tree gives the R of plain Householder QR to rounding.
// `scratch` holds the stacked R factors of two consecutive levels: 1.5 * ceil(rows / 128) * n * n doubles.
int rqr_tsqr_r_dev(const double* A, int64_t rows, int n, double* R, double* scratch, int* d_info, cudaStream_t st)
{
    const double* in = A;
    int64_t rows_in = rows;
    double* out = scratch;
    double* other = scratch + ((rows + 127) / 128) * (int64_t)n * n;
    for (;;) {
        const int64_t nb = (rows_in + 127) / 128;
        if (nb <= 1) {
            if (RQR_GEQRF_G8X && n <= 32) k_geqrf_g8x<<<1, 32 * ((n + 3) / 4), 0, st>>>(in, (int)rows_in, n, R, d_info);
            else                          k_geqrf_g8<<<1, 256, 0, st>>>(in, (int)rows_in, n, R, d_info);
            RQR_LAUNCH_CHECK();
            return RQR_OK;
        }
        k_geqrf_g8_batched<<<(unsigned)nb, 256, 0, st>>>(in, rows_in, (int)nb, n, out);
        RQR_LAUNCH_CHECK();
        in = out;
        rows_in = nb * n;
        double* t = out; out = other; other = t;
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


// ---- thread-block-cluster helpers (CTAs of a cluster run on SMs of one GPC; barrier.cluster costs
// ~380 cycles; release/acquire at cluster scope orders global-memory traffic between the CTAs) ----
__device__ __forceinline__ unsigned cluster_rank()
{
    unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r;
}
__device__ __forceinline__ unsigned cluster_size()
{
    unsigned r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// Cluster version of k_geqrf_reg for shapes whose register tile does not fit one CTA (n > 64):
// W is spread over the CTAs of one cluster, column c -> CTA c % ncta, warp (c / ncta) % 16,
// slot (c / ncta) / 16; lane l owns rows l + 32 p.  512 threads per CTA.  After the load W's own
// storage is scratch: the reflector v (double-buffered), beta and the sign flags travel through
// it (L2) with ONE cluster barrier per Householder step.
template <int RPL, int CPW>
__global__ void __launch_bounds__(512, 1)
k_geqrf_cluster(double* W, int s2, int n, double* R0, int* d_info, int64_t rows_total, int nb)
{
    __shared__ double vs[32 * RPL];          // this step's reflector (registers hold the columns only)
    const int ncta = (int)cluster_size(), rank = (int)cluster_rank();
    if (nb > 0) {
        // one level of a TSQR tree (n > 64): cluster c factors rows [c rows_total / nb, (c+1) rows_total / nb) of W
        // (at most 32 RPL each, destroyed) and writes its R factor to R0 + c n^2; a rank-deficient BLOCK is not an
        // error of the tree
        const int64_t cid = blockIdx.x / ncta;
        const int64_t r0 = cid * rows_total / nb, r1 = (cid + 1) * rows_total / nb;
        W += r0 * n;
        s2 = (int)(r1 - r0);
        R0 += cid * (int64_t)n * n;
        d_info = nullptr;
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double a[CPW][RPL];
#pragma unroll
    for (int q = 0; q < CPW; ++q)
#pragma unroll
        for (int p = 0; p < RPL; ++p) {
            const int c = (w + 16 * q) * ncta + rank, i = lane + 32 * p;
            a[q][p] = (c < n && i < s2) ? W[(int64_t)i * n + c] : 0.0;
        }
    cluster_sync_all();                      // everyone holds its columns: W is scratch from here on
    double* gv = W;                          // [2][32 * RPL]
    double* gbeta = W + 2 * 32 * RPL;        // [2]
    double* gflip = gbeta + 2;               // [n]
    for (int j = 0; j < n; ++j) {
        const int o = j % ncta, jj = j / ncta, wo = jj & 15, qo = jj >> 4, lj = j & 31;
        double* vj_buf = gv + (j & 1) * 32 * RPL;
        if (rank == o && w == wo) {
            double tail2 = 0.0, x1 = 0.0;
#pragma unroll
            for (int q = 0; q < CPW; ++q) if (q == qo) {
#pragma unroll
                for (int p = 0; p < RPL; ++p) {
                    const int i = lane + 32 * p;
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
                gbeta[j & 1] = beta;
                gflip[j] = (sgn > 0.0) ? 1.0 : 0.0;       // diagonal becomes -sgn*nrm
                if (!(nrm > 0.0) || !(nrm < 1.0e308)) rqr_set_info(d_info, RQR_INFO_SINGULAR + j + 1);
            }
#pragma unroll
            for (int q = 0; q < CPW; ++q) if (q == qo) {
#pragma unroll
                for (int p = 0; p < RPL; ++p) {
                    const int i = lane + 32 * p;
                    vj_buf[i] = (i > j) ? a[q][p] : ((i == j) ? vj : 0.0);
                    if (i == j) a[q][p] = -sgn * nrm;
                    else if (i > j) a[q][p] = 0.0;
                }
            }
        }
        cluster_sync_all();
        for (int i = threadIdx.x; i < 32 * RPL; i += 512) vs[i] = __ldcg(vj_buf + i);
        const double beta = __ldcg(gbeta + (j & 1));
        __syncthreads();
        const double* v = vs + lane;
        double dot[CPW];
#pragma unroll
        for (int q = 0; q < CPW; ++q) {
            double s0 = 0.0, s1_ = 0.0;
#pragma unroll
            for (int p = 0; p < RPL; p += 2) {
                s0 = fma(v[32 * p], a[q][p], s0);
                s1_ = fma(v[32 * (p + 1)], a[q][p + 1], s1_);
            }
            dot[q] = s0 + s1_;
        }
#pragma unroll
        for (int q = 0; q < CPW; ++q) dot[q] = warp_sum(dot[q]);
#pragma unroll
        for (int q = 0; q < CPW; ++q) {
            const int c = (w + 16 * q) * ncta + rank;
            if (c > j && c < n) {
                const double ws = beta * dot[q];
#pragma unroll
                for (int p = 0; p < RPL; ++p) a[q][p] = fma(-ws, v[32 * p], a[q][p]);
            }
        }
    }
    cluster_sync_all();
#pragma unroll
    for (int q = 0; q < CPW; ++q)
#pragma unroll
        for (int p = 0; p < RPL; ++p) {
            const int c = (w + 16 * q) * ncta + rank, i = lane + 32 * p;
            if (c < n && i < n) {
                double rv = (c >= i) ? a[q][p] : 0.0;
                if (c >= i && __ldcg(gflip + i) != 0.0) rv = -rv;
                R0[(int64_t)i * n + c] = rv;
            }
        }
}

// NC (2 or 4) columns per cluster barrier (s2 <= 512): column group pi = (NC pi .. NC pi + NC - 1) -> CTA pi % ncta,
// warp pi / ncta, all NC columns in the registers of ONE warp.  The owner warp factors its first column, applies
// that reflector to its other columns, factors the next one, ... and publishes the NC reflectors together; every
// other warp applies them in turn.  The exchange through L2 (store, cluster barrier, load: the bulk of a step of
// k_geqrf_cluster) is paid once per NC columns.
template <int RPL>
__device__ __forceinline__ double cluster2_reflect(double (&col)[RPL], int j, int lane, double* __restrict__ vout,
                                                   double (&v)[RPL], double* gflip, int* d_info)
{
    double tail2 = 0.0, x1 = 0.0;
#pragma unroll
    for (int p = 0; p < RPL; ++p) {
        const int i = lane + 32 * p;
        if (i > j) tail2 = fma(col[p], col[p], tail2);
        if (i == j) x1 = col[p];
    }
    tail2 = warp_sum(tail2);
    x1 = __shfl_sync(0xffffffffu, x1, j & 31);
    const double nrm = sqrt(tail2 + x1 * x1);
    const double sgn = (x1 < 0.0) ? -1.0 : 1.0;
    const double vj = x1 + sgn * nrm;
    const double vtv = tail2 + vj * vj;
    const double beta = (vtv > 0.0) ? 2.0 / vtv : 0.0;
    if (lane == 0) {
        gflip[j] = (sgn > 0.0) ? 1.0 : 0.0;                   // diagonal becomes -sgn * nrm, the row is negated at the end
        if (!(nrm > 0.0) || !(nrm < 1.0e308)) rqr_set_info(d_info, RQR_INFO_SINGULAR + j + 1);
    }
#pragma unroll
    for (int p = 0; p < RPL; ++p) {
        const int i = lane + 32 * p;
        v[p] = (i > j) ? col[p] : ((i == j) ? vj : 0.0);
        vout[i] = v[p];
        if (i == j) col[p] = -sgn * nrm;
        else if (i > j) col[p] = 0.0;
    }
    return beta;
}

template <int RPL, int NC>
__global__ void __launch_bounds__(RPL * NC <= 32 ? 512 : 256, 1)
k_geqrf_cluster2(double* W, int s2, int n, double* R0, int* d_info, int64_t rows_total, int nb)
{
    __shared__ double vs[NC * 32 * RPL];     // the NC reflectors of this step
    const int ncta = (int)cluster_size(), rank = (int)cluster_rank();
    if (nb > 0) {                            // one level of a TSQR tree, see k_geqrf_cluster
        const int64_t cid = blockIdx.x / ncta;
        const int64_t r0 = cid * rows_total / nb, r1 = (cid + 1) * rows_total / nb;
        W += r0 * n;
        s2 = (int)(r1 - r0);
        R0 += cid * (int64_t)n * n;
        d_info = nullptr;
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int pi = w * ncta + rank;          // my column group: columns NC pi .. NC pi + NC - 1
    double a[NC][RPL];
#pragma unroll
    for (int q = 0; q < NC; ++q)
#pragma unroll
        for (int p = 0; p < RPL; ++p) {
            const int c = NC * pi + q, i = lane + 32 * p;
            a[q][p] = (c < n && i < s2) ? W[(int64_t)i * n + c] : 0.0;
        }
    cluster_sync_all();                      // everyone holds its columns: W is scratch from here on
    double* gv = W;                          // [2 buffers][NC reflectors][32 * RPL]
    double* gbeta = W + 2 * NC * 32 * RPL;   // [2][NC]
    double* gflip = gbeta + 2 * NC;          // [n]
    const int ngroups = (n + NC - 1) / NC;
    for (int jp = 0; jp < ngroups; ++jp) {
        double* buf = gv + (jp & 1) * NC * 32 * RPL;
        if (pi == jp) {                      // the owner warp: factor its NC columns one after the other
            double beta[NC];
#pragma unroll
            for (int q = 0; q < NC; ++q) {
                beta[q] = 0.0;
                if (NC * jp + q < n) {
                    double v[RPL];
                    beta[q] = cluster2_reflect<RPL>(a[q], NC * jp + q, lane, buf + q * 32 * RPL, v, gflip, d_info);
                    double d[NC];
#pragma unroll
                    for (int q2 = q + 1; q2 < NC; ++q2) {
                        double d0 = 0.0, d1 = 0.0;
#pragma unroll
                        for (int p = 0; p < RPL; p += 2) {
                            d0 = fma(v[p], a[q2][p], d0);
                            d1 = fma(v[p + 1], a[q2][p + 1], d1);
                        }
                        d[q2] = d0 + d1;
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                        for (int q2 = q + 1; q2 < NC; ++q2) d[q2] += __shfl_xor_sync(0xffffffffu, d[q2], o);
#pragma unroll
                    for (int q2 = q + 1; q2 < NC; ++q2) {
                        const double ws = beta[q] * d[q2];
#pragma unroll
                        for (int p = 0; p < RPL; ++p) a[q2][p] = fma(-ws, v[p], a[q2][p]);
                    }
                }
            }
            if (lane < NC) {
                double bsel = beta[0];
#pragma unroll
                for (int q = 1; q < NC; ++q) bsel = (lane == q) ? beta[q] : bsel;
                gbeta[(jp & 1) * NC + lane] = bsel;
            }
        }
        cluster_sync_all();
        for (int i = threadIdx.x; i < NC * 32 * RPL; i += blockDim.x) vs[i] = __ldcg(buf + i);
        double beta[NC];
#pragma unroll
        for (int h = 0; h < NC; ++h) beta[h] = __ldcg(gbeta + (jp & 1) * NC + h);
        __syncthreads();
        if (pi > jp && NC * pi < n) {        // groups before jp are finished, jp's own columns were done by the owner
#pragma unroll
            for (int h = 0; h < NC; ++h) {
                if (NC * jp + h >= n) break;
                const double* v = vs + h * 32 * RPL + lane;
                double dot[NC];
#pragma unroll
                for (int q = 0; q < NC; ++q) {
                    double s0 = 0.0, s1_ = 0.0;
#pragma unroll
                    for (int p = 0; p < RPL; p += 2) {
                        s0 = fma(v[32 * p], a[q][p], s0);
                        s1_ = fma(v[32 * (p + 1)], a[q][p + 1], s1_);
                    }
                    dot[q] = s0 + s1_;
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                    for (int q = 0; q < NC; ++q) dot[q] += __shfl_xor_sync(0xffffffffu, dot[q], o);
#pragma unroll
                for (int q = 0; q < NC; ++q) {
                    const double ws = beta[h] * dot[q];       // a padding column (c >= n) is all zero: ws = 0
#pragma unroll
                    for (int p = 0; p < RPL; ++p) a[q][p] = fma(-ws, v[32 * p], a[q][p]);
                }
            }
        }
    }
    cluster_sync_all();
#pragma unroll
    for (int q = 0; q < NC; ++q)
#pragma unroll
        for (int p = 0; p < RPL; ++p) {
            const int c = NC * pi + q, i = lane + 32 * p;
            if (c < n && i < n) {
                double rv = (c >= i) ? a[q][p] : 0.0;
                if (c >= i && __ldcg(gflip + i) != 0.0) rv = -rv;
                R0[(int64_t)i * n + c] = rv;
            }
        }
}

template <class K, class... Args>
static int launch_cluster_grid(K kernel, int nclusters, int ncta, int threads, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(nclusters * ncta);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = ncta;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, kernel, args...) != cudaSuccess) return RQR_ERR_LAUNCH;
    return RQR_OK;
}

template <class K, class... Args>
static int launch_cluster(K kernel, int ncta, int threads, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(ncta);
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = ncta;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, kernel, args...) != cudaSuccess) return RQR_ERR_LAUNCH;
    return RQR_OK;
}

extern "C" int rqr_small_geqrf(double* W, int s2, int n, double* R0, int* d_info, void* stream)
{
    if (!W) return -1;
    if (s2 < 1 || s2 > RQR_MAX_S2) return -2;
    if (n < 2 || n > RQR_MAX_N || n > s2) return -3;
    if (!R0) return -4;
    cudaStream_t st = (cudaStream_t)stream;
    const int rpl = (s2 + 31) / 32, cpw = (n + 31) / 32;
    if (s2 <= 128 && n <= 64) {
        // four columns per warp: 8 warps cover n <= 32, 16 warps n <= 64 (k_geqrf_g8, eight columns per warp, remains
        // the block kernel of the TSQR tree)
        // n <= 32: four columns per warp, ceil(n / 4) warps (measured A/B in one run: 64 x 32 26.7 against 31.4 us,
        // 32 x 16 15.4 against 17.9); above, eight columns per warp on 8 warps (128 x 64: 55.4 against 57.4 us
        // with 16 warps: twice the warps reload the reflector from shared memory)
        if (RQR_GEQRF_G8X && n <= 32) k_geqrf_g8x<<<1, 32 * ((n + 3) / 4), 0, st>>>(W, s2, n, R0, d_info);
        else                          k_geqrf_g8<<<1, 256, 0, st>>>(W, s2, n, R0, d_info);
        RQR_LAUNCH_CHECK();
        return RQR_OK;
    }
#define GEQRF_CASE(R, C)                                                              \
    if (rpl <= R && cpw <= C) {                                                       \
        k_geqrf_reg<R, C><<<1, 1024, 0, st>>>(W, s2, n, R0, d_info);                   \
        RQR_LAUNCH_CHECK();                                                           \
        return RQR_OK;                                                                \
    }
    GEQRF_CASE(8, 1) GEQRF_CASE(8, 2) GEQRF_CASE(16, 1)
#undef GEQRF_CASE
    // n > 64: the register tile is spread over a cluster of 4 or 8 CTAs.  W's storage doubles as
    // the exchange buffer (2 * 32 * RPL + 2 + n doubles), which it always has room for here.
    if ((int64_t)s2 * n >= 2 * 32 * rpl + 2 + n) {
        if (rpl <= 16) {
            const int ncta = n <= 128 ? 4 : 8;                     // 16 warps x 2 columns per CTA
            // NC columns per cluster barrier (k_geqrf_cluster2); its exchange area is NC times as large.
            // 512 x 256: 0.56 ms (one column per barrier) -> 0.45 (two) -> 0.41 ms (four); 256 x 128: 0.23 -> 0.15 ms
            if ((int64_t)s2 * n >= 8 * 32 * rpl + 8 + n) {
                if (rpl <= 8) return launch_cluster(k_geqrf_cluster2<8, 4>, ncta, 256, st, W, s2, n, R0, d_info, (int64_t)0, 0);
                return launch_cluster(k_geqrf_cluster2<16, 4>, ncta, 256, st, W, s2, n, R0, d_info, (int64_t)0, 0);
            }
            if ((int64_t)s2 * n >= 4 * 32 * rpl + 4 + n) {
                if (rpl <= 8) return launch_cluster(k_geqrf_cluster2<8, 2>, ncta, 512, st, W, s2, n, R0, d_info, (int64_t)0, 0);
                return launch_cluster(k_geqrf_cluster2<16, 2>, ncta, 512, st, W, s2, n, R0, d_info, (int64_t)0, 0);
            }
            if (rpl <= 8) return launch_cluster(k_geqrf_cluster<8, 2>, ncta, 512, st, W, s2, n, R0, d_info, (int64_t)0, 0);
            return launch_cluster(k_geqrf_cluster<16, 2>, ncta, 512, st, W, s2, n, R0, d_info, (int64_t)0, 0);
        }
        if (n > 64 && n <= 128 && (int64_t)s2 * n >= 4 * 32 * 32 + 4 + n)   // tall sketches of the paper's grid (s2 <= 1024):
            return launch_cluster(k_geqrf_cluster2<32, 2>, 8, 256, st, W, s2, n, R0, d_info, (int64_t)0, 0);   // 64 pairs, 8 x 8 warps
        if (n <= 128)
            return launch_cluster(k_geqrf_cluster<32, 1>, n <= 64 ? 4 : 8, 512, st, W, s2, n, R0, d_info, (int64_t)0, 0);
        if (rpl <= 32 && (int64_t)s2 * n >= 4 * 32 * 32 + 4 + n) {
            // 512 < s2 <= 1024 with 128 < n <= 256: 128 column pairs need 16 CTAs of 8 warps (64 registers of tile per
            // column): a non-portable cluster size; if the device refuses it the global-memory kernel below runs
            RQR_ONCE_PER_DEVICE({
                cudaFuncSetAttribute(k_geqrf_cluster2<32, 2>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            });
            if (launch_cluster(k_geqrf_cluster2<32, 2>, 16, 256, st, W, s2, n, R0, d_info, (int64_t)0, 0) == RQR_OK)
                return RQR_OK;
            (void)cudaGetLastError();
        }
    }
    k_geqrf_gmem<<<1, 1024, 0, st>>>(W, s2, n, R0, d_info);
    RQR_LAUNCH_CHECK();
    return RQR_OK;
}

// TSQR tree for 64 < n <= 256 (the single-CountSketch variant N3 at the paper's larger widths): blocks of at most
// 1024 (n <= 128) or 512 rows go through the cluster kernel, one cluster per block, level by level; the stacked R
// factors ping-pong between `scratch` and A itself, which is DESTROYED.  scratch: ceil(rows / block rows) n^2 doubles.
int rqr_tsqr_r_wide_dev(double* A, int64_t rows, int n, double* R, double* scratch, int* d_info, cudaStream_t st)
{
    const int BR = n <= 128 ? 1024 : 512;
    double* in = A;
    double* out = scratch;
    int64_t rows_in = rows;
    for (;;) {
        const int64_t nb = (rows_in + BR - 1) / BR;
        if (nb <= 1) return rqr_small_geqrf(in, (int)rows_in, n, R, d_info, st);
        int rc;
        if (n <= 128) rc = launch_cluster_grid(k_geqrf_cluster<32, 1>, (int)nb, 8, 512, st, in, 0, n, out, (int*)nullptr, rows_in, (int)nb);
        else          rc = launch_cluster_grid(k_geqrf_cluster2<16, 4>, (int)nb, 8, 256, st, in, 0, n, out, (int*)nullptr, rows_in, (int)nb);
        if (rc != RQR_OK) return rc;
        double* t = in; in = out; out = t;
        rows_in = nb * n;
    }
}

// =========================================================================================
// A5: upper Cholesky factor  G + shift I = R1^T R1   (Alg. 2 step 2)
// =========================================================================================
// Blocked right-looking Cholesky for n <= 64 on the FP64 tensor path: 8 x 8 blocks, the matrix in shared memory.
// Per block step K: (1) warp 0 factors the diagonal block in registers (every lane the same arithmetic: no
// shuffles; r = d rsqrt(d)) and inverts it, (2) the row panel R[K,J] = inv(R_KK)^T A[K,J] and (3) the trailing
// update A[I,J] -= R[K,I]^T R[K,J] (K < I <= J) are mma.sync m8n8k4 products spread over the 8 warps.
// 3 barriers per 8 columns instead of 1 per column: 31 -> 14 us at n = 64.  Pivots are mathematically the same
// as in the unblocked algorithm, so the first failing pivot index is the same.
__device__ __forceinline__ void cholb_dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// Where the two-level driver parks inv(R_KK) of the first half (16 blocks of 8 x 8): in the strictly lower
// triangle of R1's leading 128 x 128 block, which is zero in the result and re-zeroed by k_chol2_syrk:
// block (K + 1, K) for K < 15, block (15, 0) for K = 15.
__device__ __forceinline__ double* chol2_tslot(double* base, int ld, int K)
{
    return (K < 15) ? base + (int64_t)(8 * (K + 1)) * ld + 8 * K : base + (int64_t)(8 * 15) * ld;
}

// threads of k_chol_blocked: 8 warps up to n = 48 (at most 15 trailing blocks), 16 warps above (A/B: RQR_CHOL_WIDE)
#ifndef RQR_CHOL_WIDE
#define RQR_CHOL_WIDE 1
#endif
#define RQR_CHOL_THREADS(nn) ((RQR_CHOL_WIDE && (nn) > 48) ? 512 : 256)
template <int THREADS>
__global__ void __launch_bounds__(THREADS, 1)
k_chol_blocked(const double* G, int ldg, int n, double shift_h, const double* __restrict__ d_shift,
               double* R1, int ldr, int* d_info, int info_off, const double* __restrict__ Rprev,
               double* __restrict__ Rprod, double* Tsave, int ldt, double* zero_src, int zero_cols)
{
    // G, R1: n x n with leading dimensions ldg, ldr (the two-level driver for n > 128 factors sub-blocks in place).
    // Tsave != NULL: inv(R_KK) of block K is also stored (8 x 8, leading dimension ldt) at Tsave + T-slot(K), see
    // chol2_tslot.  zero_src != NULL: the scratch area that held the input (== G; n rows x zero_cols columns, leading
    // dimension ldg) is zeroed once the input is in shared memory.
    extern __shared__ double dyn[];
    const int NB = (n + 7) >> 3, np = 8 * NB;
    const int LD = np + 8 + (np & 8);         // row stride = 8 mod 16 doubles: the 128-bit C-fragment accesses are conflict free
    double* A = dyn;                          // np x LD, padded with the identity beyond n
    __shared__ double Ts[8][9];               // inverse of the current diagonal block
    __shared__ int fail_s;
    const double shift = shift_h + (d_shift ? *d_shift : 0.0);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x, nwarps = nthr >> 5;             // 8 or 16 warps (CHOL_THREADS_OF)
    for (int e = tid; e < np * np; e += nthr) {
        const int i = e / np, c = e - i * np;
        double v = (i == c) ? 1.0 : 0.0;
        if (i < n && c < n) v = G[(int64_t)i * ldg + c] + ((i == c) ? shift : 0.0);
        A[i * LD + c] = v;
    }
    if (zero_src != nullptr) {
        __syncthreads();                                  // every thread has read its part of the scratch input
        for (int e = tid; e < n * zero_cols; e += nthr) {
            const int i = e / zero_cols, c = e - i * zero_cols;
            zero_src[(int64_t)i * ldg + c] = 0.0;
        }
    }
    for (int e = tid; e < n * n; e += nthr) {              // exact zeros below the diagonal
        const int i = e / n, c = e - i * n;
        if (c < i) R1[(int64_t)i * ldr + c] = 0.0;
    }
    if (tid == 0) fail_s = 0;
    if (tid < 64) Ts[tid >> 3][tid & 7] = 0.0;            // the strict lower triangle of T stays zero
    __syncthreads();
    const int r = lane >> 2, q = lane & 3;
    for (int K = 0; K < NB; ++K) {
        if (warp == 0) {
            // (1) diagonal block: unblocked Cholesky + inverse, identical in every lane
            double d[8][8];
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int c = i; c < 8; ++c) d[i][c] = A[(8 * K + i) * LD + 8 * K + c];
            double rinv[8];
            int fail = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const double dj = d[j][j];
                if (!fail && (!(dj > 0.0) || !(dj < 1.0e308))) fail = 8 * K + j + 1;
                rinv[j] = rsqrt(dj);
                d[j][j] = dj * rinv[j];
#pragma unroll
                for (int c = j + 1; c < 8; ++c) d[j][c] *= rinv[j];
#pragma unroll
                for (int i = j + 1; i < 8; ++i)
#pragma unroll
                    for (int c = i; c < 8; ++c) d[i][c] = fma(-d[j][i], d[j][c], d[i][c]);
            }
            // T = inv(R_KK), upper: column c by back substitution
            double t[8][8];
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                t[c][c] = rinv[c];
#pragma unroll
                for (int i = c - 1; i >= 0; --i) {
                    double sacc = 0.0;
#pragma unroll
                    for (int k = i + 1; k <= c; ++k) sacc = fma(d[i][k], t[k][c], sacc);
                    t[i][c] = -sacc * rinv[i];
                }
            }
            // publish R_KK and T: every lane stores the same value to the same address (one broadcast store each)
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    if (c >= i) {
                        A[(8 * K + i) * LD + 8 * K + c] = d[i][c];
                        Ts[i][c] = t[i][c];
                    }
                }
            if (lane == 0 && fail) fail_s = fail;
        }
        __syncthreads();
        if (fail_s) break;
        if (warp == nwarps - 1) {                                      // R_KK to global
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int i = (lane + 32 * h) >> 3, c = (lane + 32 * h) & 7;
                if (c >= i && 8 * K + c < n) R1[(int64_t)(8 * K + i) * ldr + 8 * K + c] = A[(8 * K + i) * LD + 8 * K + c];
                if (Tsave != nullptr) chol2_tslot(Tsave, ldt, K)[i * ldt + c] = Ts[i][c];
            }
        }
        // (2) row panel: R[K,J] = T^T A[K,J], J > K
        for (int J = K + 1 + warp; J < NB; J += nwarps) {
            double c0 = 0.0, c1 = 0.0;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const double a = Ts[4 * h + q][r];                                    // T^T[r][4h+q]
                const double b = A[(8 * K + 4 * h + q) * LD + 8 * J + r];       // A[K,J][4h+q][r]
                cholb_dmma(c0, c1, a, b);
            }
            __syncwarp();
            *reinterpret_cast<double2*>(A + (8 * K + r) * LD + 8 * J + 2 * q) = make_double2(c0, c1);
            const int row = 8 * K + r, col = 8 * J + 2 * q;
            if (row < n && col < n) R1[(int64_t)row * ldr + col] = c0;
            if (row < n && col + 1 < n) R1[(int64_t)row * ldr + col + 1] = c1;
        }
        __syncthreads();
        // (3) trailing update: A[I,J] -= R[K,I]^T R[K,J], K < I <= J
        const int nt = NB - K - 1;
        for (int pidx = warp; pidx < nt * (nt + 1) / 2; pidx += nwarps) {
            int I = 0, rem = pidx;
            while (rem >= nt - I) { rem -= nt - I; ++I; }
            const int J = K + 1 + I + rem;
            I += K + 1;
            double2 c = *reinterpret_cast<const double2*>(A + (8 * I + r) * LD + 8 * J + 2 * q);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const double a = -A[(8 * K + 4 * h + q) * LD + 8 * I + r];      // -R[K,I]^T[r][4h+q]
                const double b = A[(8 * K + 4 * h + q) * LD + 8 * J + r];       //  R[K,J][4h+q][r]
                cholb_dmma(c.x, c.y, a, b);
            }
            *reinterpret_cast<double2*>(A + (8 * I + r) * LD + 8 * J + 2 * q) = c;
        }
        __syncthreads();
    }
    if (fail_s) {
        if (tid == 0) rqr_set_info(d_info, RQR_INFO_NOT_SPD + info_off + fail_s);
        return;
    }
    if (Rprod != nullptr) {
        // fused A7 of the one-shot drivers: Rprod = R1 Rprev (upper x upper, Alg. 3 step 3 PAPER.md:206).  R1 is the
        // upper triangle of A; Rprev^T is staged into the (now free) strict lower triangle, its diagonal into the
        // first pad column; the product runs block-wise on mma.sync like the trailing update.
        for (int e = tid; e < n * n; e += nthr) {
            const int k = e / n, c = e - k * n;
            if (k < c) A[c * LD + k] = __ldg(Rprev + e);
            else if (k == c) A[k * LD + np] = __ldg(Rprev + e);
            else if ((c >> 3) < (k >> 3)) Rprod[e] = 0.0;
        }
        __syncthreads();
        for (int blk = warp; blk < NB * (NB + 1) / 2; blk += nwarps) {
            int I = 0, rem = blk;
            while (rem >= NB - I) { rem -= NB - I; ++I; }
            const int J = I + rem;
            const int row = 8 * I + r, col = 8 * J + r;
            double c0 = 0.0, c1 = 0.0;
            for (int K = I; K <= J; ++K) {
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int kk = 8 * K + 4 * h + q;
                    const double a = (kk >= row) ? A[row * LD + kk] : 0.0;
                    const double b = (kk < col) ? A[col * LD + kk] : ((kk == col) ? A[kk * LD + np] : 0.0);
                    cholb_dmma(c0, c1, a, b);
                }
            }
            const int oc = 8 * J + 2 * q;
            if (row < n && oc < n) Rprod[(int64_t)row * n + oc] = (oc >= row) ? c0 : 0.0;
            if (row < n && oc + 1 < n) Rprod[(int64_t)row * n + oc + 1] = (oc + 1 >= row) ? c1 : 0.0;
        }
    }
}

// ---- two-level Cholesky for 128 < n <= 256 on the blocked kernel: with h = 128 and G = [G11 G12; G12^T G22]
//   R11 = chol(G11)                     k_chol_blocked, keeps inv(R_KK) of its 16 diagonal blocks
//   R12 = R11^-T G12                    k_chol2_trsm: one warp per 8 columns, block forward substitution
//   S   = G22 - R12^T R12               k_chol2_syrk: one warp per 8 x 8 block of the upper triangle
//   R22 = chol(S)                       k_chol_blocked again (pivot indices offset by h)
// Scratch is the part of R1 that is zero in the result: the T blocks in the strict lower triangle of the
// leading block (chol2_tslot), S in the lower-left block R1[h:n, 0:h]; both are zeroed again on the way.
// k_chol2_trsm computes the TRANSPOSED slice X^T = (B^T[K] - sum_{I<K} X^T[I] R11[I,K]) inv(R_KK): the C fragment
// of X^T[I] is the A operand of the later products with the k-permuted B fragments (k slot q <-> row 2q + s),
// so the 16-step chain never leaves the registers.
__global__ void __launch_bounds__(32)
k_chol2_trsm(const double* __restrict__ G, int n, double* R1)
{
    constexpr int H = 128, NBH = 16;
    const int lane = threadIdx.x, r = lane >> 2, q = lane & 3;
    const int col = H + 8 * blockIdx.x + r;                   // my column of G12 / R12 (row r of the slice^T)
    const bool colok = col < n;
    double xs[NBH][2];
#pragma unroll
    for (int K = 0; K < NBH; ++K) {
        // acc = B^T[K]: C fragment (row r, columns 2q, 2q+1) = G[8K + 2q + s][col]
        double a0 = colok ? G[(int64_t)(8 * K + 2 * q) * n + col] : 0.0;
        double a1 = colok ? G[(int64_t)(8 * K + 2 * q + 1) * n + col] : 0.0;
        double b0 = 0.0, b1 = 0.0;                            // second accumulator: two independent chains
#pragma unroll
        for (int I = 0; I < K; ++I) {
            const double* Rb = R1 + (int64_t)(8 * I + 2 * q) * n + 8 * K + r;     // R11[I,K][2q + s][r]
            cholb_dmma(a0, a1, -xs[I][0], Rb[0]);
            cholb_dmma(b0, b1, -xs[I][1], Rb[n]);
        }
        a0 += b0; a1 += b1;
        const double* T = chol2_tslot(R1, n, K);
        double y0 = 0.0, y1 = 0.0;
        cholb_dmma(y0, y1, a0, T[(2 * q) * n + r]);
        cholb_dmma(y0, y1, a1, T[(2 * q + 1) * n + r]);
        xs[K][0] = y0; xs[K][1] = y1;
        if (colok) {
            R1[(int64_t)(8 * K + 2 * q) * n + col] = y0;
            R1[(int64_t)(8 * K + 2 * q + 1) * n + col] = y1;
        }
    }
}

__global__ void __launch_bounds__(256)
k_chol2_syrk(const double* __restrict__ G, int n, double shift_h, const double* __restrict__ d_shift, double* R1)
{
    constexpr int H = 128, NBH = 16;
    const double shift = shift_h + (d_shift ? *d_shift : 0.0);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, r = lane >> 2, q = lane & 3;
    const int n2 = n - H, NB2 = (n2 + 7) >> 3;
    if (blockIdx.x == 0) {                                    // the T blocks are not needed any more
        for (int e = threadIdx.x; e < NBH * 64; e += 256) {
            const int K = e >> 6, i = (e >> 3) & 7, c = e & 7;
            chol2_tslot(R1, n, K)[i * n + c] = 0.0;
        }
    }
    const int blk = blockIdx.x * 8 + warp;
    if (blk >= NB2 * (NB2 + 1) / 2) return;
    int I = 0, rem = blk;
    while (rem >= NB2 - I) { rem -= NB2 - I; ++I; }
    const int J = I + rem;
    const int row = 8 * I + r, c0 = 8 * J + 2 * q;            // inside the trailing block
    double s0 = 0.0, s1 = 0.0, t0 = 0.0, t1 = 0.0;
    if (row < n2 && c0 < n2) s0 = G[(int64_t)(H + row) * n + H + c0] + ((row == c0) ? shift : 0.0);
    if (row < n2 && c0 + 1 < n2) s1 = G[(int64_t)(H + row) * n + H + c0 + 1] + ((row == c0 + 1) ? shift : 0.0);
    const bool aok = H + 8 * I + r < n, bok = H + 8 * J + r < n;
#pragma unroll 4
    for (int k = 0; k < H; k += 8) {
        const double* Ra = R1 + (int64_t)(k + q) * n + H;     // R12[k + q][.]
        const double a0 = aok ? -Ra[8 * I + r] : 0.0, a1 = aok ? -Ra[4 * n + 8 * I + r] : 0.0;
        const double b0 = bok ? Ra[8 * J + r] : 0.0, b1 = bok ? Ra[4 * n + 8 * J + r] : 0.0;
        cholb_dmma(s0, s1, a0, b0);
        cholb_dmma(t0, t1, a1, b1);
    }
    double* S = R1 + (int64_t)H * n;                          // scratch: R1[h:n, 0:h], leading dimension n
    if (row < n2 && c0 < n2) S[(int64_t)row * n + c0] = s0 + t0;
    if (row < n2 && c0 + 1 < n2) S[(int64_t)row * n + c0 + 1] = s1 + t1;
}

int rqr_chol_dev(const double* G, int n, double shift, const double* d_shift, double* R1,
                 int* d_info, cudaStream_t st, const double* Rprev, double* Rprod);

extern "C" int rqr_chol(const double* G, int n, double shift, double* R1, int* d_info, void* stream)
{
    return rqr_chol_dev(G, n, shift, nullptr, R1, d_info, (cudaStream_t)stream, nullptr, nullptr);
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

// Rprod != NULL: also Rprod = R1 Rprev (the one-shot drivers' A7), fused into the single-CTA blocked kernel
// for n <= 128, a separate k_triu_mul launch above that (two-level factorization, see k_chol2_trsm).
int rqr_chol_dev(const double* G, int n, double shift, const double* d_shift, double* R1,
                 int* d_info, cudaStream_t st, const double* Rprev, double* Rprod)
{
    if (!G) return -1;
    if (n < 2 || n > RQR_MAX_N) return -2;
    if (!R1) return -4;
    if (G == R1) return -4;
    RQR_ONCE_PER_DEVICE({
        cudaFuncSetAttribute(k_chol_blocked<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, 144 * 1024);
        cudaFuncSetAttribute(k_chol_blocked<512>, cudaFuncAttributeMaxDynamicSharedMemorySize, 144 * 1024);
    });
    auto smem_of = [](int nn) { const int np = (nn + 7) & ~7; return (size_t)np * (np + 8 + (np & 8)) * sizeof(double); };
#define CHOL_LAUNCH(nn, ...)                                                                          \
    do {                                                                                              \
        if (RQR_CHOL_THREADS(nn) == 512) k_chol_blocked<512><<<1, 512, smem_of(nn), st>>>(__VA_ARGS__); \
        else                             k_chol_blocked<256><<<1, 256, smem_of(nn), st>>>(__VA_ARGS__); \
    } while (0)
    if (n <= 128) {
        CHOL_LAUNCH(n, G, n, n, shift, d_shift, R1, n, d_info, 0, Rprev, Rprod,
                                                   nullptr, 0, nullptr, 0);
    } else {
        // two-level (see k_chol2_trsm): 0.51 ms -> 0.12 ms at n = 256
        const int h = 128, n2 = n - h, nb2 = (n2 + 7) / 8;
        double* S = R1 + (int64_t)h * n;
        CHOL_LAUNCH(h, G, n, h, shift, d_shift, R1, n, d_info, 0, nullptr, nullptr,
                                                   R1, n, nullptr, 0);
        RQR_LAUNCH_CHECK();
        k_chol2_trsm<<<nb2, 32, 0, st>>>(G, n, R1);
        RQR_LAUNCH_CHECK();
        k_chol2_syrk<<<(nb2 * (nb2 + 1) / 2 + 7) / 8, 256, 0, st>>>(G, n, shift, d_shift, R1);
        RQR_LAUNCH_CHECK();
        CHOL_LAUNCH(n2, S, n, n2, 0.0, nullptr, R1 + (int64_t)h * n + h, n, d_info, h,
                                                    nullptr, nullptr, nullptr, 0, S, h);
        RQR_LAUNCH_CHECK();
        if (!Rprod) return RQR_OK;
        return rqr_triu_mul(R1, Rprev, n, Rprod, st);
    }
    RQR_LAUNCH_CHECK();
    return RQR_OK;
#undef CHOL_LAUNCH
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
