// rqr_api.cu -- workspace query and the one-shot drivers (Alg. 3 rand_cholQR and the
// comparators on the same kernels).  Each driver is a fixed sequence of the step entry points
// on one stream: no host synchronisation, CUDA-graph capturable.
#include "rqr_common.cuh"

int rqr_chol_dev(const double* G, int n, double shift, const double* d_shift, double* R1,
                 int* d_info, cudaStream_t st, const double* Rprev, double* Rprod);
int rqr_scholqr3_shift(const double* G, int n, int64_t m, double* d_out, cudaStream_t st);
int rqr_tsqr_r_dev(const double* A, int64_t rows, int n, double* R, double* scratch, int* d_info, cudaStream_t st);
int rqr_tsqr_r_wide_dev(double* A, int64_t rows, int n, double* R, double* scratch, int* d_info, cudaStream_t st);

extern "C" const char* rqr_version(void) { return "rqr 0.1 (sm_100a)"; }

extern "C" size_t rqr_workspace_bytes(int64_t m, int n, int64_t s1, int s2, int variant)
{
    if (m < 1 || n < 2 || n > RQR_MAX_N || s1 < 1 || s2 < 1 || s2 > RQR_MAX_S2) return 0;
    return rqr_layout(m, n, s1, (variant & RQR_S2_RADEMACHER) != 0).total;
}

#define RQR_TRY(call)                 \
    do {                              \
        int rc__ = (call);            \
        if (rc__ != RQR_OK) return rc__; \
    } while (0)

static inline double* small_mat(void* work, const RqrLayout& L, int n, int which)
{
    return (double*)((char*)work + L.A_small) + (size_t)which * n * n;
}

static int check_common(const double* V, int64_t m, int n, double* Q, double* R, void* work)
{
    if (!V) return -1;
    if (m < 1 || m >= ((int64_t)1 << 31)) return -2;
    if (n < 2 || n > RQR_MAX_N || n > m) return -3;
    if (!Q || !R || !work) return -100;
    return RQR_OK;
}

// cholQR of V R0^-1: shared tail of every driver.  A4 with R0 writes V1 into Q, A5 (which also forms
// Rprod = R1 R0, the drivers' A7, when Rprod != NULL), A6 in place.
static int tail_cholqr(const double* V, int64_t m, int n, const double* R0, double* Q, double* R1,
                       double* G, void* work, int* d_info, int recompute, cudaStream_t st, double* Rprod)
{
    if (recompute && R0 && n <= 64) {     // n > 64: A4 is FP64-bound either way and V1 is always stored
        RQR_TRY(rqr_trsm_gram(V, m, n, n, R0, G, nullptr, n, work, st));
        RQR_TRY(rqr_chol_dev(G, n, 0.0, nullptr, R1, d_info, st, R0, Rprod));
        RQR_TRY(rqr_apply(V, m, n, n, R0, R1, Q, n, work, st));
    } else {
        RQR_TRY(rqr_trsm_gram(V, m, n, n, R0, G, Q, n, work, st));
        RQR_TRY(rqr_chol_dev(G, n, 0.0, nullptr, R1, d_info, st, R0, Rprod));
        RQR_TRY(rqr_apply(Q, m, n, n, nullptr, R1, Q, n, work, st));
    }
    return RQR_OK;
}

extern "C" int rqr_rand_cholqr(const double* V, int64_t m, int n, int64_t s1, int s2, uint64_t seed,
                               double* Q, double* R, void* work, int* d_info, int variant,
                               int flags, void* stream)
{
    int rc = check_common(V, m, n, Q, R, work);
    if (rc == -100) return !Q ? -7 : (!R ? -8 : -9);
    if (rc != RQR_OK) return rc;
    if (s1 < 1 || s1 >= ((int64_t)1 << 31) || s1 > m) return -4;
    if (s2 < n || s2 > s1 || s2 > RQR_MAX_S2) return -5;      // eq. (20)
    const int rad = variant & RQR_S2_RADEMACHER;                 // N4: Count-Rademacher multisketch
    if ((variant & ~RQR_S2_RADEMACHER) != RQR_VARIANT_SORTED && (variant & ~RQR_S2_RADEMACHER) != RQR_VARIANT_SCATTER)
        return -11;
    cudaStream_t st = (cudaStream_t)stream;
    RqrLayout L = rqr_layout(m, n, s1, rad != 0);
    double* R0 = small_mat(work, L, n, RQR_SM_R0);
    double* R1 = small_mat(work, L, n, RQR_SM_R1);
    double* G = small_mat(work, L, n, RQR_SM_G);
    double* W1 = (double*)((char*)work + L.F_W1);
    double* W = (double*)((char*)work + L.F_W);
    if (d_info && cudaMemsetAsync(d_info, 0, sizeof(int), st) != cudaSuccess) return RQR_ERR_LAUNCH;
    if (!(flags & RQR_FLAG_PREPARED))
        RQR_TRY(rqr_sketch_prepare(m, n, 0, s1, s2, seed, variant, work, st));
    // Alg. 1 randQR: W = S2 S1 V; R0 = hhqr(W).R; V1 = V R0^-1
    RQR_TRY(rqr_countsketch(V, m, n, n, 0, s1, seed, W1, work, variant, RQR_FLAG_PREPARED, st));
    RQR_TRY(rqr_gauss_sketch(W1, s1, n, s2, seed, W, work, RQR_FLAG_PREPARED | rad, st));
    RQR_TRY(rqr_small_geqrf(W, s2, n, R0, d_info, st));
    // Alg. 2 cholQR of V1; Alg. 3 step 3
    RQR_TRY(tail_cholqr(V, m, n, R0, Q, R1, G, work, d_info, flags & RQR_FLAG_RECOMPUTE_V1, st, R));
    return RQR_OK;
}

extern "C" int rqr_rand_cholqr_batched(const double* V, int64_t m, int n, int batch, int64_t strideV, int64_t s1,
                                       int s2, uint64_t seed, double* Q, int64_t strideQ, double* R, void* work,
                                       int* d_info, int variant, int flags, void* stream)
{
    if (batch < 1) return -4;
    if (strideV < m * n || strideQ < m * n) return -5;
    if (!V || !Q || !R) return !V ? -1 : (!Q ? -9 : -11);
    if (!(flags & RQR_FLAG_PREPARED)) {
        if (m < 1 || n < 2 || n > RQR_MAX_N || !work) return -2;
        RQR_TRY(rqr_sketch_prepare(m, n, 0, s1, s2, seed, variant, work, (cudaStream_t)stream));
    }
    for (int b = 0; b < batch; ++b)
        RQR_TRY(rqr_rand_cholqr(V + (int64_t)b * strideV, m, n, s1, s2, seed, Q + (int64_t)b * strideQ,
                                R + (int64_t)b * n * n, work, d_info ? d_info + b : nullptr, variant,
                                flags | RQR_FLAG_PREPARED, stream));
    return RQR_OK;
}

extern "C" int rqr_gauss_randcholqr(const double* V, int64_t m, int n, int s, uint64_t seed,
                                    double* Q, double* R, void* work, int* d_info, void* stream)
{
    int rc = check_common(V, m, n, Q, R, work);
    if (rc == -100) return !Q ? -6 : (!R ? -7 : -8);
    if (rc != RQR_OK) return rc;
    if (s < n || s > RQR_MAX_S2 || s > m) return -4;
    cudaStream_t st = (cudaStream_t)stream;
    RqrLayout L = rqr_layout(m, n, n);
    double* R0 = small_mat(work, L, n, RQR_SM_R0);
    double* R1 = small_mat(work, L, n, RQR_SM_R1);
    double* G = small_mat(work, L, n, RQR_SM_G);
    double* W = (double*)((char*)work + L.F_W);        // s x n, s <= RQR_MAX_S2
    if (d_info && cudaMemsetAsync(d_info, 0, sizeof(int), st) != cudaSuccess) return RQR_ERR_LAUNCH;
    RQR_TRY(rqr_dense_gauss_sketch(V, m, n, n, 0, m, s, seed, W, work, st));
    RQR_TRY(rqr_small_geqrf(W, s, n, R0, d_info, st));
    RQR_TRY(tail_cholqr(V, m, n, R0, Q, R1, G, work, d_info, 0, st, R));
    return RQR_OK;
}

// rows the TSQR scratch (region A of the workspace) can take
static int64_t tsqr_max_rows(int n) { return (int64_t)128 * rqr_gram_partial_cap(n) * 2 / 3; }

extern "C" int rqr_tsqr_r(const double* A, int64_t rows, int n, double* R, void* work, int* d_info, void* stream)
{
    if (!A) return -1;
    if (n < 2 || n > 64) return -3;
    if (rows < n || rows > tsqr_max_rows(n)) return -2;
    if (!R) return -4;
    if (!work) return -5;
    return rqr_tsqr_r_dev(A, rows, n, R, (double*)((char*)work + 256), d_info, (cudaStream_t)stream);
}

// rand_cholQR with ONE CountSketch (the paper's "Sparse" rows, Tables 1-3): R0 is the R
// factor of the Householder QR of the s1 x n sketch W1 itself -- the O(n^2)-row factorization that the second,
// Gaussian, sketch of the multisketch avoids.  Here it is a TSQR tree (n <= 64).
extern "C" int rqr_count_randcholqr(const double* V, int64_t m, int n, int64_t s1, uint64_t seed, double* Q,
                                    double* R, void* work, int* d_info, int variant, int flags, void* stream)
{
    int rc = check_common(V, m, n, Q, R, work);
    if (rc == -100) return !Q ? -6 : (!R ? -7 : -8);
    if (rc != RQR_OK) return rc;
    // n <= 64: tree of 128-row register-resident blocks; n > 64: blocks of 1024 / 512 rows in the cluster kernel
    const int64_t max_rows = n <= 64 ? tsqr_max_rows(n) : (int64_t)(n <= 128 ? 1024 : 512) * rqr_gram_partial_cap(n);
    if (s1 < n || s1 >= ((int64_t)1 << 31) || s1 > m || s1 > max_rows) return -4;
    if (variant != RQR_VARIANT_SORTED && variant != RQR_VARIANT_SCATTER) return -10;
    cudaStream_t st = (cudaStream_t)stream;
    RqrLayout L = rqr_layout(m, n, s1);
    double* R0 = small_mat(work, L, n, RQR_SM_R0);
    double* R1 = small_mat(work, L, n, RQR_SM_R1);
    double* G = small_mat(work, L, n, RQR_SM_G);
    double* W1 = (double*)((char*)work + L.F_W1);
    if (d_info && cudaMemsetAsync(d_info, 0, sizeof(int), st) != cudaSuccess) return RQR_ERR_LAUNCH;
    RQR_TRY(rqr_countsketch(V, m, n, n, 0, s1, seed, W1, work, variant, flags & RQR_FLAG_PREPARED, st));
    if (n <= 64) RQR_TRY(rqr_tsqr_r_dev(W1, s1, n, R0, (double*)((char*)work + 256), d_info, st));
    else RQR_TRY(rqr_tsqr_r_wide_dev(W1, s1, n, R0, (double*)((char*)work + 256), d_info, st));
    RQR_TRY(tail_cholqr(V, m, n, R0, Q, R1, G, work, d_info, flags & RQR_FLAG_RECOMPUTE_V1, st, R));
    return RQR_OK;
}

extern "C" int rqr_cholqr2(const double* V, int64_t m, int n, double* Q, double* R, void* work,
                           int* d_info, void* stream)
{
    int rc = check_common(V, m, n, Q, R, work);
    if (rc == -100) return !Q ? -4 : (!R ? -5 : -6);
    if (rc != RQR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    RqrLayout L = rqr_layout(m, n, n);
    double* RA = small_mat(work, L, n, RQR_SM_RA);
    double* RB = small_mat(work, L, n, RQR_SM_RB);
    double* G = small_mat(work, L, n, RQR_SM_G);
    if (d_info && cudaMemsetAsync(d_info, 0, sizeof(int), st) != cudaSuccess) return RQR_ERR_LAUNCH;
    // Alg. 4 step 1: cholQR(V): G = V^T V, RA = chol(G); Q0 = V RA^-1 is formed inside step 2's A4
    RQR_TRY(rqr_trsm_gram(V, m, n, n, nullptr, G, nullptr, n, work, st));
    RQR_TRY(rqr_chol_dev(G, n, 0.0, nullptr, RA, d_info, st, nullptr, nullptr));
    // step 2: cholQR(Q0); R = RB RA
    RQR_TRY(tail_cholqr(V, m, n, RA, Q, RB, G, work, d_info, 0, st, R));
    return RQR_OK;
}

extern "C" int rqr_scholqr3(const double* V, int64_t m, int n, double* Q, double* R, void* work,
                            int* d_info, void* stream)
{
    int rc = check_common(V, m, n, Q, R, work);
    if (rc == -100) return !Q ? -4 : (!R ? -5 : -6);
    if (rc != RQR_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    RqrLayout L = rqr_layout(m, n, n);
    double* RA = small_mat(work, L, n, RQR_SM_RA);
    double* RB = small_mat(work, L, n, RQR_SM_RB);
    double* RC = small_mat(work, L, n, RQR_SM_RC);
    double* T = small_mat(work, L, n, RQR_SM_R0);
    double* G = small_mat(work, L, n, RQR_SM_G);
    double* d_shift = (double*)work + 8;               // header slot
    if (d_info && cudaMemsetAsync(d_info, 0, sizeof(int), st) != cudaSuccess) return RQR_ERR_LAUNCH;
    RQR_TRY(rqr_trsm_gram(V, m, n, n, nullptr, G, nullptr, n, work, st));
    RQR_TRY(rqr_scholqr3_shift(G, n, m, d_shift, st));
    RQR_TRY(rqr_chol_dev(G, n, 0.0, d_shift, RA, d_info, st, nullptr, nullptr));
    // Q1 = V RA^-1 and its Gram; then cholQR2 of Q1
    RQR_TRY(rqr_trsm_gram(V, m, n, n, RA, G, Q, n, work, st));
    RQR_TRY(rqr_chol_dev(G, n, 0.0, nullptr, RB, d_info, st, nullptr, nullptr));
    RQR_TRY(tail_cholqr(Q, m, n, RB, Q, RC, G, work, d_info, 0, st, T));       // T = RC RB
    RQR_TRY(rqr_triu_mul(T, RA, n, R, st));
    return RQR_OK;
}
