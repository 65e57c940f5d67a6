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

// header slot of the workspace that rqr_scholqr3 writes its shift to
#define RQR_HDR_SHIFT_SLOT 8
extern "C" const double* rqr_workspace_scholqr3_shift(void* work)
{
    return work ? (const double*)work + RQR_HDR_SHIFT_SLOT : nullptr;
}

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

// V1 = V R0^-1 stored or recomputed (PAPER.md:220-222 flop terms; reading S20).  Stored: A4 writes V1
// into Q and A6 transforms it in place: 40mn bytes, 3mn^2 flops.  Recomputed: A4 stores nothing and A6 re-forms V1
// with the bit-identical routine: 32mn bytes, 4mn^2 flops.  Measured (profiles/r2_summary.md sections 3 and 9): with
// 8 x 8 tiles A4 executes NB (NB + 1) DMMA per 8 rows for the substitution and as many for the Gram, so from n = 32 up
// it is bound by the FP64 tensor pipe with or without the store (0.343 vs 0.348 ms at 2^22 x 32), and the second
// substitution in A6 costs more than the store saves from n = 40 up.  Recomputing wins for n <= 24 (10^7 x 16: A4 + A6
// 0.76 vs 0.90 ms; 10^7 x 24: 1.13 vs 1.23), ties at 32 and loses above (n = 40: 0.98 vs 0.91; n = 64: 2.82 vs 2.41).
// Default: "recompute iff n <= RQR_AUTO_RECOMPUTE_MAX_N"; RQR_FLAG_RECOMPUTE_V1 / RQR_FLAG_STORE_V1 override it.
// Every driver (CholeskyQR2 and sCholQR3 included) takes the same decision: the comparison stays on the same kernels.
#define RQR_AUTO_RECOMPUTE_MAX_N 24
static bool use_recompute(const double* V, int n, const double* R0, const double* Q, int flags)
{
    if (!R0 || n > 64) return false;      // n > 64: A4 is FP64-bound either way and V1 is always stored
    bool want = n <= RQR_AUTO_RECOMPUTE_MAX_N;
    if (flags & RQR_FLAG_RECOMPUTE_V1) want = true;
    if (flags & RQR_FLAG_STORE_V1) want = false;
    // A4 (no V1 stored) dispatches on V alone, A6 on V and Q: a V1 re-formed by the other kernel family would have
    // other rounding (hazard H1).  Both take the same family iff n is odd (generic for both), V is misaligned
    // (generic for both) or Q is aligned too (DMMA for both); otherwise V1 is stored.
    const bool same_family = (n & 1) || (((uintptr_t)V & 15) != 0) || (((uintptr_t)Q & 15) == 0);
    return want && same_family;
}

// cholQR of V R0^-1: shared tail of every driver.  A4 with R0 (stores V1 into Q unless V1 is recomputed), A5 (which
// also forms Rprod = R1 R0, the drivers' A7, when Rprod != NULL), A6.
// ar != NULL (row-sharded form): the Gram matrices of the ranks are summed between A4 and A5 (the
// second of the two synchronizations).
static int tail_cholqr(const double* V, int64_t m, int n, const double* R0, double* Q, double* R1,
                       double* G, void* work, int* d_info, int flags, cudaStream_t st, double* Rprod,
                       rqr_allreduce_fn ar = nullptr, void* ar_ctx = nullptr)
{
    const bool recompute = use_recompute(V, n, R0, Q, flags);
    RQR_TRY(rqr_trsm_gram(V, m, n, n, R0, G, recompute ? nullptr : Q, n, work, st));
    if (ar && ar(ar_ctx, G, (int64_t)n * n, (void*)st) != 0) return RQR_ERR_COMM;
    RQR_TRY(rqr_chol_dev(G, n, 0.0, nullptr, R1, d_info, st, R0, Rprod));
    if (recompute) RQR_TRY(rqr_apply(V, m, n, n, R0, R1, Q, n, work, st));
    else           RQR_TRY(rqr_apply(Q, m, n, n, nullptr, R1, Q, n, work, st));
    return RQR_OK;
}

// Alg. 3 on the rows [row0, row0 + m) of an m_total-row matrix; ar == NULL: the whole matrix (row0 = 0, m_total = m)
static int rand_cholqr_impl(const double* V, int64_t m, int64_t row0, int64_t m_total, int n, int64_t s1, int s2,
                            uint64_t seed, double* Q, double* R, void* work, int* d_info, int variant, int flags,
                            rqr_allreduce_fn ar, void* ar_ctx, void* stream)
{
    int rc = check_common(V, m, n, Q, R, work);
    if (rc == -100) return !Q ? -7 : (!R ? -8 : -9);
    if (rc == -3 && n >= 2 && n <= RQR_MAX_N && n <= m_total) rc = RQR_OK;    // a shard may hold fewer than n rows
    if (rc != RQR_OK) return rc;
    if (s1 < 1 || s1 >= ((int64_t)1 << 31) || s1 > m_total) return -4;
    if (s2 < n || s2 > s1 || s2 > RQR_MAX_S2) return -5;      // eq. (20)
    const int rad = variant & RQR_S2_RADEMACHER;                 // N4: Count-Rademacher multisketch
    {
        const int cs = variant & ~RQR_S2_RADEMACHER;
        if (cs != RQR_VARIANT_SORTED && cs != RQR_VARIANT_SCATTER && cs != RQR_VARIANT_STREAM) return -11;
    }
    cudaStream_t st = (cudaStream_t)stream;
    RqrLayout L = rqr_layout(m, n, s1, rad != 0);
    double* R0 = small_mat(work, L, n, RQR_SM_R0);
    double* R1 = small_mat(work, L, n, RQR_SM_R1);
    double* G = small_mat(work, L, n, RQR_SM_G);
    double* W1 = (double*)((char*)work + L.F_W1);
    double* W = (double*)((char*)work + L.F_W);
    if (d_info && cudaMemsetAsync(d_info, 0, sizeof(int), st) != cudaSuccess) return RQR_ERR_LAUNCH;
    if (!(flags & RQR_FLAG_PREPARED))
        RQR_TRY(rqr_sketch_prepare(m, n, row0, s1, s2, seed, variant, work, st));
    // Alg. 1 randQR: W = S2 S1 V; R0 = hhqr(W).R; V1 = V R0^-1
    RQR_TRY(rqr_countsketch(V, m, n, n, row0, s1, seed, W1, work, variant, RQR_FLAG_PREPARED, st));
    RQR_TRY(rqr_gauss_sketch(W1, s1, n, s2, seed, W, work, RQR_FLAG_PREPARED | rad, st));
    // row-sharded: W = sum over the ranks of S2 (S1)_k V_k (PAPER.md:228 footnote 3), the first synchronization
    if (ar && ar(ar_ctx, W, (int64_t)s2 * n, stream) != 0) return RQR_ERR_COMM;
    RQR_TRY(rqr_small_geqrf(W, s2, n, R0, d_info, st));
    // Alg. 2 cholQR of V1; Alg. 3 step 3
    RQR_TRY(tail_cholqr(V, m, n, R0, Q, R1, G, work, d_info, flags, st, R, ar, ar_ctx));
    return RQR_OK;
}

extern "C" int rqr_rand_cholqr(const double* V, int64_t m, int n, int64_t s1, int s2, uint64_t seed,
                               double* Q, double* R, void* work, int* d_info, int variant,
                               int flags, void* stream)
{
    return rand_cholqr_impl(V, m, 0, m, n, s1, s2, seed, Q, R, work, d_info, variant, flags, nullptr, nullptr, stream);
}

// Row-sharded Alg. 3 (SURVEY.md 8(e); PAPER.md:208 "only requires two synchronizations total", :228 footnote 3).
extern "C" int rqr_rand_cholqr_sharded(const double* V, int64_t m, int64_t row0, int64_t m_total, int n, int64_t s1,
                                       int s2, uint64_t seed, double* Q, double* R, void* work, int* d_info,
                                       int variant, int flags, rqr_allreduce_fn allreduce, void* ctx, void* stream)
{
    if (row0 < 0) return -3;
    if (m_total < row0 + m || m_total >= ((int64_t)1 << 40)) return -4;
    int rc = rand_cholqr_impl(V, m, row0, m_total, n, s1, s2, seed, Q, R, work, d_info, variant, flags, allreduce,
                              ctx, stream);
    // argument numbers of this entry point: V 1, m 2, n 5, s1 6, s2 7, Q 9, R 10, work 11, variant 13
    switch (rc) {
        case -3: return -5;
        case -4: return -6;
        case -5: return -7;
        case -7: return -9;
        case -8: return -10;
        case -9: return -11;
        case -11: return -13;
        default: return rc;
    }
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

// rows the TSQR scratch (region A of the workspace: cap blocks of n^2 doubles) can take.  The stacked R factors
// ping-pong inside region A: level 1 writes nb0 = ceil(rows / 128) blocks, level 2 the next ceil(nb0 n / 128) <=
// nb0 / 2 + 1 (n <= 64) behind them, and every later level fits into the space of the level two before it.
// nb0 + nb0 / 2 + 1 <= cap - 1 holds for rows <= 128 * ((cap - 2) * 2 / 3).
static int64_t tsqr_max_rows(int n) { return (int64_t)128 * (((int64_t)rqr_gram_partial_cap(n) - 2) * 2 / 3); }

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
    if (variant != RQR_VARIANT_SORTED && variant != RQR_VARIANT_SCATTER && variant != RQR_VARIANT_STREAM) return -10;
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
    RQR_TRY(tail_cholqr(V, m, n, R0, Q, R1, G, work, d_info, flags, st, R));
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
    double* d_shift = (double*)work + RQR_HDR_SHIFT_SLOT;
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
