/*
 * rqr.h -- C ABI of librqr: the hot path of rand_cholQR with Count-Gauss multisketching
 * (Higgins, Szyld, Boman, Yamazaki, arxiv 2309.05868; cited as PAPER.md:<line>) for one
 * NVIDIA B200 (sm_100a).  Every step is a hand-written CUDA kernel; no cuBLAS / cuSOLVER /
 * cuSPARSE, no CPU fallback.
 *
 * Letters follow BASELINE.json: V is m x n (m rows >> n columns), s1 = CountSketch rows,
 * s2 = Gaussian sketch rows.  The paper writes V in R^{n x m}, S1 in R^{p1 x n},
 * S2 in R^{p2 x p1}.
 *
 * Conventions common to every entry point
 *  - All matrix pointers are DEVICE pointers to float64, ROW-MAJOR, with an element leading
 *    dimension where one is given (ldv, ldq >= n).  Small matrices (W1, W, R0, G, R1, R) are
 *    dense row-major with leading dimension n.  Bases must be 16-byte aligned.
 *  - The caller owns every buffer.  The library allocates nothing; scratch comes from `work`,
 *    a device buffer of at least rqr_workspace_bytes(...) bytes, 256-byte aligned.
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Every call is
 *    asynchronous on it, performs no synchronisation or allocation, and is CUDA-graph
 *    capturable.
 *  - Return value: RQR_OK, or -k if argument k (1-based) is invalid, or RQR_ERR_LAUNCH if a
 *    kernel launch failed.  NUMERICAL status goes to a device int (`d_info`, may be NULL):
 *      0                        success
 *      RQR_INFO_NOT_SPD + j     Cholesky pivot j (1-based) not > 0 or NaN  (cholQR2 at
 *                               kappa >~ u^-1/2)
 *      RQR_INFO_SINGULAR + j    Householder column j has zero / non-finite norm: V is rank
 *                               deficient for randQR
 *    d_info is written only on failure (first failure wins); the caller zeroes it (the
 *    one-shot drivers zero it themselves).  Outputs are undefined when *d_info != 0.
 *  - Argument limits: 2 <= n <= 256, n <= s2 <= s1 <= m_total (eq. (20)),
 *    s2 <= 1024 (s2 > 512 needs n <= 128 for the register-resident Householder kernel, else a
 *    slow fallback runs), s1 < 2^31, m < 2^31 per call.
 *  - Fast paths: the FP64 DMMA kernels of rqr_trsm_gram / rqr_apply need an even n, even leading
 *    dimensions and 16-byte aligned bases (2 <= n <= 64: fused kernels; 64 < n <= 256: panel
 *    kernels); rqr_gauss_sketch uses its DMMA GEMM for even n >= 96, and for even 32 <= n < 96 when the product is
 *    large (s2 >= 128 and s2 s1 n >= 5e7).  Any other
 *    shape runs the generic kernels: same results to rounding, much slower.
 *  - Thread safety: calls on different streams with different buffers are independent, from any host thread and on
 *    any device.  The library keeps no state besides the per-device "kernel attributes set" flags (atomic; the
 *    opt-in to > 48 KB of shared memory is per device and is repeated on the first call on each device).
 *  - Dynamic range: the Householder and Cholesky kernels form sums of squares of the sketch entries without
 *    scaling, so |V| must stay within about [1e-140, 1e140] (entries of W = S2 S1 V below 1e-154 or above 1e154
 *    would under/overflow in the squares and be reported as RQR_INFO_SINGULAR).
 */
#ifndef RQR_H
#define RQR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RQR_OK 0
#define RQR_ERR_LAUNCH (-1000)
#define RQR_ERR_COMM (-1001)   /* the caller's all-reduce callback of rqr_rand_cholqr_sharded returned non-zero */
#define RQR_INFO_NOT_SPD 1000
#define RQR_INFO_SINGULAR 2000

/* CountSketch variants */
#define RQR_VARIANT_SORTED 0  /* gather over the bucket-sorted row list (CSR form of S1, the
                                 paper's SpMM form); deterministic            */
#define RQR_VARIANT_SCATTER 1 /* stream V, hash on the fly, red.global.add.f64; the last
                                 bits depend on the order of the atomics                    */

#define RQR_VARIANT_STREAM 2  /* stream V in row order through shared memory (bulk async copies), hash on
                                 the fly, flip the sign in shared memory, and add every row to its bucket with
                                 ONE bulk reduction (cp.reduce.async.bulk ... add.f64, SASS UBLKRED) instead of n
                                 atomics: no stored S1 at all ("storage of only O(n) values"; :947
                                 "adding/subtracting subsets of rows"), nothing to prepare in A0; the order of
                                 the reductions is not fixed.  Needs even n and ld and 16-byte aligned bases
                                 (else it runs as RQR_VARIANT_SCATTER).  When the whole sketch fits shared
                                 memory (n <= 20 and 8 s1 n <= 224 KB; any ld, any alignment) every CTA
                                 accumulates its rows in a shared-memory bucket tile with shared-memory
                                 atomics and flushes it once (north_star's "shared-memory bucket tiles").  */

/* flags */
#define RQR_FLAG_PREPARED 1   /* `work` already holds the sketch state written by
                                 rqr_sketch_prepare with the same (m, n, row0, s1, s2,
                                 seed, variant): skip sketch generation (the paper's timing
                                 convention).  Without it the call generates
                                 what it needs first, on the same stream.                   */
#define RQR_FLAG_RECOMPUTE_V1 2 /* one-shot drivers: do not store V1 = V R0^-1; re-form it in
                                 the apply pass with bit-identical arithmetic (32mn bytes of
                                 traffic instead of 40mn, 4mn^2 flops instead of 3mn^2).
                                 Honoured for n <= 64; for n > 64 V1 is always stored.       */
#define RQR_FLAG_STORE_V1 4   /* one-shot drivers: store V1 into Q in A4 and transform it in place in A6.
                                 With neither flag the drivers choose per n: recomputed for n <= 24 (the
                                 path is HBM-bound there and moves 32mn instead of 40mn bytes), stored above
                                 (measured: from n = 32 up A4 is bound by the FP64 tensor pipe with or without
                                 the store, and the extra mn^2 flops of A6 do not hide).  When V and
                                 Q would not take the same kernel family (Q not 16-byte aligned while V is,
                                 even n) V1 is stored whatever the flags say: a V1 re-formed by different
                                 arithmetic would break the orthogonality of Q (DESIGN.md hazard H1).      */

#define RQR_S2_RADEMACHER 16  /* SURVEY.md 8(f) N4, PAPER.md:947 ("dense Rademacher sketch matrices in
                                 place of dense Gaussian sketches"): S2 has entries +-1/sqrt(s2)
                                 (reading S21; sign bits from Philox stream 4) and is
                                 generated on the fly inside the A2 product -- no S2 in memory
                                 (8 s2 s1 bytes: 512 MiB at n = 256), nothing to generate in A0.
                                 OR it into `variant` of rqr_workspace_bytes, rqr_sketch_prepare,
                                 rqr_countsketch (it only moves a workspace region there) and
                                 rqr_rand_cholqr, and into `flags` of rqr_gauss_sketch; a workspace
                                 must be used with the setting it was sized and prepared for.      */

/* Size in bytes of the workspace every call below accepts for this problem shape. */
size_t rqr_workspace_bytes(int64_t m, int n, int64_t s1, int s2, int variant);

/* A0 -- sketch generation, off the paper's clock.  Writes into `work`:
 * S2 (s2 x s1, entries N(0,1)/sqrt(s2)) from Philox4x32-10 stream 1 and, for
 * RQR_VARIANT_SORTED, the rows [row0, row0+m) sorted by CountSketch bucket (stable, ascending
 * row inside a bucket) with their signs, plus the s1+1 bucket offsets.  Bucket and sign of a
 * row are a function of its GLOBAL index row0 + i (Philox stream 0; reading S1).  */
int rqr_sketch_prepare(int64_t m, int n, int64_t row0, int64_t s1, int s2, uint64_t seed,
                       int variant, void* work, void* stream);

/* A1 -- CountSketch, Alg. 1 step 1 first half: W1 = S1 V,
 * W1[h(i),:] += sigma(i) V[i,:], S1 unscaled.  W1 (s1 x n) is overwritten.
 * RQR_VARIANT_SORTED with few buckets (2 s1 <= 1184): the bucket row lists are split into segments so that the
 * grid is full, and the partial sketches pass through the Gram-partial scratch of `work` (contents lost), summed
 * in a fixed order: the result stays bit-reproducible.                                                        */
int rqr_countsketch(const double* V, int64_t m, int n, int64_t ldv, int64_t row0, int64_t s1,
                    uint64_t seed, double* W1, void* work, int variant, int flags, void* stream);

/* A2 -- Gaussian sketch, Alg. 1 step 1 second half: W = S2 W1, W s2 x n.      */
int rqr_gauss_sketch(const double* W1, int64_t s1, int n, int s2, uint64_t seed, double* W,
                     void* work, int flags, void* stream);

/* A3 -- R factor of the Householder QR of W (Alg. 1 step 2).  W (s2 x n) is
 * destroyed (for n > 64 its storage carries the reflectors between the CTAs of the cluster).
 * R0 is n x n upper triangular with diag > 0 and exact zeros below.                         */
int rqr_small_geqrf(double* W, int s2, int n, double* R0, int* d_info, void* stream);

/* A4 -- fused V1 = V R0^-1 (Alg. 1 step 3; row-wise substitution, eq. (42)
 * PAPER.md:449-453) and Gram matrix G = V1^T V1 (Alg. 2 step 1), split over
 * row tiles with a fixed-order reduction.  R0 == NULL means identity (plain Gram of V).
 * G (n x n) is written full symmetric.  V1 != NULL: V1 (m x n, ld ldq) is also stored;
 * V1 == V is allowed.  For n > 64 with R0 != NULL the tensor-core path needs V1 (returns -7
 * otherwise): the substitution and the Gram are two kernels there, and a V1 re-formed by other
 * arithmetic would not be the matrix rqr_apply transforms (orthogonality would drop to
 * u kappa(V)).                                                                                */
int rqr_trsm_gram(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* G,
                  double* V1, int64_t ldq, void* work, void* stream);

/* A4 for callers that cannot allocate or carry a workspace (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same operation and the same kernels as rqr_trsm_gram (Alg. 1 step 3 +
 * Alg. 2 step 1), with NO `work` argument.  The per-CTA Gram partials (the only scratch A4
 * needs for n <= 64) live in a file-scope `static __device__` array inside the library:
 *     RQR_NOALLOC_MAX_PARTIALS x RQR_NOALLOC_MAX_N^2 doubles = 148 x 64 x 64 x 8 = 4 849 664 bytes,
 * held by every GPU that loads librqr.so until the process exits.  The call performs no cudaMalloc / cudaFree and
 * calls no allocating routine; the first call on each device looks the array's device address up once
 * (cudaGetSymbolAddress, with that device current) and sets the kernels' shared-memory attributes -- make that
 * first call outside stream capture.
 *  - Limits: 2 <= n <= RQR_NOALLOC_MAX_N (64) and 1 <= m <= RQR_NOALLOC_MAX_M (2^23 rows, one accumulation chunk).
 *    A shape beyond either returns RQR_ERR_SCRATCH_LIMIT and launches nothing.  Other arguments as rqr_trsm_gram
 *    (return -k for argument k of THIS signature).
 *  - Results: on the DMMA path (even n, even ld, 16-byte aligned bases) G and V1 are bit-identical to
 *    rqr_trsm_gram's; on the generic path the partial count is capped at 148 (rqr_trsm_gram: 304), so G agrees to
 *    rounding (1e-13 relative), V1 bit for bit.
 *  - The array is SHARED by every call on a device and keeps the last call's contents.  Nothing in it has to
 *    start at zero: each launch overwrites the partials it reads back (CTA p writes partial p in full before the
 *    reduction reads partials 0 .. grid-1).  Two calls that overlap on the GPU (different streams, or concurrent
 *    graph branches) RACE on it: serialise them, or use rqr_trsm_gram with one workspace per stream.            */
#define RQR_ERR_SCRATCH_LIMIT (-1002)
#define RQR_NOALLOC_MAX_N 64
#define RQR_NOALLOC_MAX_M ((int64_t)1 << 23)
#define RQR_NOALLOC_MAX_PARTIALS 148
int rqr_trsm_gram_noalloc(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* G,
                          double* V1, int64_t ldq, void* stream);

/* A5 -- upper Cholesky factor, G + shift I = R1^T R1 (Alg. 2 step 2).  R1 is n x n
 * upper triangular with diag > 0 and exact zeros below; it must not alias G (for n > 128 the part
 * of R1 that ends up zero is scratch during the call: inverse diagonal blocks and the Schur
 * complement of the two-level factorization live there).  First failing pivot j (0-based):
 * *d_info = RQR_INFO_NOT_SPD + j + 1.                                                         */
int rqr_chol(const double* G, int n, double shift, double* R1, int* d_info, void* stream);

/* A6 -- Q = (V R0^-1) R1^-1 (Alg. 2 step 3), never V (R0^-1 R1^-1).
 * R0 == NULL: V already holds V1 (stored by rqr_trsm_gram) and Q = V R1^-1.  R0 != NULL: V1
 * is re-formed with arithmetic bit-identical to rqr_trsm_gram's.  Q == V is allowed.         */
int rqr_apply(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
              double* Q, int64_t ldq, void* work, void* stream);

/* A7 -- R = R1 R0, upper x upper (Alg. 3 step 3).                              */
int rqr_triu_mul(const double* R1, const double* R0, int n, double* R, void* stream);

/* One-shot Alg. 3 rand_cholQR with Count-Gauss: Q (m x n, ld n), R (n x n).
 * V has leading dimension n.  Q == V is allowed.                                             */
int rqr_rand_cholqr(const double* V, int64_t m, int n, int64_t s1, int s2, uint64_t seed,
                    double* Q, double* R, void* work, int* d_info, int variant, int flags,
                    void* stream);

/* Row-sharded Alg. 3 over several GPUs, one process per GPU: this rank holds the rows
 * [row0, row0 + m) of an m_total x n matrix (V, Q: m x n, ld n; a rank may hold fewer than n rows).  Bucket and
 * sign of a row are functions of its GLOBAL index, S2 is replicated, and the ranks meet exactly twice -- "rand_cholQR
 * only requires two synchronizations total": the sum of the local sketches W_k = S2 (S1)_k V_k
 * (s2 x n; PAPER.md:228 footnote 3) and the sum of the local Gram matrices (n x n).  The library links no
 * communication library: `allreduce(ctx, buf, count, stream)` is the caller's in-place sum of `count` doubles at
 * the DEVICE pointer `buf` over all ranks, enqueued on `stream` (e.g. ncclAllReduce(buf, buf, count, ncclDouble,
 * ncclSum, comm, stream)); it must return 0, give every rank the same bits, and be capturable if the call is
 * captured.  allreduce == NULL: one rank.  Every rank ends with the same R; Q holds this rank's rows.
 * A workspace prepared with RQR_FLAG_PREPARED must have been prepared with the same row0.                      */
typedef int (*rqr_allreduce_fn)(void* ctx, double* buf, int64_t count, void* stream);
int rqr_rand_cholqr_sharded(const double* V, int64_t m, int64_t row0, int64_t m_total, int n, int64_t s1, int s2,
                            uint64_t seed, double* Q, double* R, void* work, int* d_info, int variant, int flags,
                            rqr_allreduce_fn allreduce, void* ctx, void* stream);

/* Batched / strided form for block-Krylov use ("Krylov subspace methods that
 * require tall-and-skinny QR factorizations, particularly block ..."): `batch` problems of the same shape,
 * problem b at V + b strideV (m x n, ld n), Q + b strideQ, R + b n^2, d_info + b.  The sketch operator is the
 * same for every problem (one seed), so the sketch state in `work` is generated once (or not at all with
 * RQR_FLAG_PREPARED) and the problems run back to back on the stream; each is bit-identical to the single call. */
int rqr_rand_cholqr_batched(const double* V, int64_t m, int n, int batch, int64_t strideV, int64_t s1, int s2,
                            uint64_t seed, double* Q, int64_t strideQ, double* R, void* work, int* d_info,
                            int variant, int flags, void* stream);

/* Comparators on the same kernels.  Alg. 4 CholeskyQR2.                   */
int rqr_cholqr2(const double* V, int64_t m, int n, double* Q, double* R, void* work, int* d_info,
                void* stream);
/* Shifted CholeskyQR3 (cited only; reading S9): shift =
 * 11 (m n + n(n+1)) 2^-53 tr(V^T V).                                                         */
int rqr_scholqr3(const double* V, int64_t m, int n, double* Q, double* R, void* work, int* d_info,
                 void* stream);
/* rand_cholQR with ONE dense Gaussian sketch S (s x m, N(0,1)/sqrt(s), Philox stream 3,
 * generated on the fly).                                             */
int rqr_gauss_randcholqr(const double* V, int64_t m, int n, int s, uint64_t seed, double* Q,
                         double* R, void* work, int* d_info, void* stream);
/* rand_cholQR with ONE CountSketch (the paper's "Sparse" rows): R0 = R factor of the
 * Householder QR of the s1 x n sketch W1 = S1 V itself, computed by a TSQR tree (n <= 64: 128-row blocks in the
 * register-resident kernel; n > 64: 1024- / 512-row blocks, one thread-block cluster per block).              */
int rqr_count_randcholqr(const double* V, int64_t m, int n, int64_t s1, uint64_t seed, double* Q,
                         double* R, void* work, int* d_info, int variant, int flags, void* stream);
/* R factor (n x n upper, diag > 0) of the Householder QR of a tall A (rows x n row-major, ld n, n <= 64,
 * rows >= n) by a TSQR tree of 128-row blocks; A is not modified; `work` as for the other calls.            */
int rqr_tsqr_r(const double* A, int64_t rows, int n, double* R, void* work, int* d_info, void* stream);
/* The dense sketch step alone: W (s x n) = S V for rows [row0, row0+m) of m_total.           */
int rqr_dense_gauss_sketch(const double* V, int64_t m, int n, int64_t ldv, int64_t row0,
                           int64_t m_total, int s, uint64_t seed, double* W, void* work,
                           void* stream);

/* Measurement hook: only the draw of the s x m Gaussians of rqr_dense_gauss_sketch (same launch shape, no V traffic,
 * no products): the generation bound of the single-Gaussian-sketch comparator.  n even.                          */
int rqr_debug_dense_gauss_draw_only(int64_t m, int n, int s, uint64_t seed, void* work, void* stream);

/* Inspection helpers for parity tests (device outputs): bucket (uint32) and sign (int8, +-1)
 * of rows [row0, row0+count); Gaussian stream entries z(first .. first+count-1).            */
int rqr_debug_hash_sign(uint64_t seed, int64_t row0, int64_t count, int64_t s1, uint32_t* bucket,
                        int8_t* sign, void* stream);
int rqr_debug_gauss(uint64_t seed, uint32_t stream_id, uint64_t first, int64_t count, double* z,
                    void* stream);
/* Pointer to S2 (s2 x s1) inside a workspace prepared for (n, s1).  Row r starts at r * ld with
 * ld = s1 rounded up to a multiple of 16; the pad columns hold zeros.                         */
const double* rqr_workspace_S2(void* work, int n, int64_t s1);
/* Pointers to the bucket offsets (s1 + 1 uint32) and the bucket-sorted row list (m uint32: local row index in the
 * low 31 bits, sign bit 31 set for sigma = -1) that rqr_sketch_prepare (RQR_VARIANT_SORTED) wrote into a workspace
 * sized for (m, n, s1, variant).                                                                           */
int rqr_workspace_rows(void* work, int64_t m, int n, int64_t s1, int variant, const uint32_t** offsets,
                       const uint32_t** entries);
/* Device pointer to the shift the last rqr_scholqr3 call on this workspace used (reading S9).                 */
const double* rqr_workspace_scholqr3_shift(void* work);
/* test hook: the signs (+1 / -1) of the Rademacher S2 entries (row, c0 .. c0 + count) for sketch width s1 */
int rqr_debug_rademacher(uint64_t seed, int64_t s1, int row, int64_t c0, int64_t count, int8_t* sign,
                         void* stream);

/* Test hooks: rqr_trsm_gram / rqr_apply on the generic (non-DMMA) kernels whatever the shape.    */
int rqr_debug_trsm_gram_generic(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* G,
                                double* V1, int64_t ldq, void* work, void* stream);
int rqr_debug_apply_generic(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                            double* Q, int64_t ldq, void* work, void* stream);

/* Library version string. */
const char* rqr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RQR_H */
