/*
 * oracle/rqr_oracle.c -- CPU ORACLE for rand_cholQR with Count-Gauss multisketching.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or constant generator with the CUDA path
 * (paper_2309_05868_b200/csrc) and neither includes the other.
 *
 * A plain, slow, obviously-correct double-precision restatement of
 *   Higgins, Szyld, Boman, Yamazaki, "Analysis of Randomized Householder-Cholesky QR
 *   Factorization with Multisketching" (arxiv 2309.05868), cited below as PAPER.md:<line>.
 * Every function follows the algorithm step by step in the paper's order; there is no
 * blocking, fusion or reordering beyond what is stated here:
 *   - orc_gram and orc_dense_gauss_sketch sum over the m rows in blocks of ORC_SUM_BLOCK
 *     rows (block sums, then the block sums in ascending order).  Reading S10 in
 *     a strictly sequential double sum over m = 2^21..2^23 terms random-walks
 *     to ~1e-13, which is the size of the tolerance the paper's claim is tested at.
 *   - OpenMP is used only over independent rows / independent output entries / the
 *     blocks above, so results are bit-identical for any thread count.
 *
 * Letters follow BASELINE.json: V is m x n (m rows >> n columns), s1 = p1, s2 = p2.
 * The paper writes V in R^{n x m}, S1 in R^{p1 x n}, S2 in R^{p2 x p1}.
 * All matrices are row-major.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   philox            Random123 known-answer vectors (tests/golden/philox_kat.txt)
 *   hash/sign         worked example seed 42 (tests/golden/sketch_seed42.txt), uniformity
 *   gaussian          worked example, moments, Kolmogorov-Smirnov against N(0,1)
 *   countsketch       dense S1 @ V through numpy; exact integer case; column-sum identity
 *   gauss_sketch      numpy S2 @ W1
 *   rademacher        sign bits against the Philox words spelled out, +-1/sqrt(s2) exactly, balance and
 *                     pairwise independence of rows, E||S x||^2 = ||x||^2, embedding of a random subspace,
 *                     numpy S2 @ W1; rand_cholqr with it: the Thm 5.3 invariants
 *   hhqr_r/hhqr_full  LAPACK QR through numpy; R^T R = W^T W
 *   trsm, chol, gram, triu_mul   scipy/numpy library routines; exact integer cases
 *   rand_cholqr       Thm 5.3 invariants over kappa = 1 .. 1e15,
 *                     R against Householder QR of V (uniqueness of QR), kappa(V1) = O(1)
 *                     (Thm 5.2)
 *   cholqr2, scholqr3 failure thresholds of Fig. 4
 * Unpinned: nothing in this file.  The curves of Figs 1-7 are images and are not
 * reproduced ("parity unpinned" for those).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_SUM_BLOCK 256

/* status codes (the oracle's own; the CUDA library defines its own in include/rqr.h) */
#define ORC_OK 0
#define ORC_NOT_SPD 1000      /* + j (1-based): Cholesky pivot j not positive / NaN  */
#define ORC_SINGULAR 2000     /* + j (1-based): Householder column j has zero norm   */

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  The paper is silent on the RNG
 * (PAPER.md:93 "chosen uniformly at random"; :883 generation is off the clock); reading
 * S1 in DESIGN.md fixes it:  key = (seed lo, seed hi), counter = (idx lo, idx hi, stream, 0),
 * stream 0 = CountSketch, 1 = S2, 3 = single dense Gaussian sketch.
 * ---------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static void philox_stream(uint64_t seed, uint64_t idx, uint32_t stream, uint32_t out[4])
{
    uint32_t ctr[4] = { (uint32_t)idx, (uint32_t)(idx >> 32), stream, 0u };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    orc_philox4x32_10(ctr, key, out);
}

/* ------------------------------------------------------------------------------------
 * O1  CountSketch hash and sign.  PAPER.md:93: S1 has "a single +-1 per column, where
 * the row storing the entry and its sign are chosen uniformly at random".  Column i of
 * S1 (= row i of V) gets bucket h_i in [0,s1) and sign sigma_i from one Philox call:
 *   bucket = (uint64(out[0]) * s1) >> 32,   sigma = -1 if (out[1] & 1) else +1.
 * Rows are numbered globally: index = row0 + local row.
 * ---------------------------------------------------------------------------------- */
void orc_hash_sign(uint64_t seed, uint64_t row0, int64_t count, uint64_t s1,
                   uint32_t *bucket, int8_t *sign)
{
    for (int64_t t = 0; t < count; ++t) {
        uint32_t o[4];
        philox_stream(seed, row0 + (uint64_t)t, 0u, o);
        bucket[t] = (uint32_t)(((uint64_t)o[0] * s1) >> 32);
        sign[t] = (o[1] & 1u) ? (int8_t)-1 : (int8_t)1;
    }
}

/* ------------------------------------------------------------------------------------
 * O2  W1 = S1 V, S1 unscaled ("unscaled CountSketch"), computed as
 * "adding/subtracting subsets of rows of V":
 *   W1 = 0;  for i ascending:  W1[h_i, :] += sigma_i * V[i, :].
 * OpenMP splits the COLUMNS, so every entry still sees its terms in ascending i.
 * ---------------------------------------------------------------------------------- */
void orc_countsketch(const double *V, int64_t m, int n, int64_t ldv, int64_t s1,
                     uint64_t seed, uint64_t row0, double *W1 /* s1 x n */)
{
    uint32_t *h = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)(m > 0 ? m : 1));
    int8_t *sg = (int8_t *)malloc((size_t)(m > 0 ? m : 1));
    orc_hash_sign(seed, row0, m, (uint64_t)s1, h, sg);
    memset(W1, 0, sizeof(double) * (size_t)s1 * (size_t)n);
#pragma omp parallel for schedule(static)
    for (int j = 0; j < n; ++j)
        for (int64_t i = 0; i < m; ++i)
            W1[(int64_t)h[i] * n + j] += (double)sg[i] * V[i * ldv + j];
    free(h); free(sg);
}

/* ------------------------------------------------------------------------------------
 * Gaussian entries (reading S3 in DESIGN.md).  PAPER.md:89: S = G / sqrt(p) with G a
 * dense standard Gaussian.  Entry e (row-major linear index) lives in pair q = e >> 1:
 *   o = philox(q, stream);  x1 = (o[0]*2^32 + o[1]) >> 12;  u1 = (2 x1 + 1) 2^-53 in (0,1)
 *   u2 likewise from o[2], o[3];  rho = sqrt(-2 ln u1);
 *   z_even = rho cos(2 pi u2),  z_odd = rho sin(2 pi u2)      (Box-Muller)
 * cos/sin(2 pi u2) by exact argument reduction: t = 4 u2, k = nearest integer to t,
 * r = t - k (exact), then sin/cos(pi/2 r) and a quadrant swap -- glibc has no sinpi.
 * ---------------------------------------------------------------------------------- */
static void sincos_2pi(double u, double *s, double *c)
{
    double t = 4.0 * u;                 /* exact */
    double k = nearbyint(t);            /* 0..4 */
    double r = t - k;                   /* exact, |r| <= 0.5 */
    double a = 1.5707963267948966 * r;  /* pi/2 * r */
    double sr = sin(a), cr = cos(a);
    int q = ((int)k) & 3;
    switch (q) {
    case 0: *s = sr;  *c = cr;  break;
    case 1: *s = cr;  *c = -sr; break;
    case 2: *s = -sr; *c = -cr; break;
    default:*s = -cr; *c = sr;  break;
    }
}

static void gauss_pair(uint64_t seed, uint64_t q, uint32_t stream, double *z0, double *z1,
                       double *u1_out, double *u2_out)
{
    uint32_t o[4];
    philox_stream(seed, q, stream, o);
    uint64_t x1 = (((uint64_t)o[0] << 32) | o[1]) >> 12;
    uint64_t x2 = (((uint64_t)o[2] << 32) | o[3]) >> 12;
    double u1 = (double)(2 * x1 + 1) * 0x1p-53;
    double u2 = (double)(2 * x2 + 1) * 0x1p-53;
    double rho = sqrt(-2.0 * log(u1));
    double s, c;
    sincos_2pi(u2, &s, &c);
    *z0 = rho * c;
    *z1 = rho * s;
    if (u1_out) *u1_out = u1;
    if (u2_out) *u2_out = u2;
}

/* standard normal z(e) for linear entry indices first .. first+count-1 of a stream */
void orc_gauss_z(uint64_t seed, uint32_t stream, uint64_t first, int64_t count, double *z)
{
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < count; ++t) {
        uint64_t e = first + (uint64_t)t;
        double z0, z1;
        gauss_pair(seed, e >> 1, stream, &z0, &z1, NULL, NULL);
        z[t] = (e & 1) ? z1 : z0;
    }
}

/* the uniforms of pair q, for the worked-example pin */
void orc_gauss_pair_debug(uint64_t seed, uint32_t stream, uint64_t q, uint32_t words[4],
                          double u[2], double z[2])
{
    philox_stream(seed, q, stream, words);
    gauss_pair(seed, q, stream, &z[0], &z[1], &u[0], &u[1]);
}

/* S2[r,c] = z(r*s1 + c) / sqrt(s2), stream 1 ("scaled Gaussian sketch") */
void orc_gauss_matrix(uint64_t seed, int s2, int64_t s1, double *S2 /* s2 x s1 */)
{
    int64_t total = (int64_t)s2 * s1;
    orc_gauss_z(seed, 1u, 0, total, S2);
    double d = sqrt((double)s2);
    for (int64_t e = 0; e < total; ++e) S2[e] = S2[e] / d;
}

/* ------------------------------------------------------------------------------------
 * O3  W = S2 W1 ("first computing W1 = S1 V, then W = S2 W1"):
 *   W[r, j] = sum_{c ascending} S2[r, c] * W1[c, j].
 * ---------------------------------------------------------------------------------- */
void orc_gauss_sketch(const double *W1, int64_t s1, int n, int s2, uint64_t seed,
                      double *W /* s2 x n */)
{
    double *S2 = (double *)malloc(sizeof(double) * (size_t)s2 * (size_t)s1);
    orc_gauss_matrix(seed, s2, s1, S2);
    /* loop nest r, c, j: every entry W[r,j] still receives its terms in ascending c (the
     * stated order); only the memory walk is contiguous */
#pragma omp parallel for schedule(static)
    for (int r = 0; r < s2; ++r) {
        double *w = W + (int64_t)r * n;
        for (int j = 0; j < n; ++j) w[j] = 0.0;
        for (int64_t c = 0; c < s1; ++c) {
            const double a = S2[(int64_t)r * s1 + c];
            const double *b = W1 + c * n;
            for (int j = 0; j < n; ++j) w[j] += a * b[j];
        }
    }
    free(S2);
}

/* ------------------------------------------------------------------------------------
 * N4  Dense Rademacher S2 in place of the Gaussian one (future work: "dense
 * Rademacher sketch matrices in place of dense Gaussian sketches ... far lower storage
 * requirements ... can be generated much more efficiently"; the analysis "is amenable to any
 * multisketching strategy", same paragraph).  Reading S21 in DESIGN.md:
 *   S2[r, c] = sigma(r, c) / sqrt(s2),  sigma = -1 if bit (c mod 128) of the 128-bit Philox output
 *   o = philox(idx = r * ceil(s1 / 128) + (c div 128), stream 4) is set, else +1;  bit b of the
 *   output is bit (b mod 32) of word o[b div 32].
 * W = S2 W1 as in O3: W[r, j] = sum_{c ascending} S2[r, c] * W1[c, j].
 * ---------------------------------------------------------------------------------- */
void orc_rademacher_matrix(uint64_t seed, int s2, int64_t s1, double *S2 /* s2 x s1 */)
{
    const uint64_t ng = (uint64_t)((s1 + 127) / 128);
    const double d = sqrt((double)s2);
    for (int r = 0; r < s2; ++r)
        for (int64_t c = 0; c < s1; ++c) {
            uint32_t o[4];
            philox_stream(seed, (uint64_t)r * ng + (uint64_t)(c / 128), 4u, o);
            const int b = (int)(c % 128);
            const int set = (int)((o[b / 32] >> (b % 32)) & 1u);
            S2[(int64_t)r * s1 + c] = (set ? -1.0 : 1.0) / d;
        }
}

void orc_rademacher_sketch(const double *W1, int64_t s1, int n, int s2, uint64_t seed,
                           double *W /* s2 x n */)
{
    double *S2 = (double *)malloc(sizeof(double) * (size_t)s2 * (size_t)s1);
    orc_rademacher_matrix(seed, s2, s1, S2);
#pragma omp parallel for schedule(static)
    for (int r = 0; r < s2; ++r) {
        double *w = W + (int64_t)r * n;
        for (int j = 0; j < n; ++j) w[j] = 0.0;
        for (int64_t c = 0; c < s1; ++c) {
            const double a = S2[(int64_t)r * s1 + c];
            const double *b = W1 + c * n;
            for (int j = 0; j < n; ++j) w[j] += a * b[j];
        }
    }
    free(S2);
}

/* ------------------------------------------------------------------------------------
 * Single dense Gaussian sketch W = S V, S = G/sqrt(s), s x m (PAPER.md:218-220, :234,
 * :877), generated on the fly from stream 3: S[r, i] = z(r*m_total + row0 + i)/sqrt(s).
 * Sum over the m rows in blocks of ORC_SUM_BLOCK (see header).
 * ---------------------------------------------------------------------------------- */
void orc_dense_gauss_sketch(const double *V, int64_t m, int n, int64_t ldv, int s,
                            uint64_t seed, uint64_t row0, uint64_t m_total,
                            double *W /* s x n */)
{
    double d = sqrt((double)s);
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < s; ++r) {
        double *tot = (double *)calloc((size_t)n, sizeof(double));
        double *blk = (double *)malloc(sizeof(double) * (size_t)n);
        double *zr = (double *)malloc(sizeof(double) * ORC_SUM_BLOCK);
        for (int64_t b0 = 0; b0 < m; b0 += ORC_SUM_BLOCK) {
            int64_t b1 = b0 + ORC_SUM_BLOCK < m ? b0 + ORC_SUM_BLOCK : m;
            for (int j = 0; j < n; ++j) blk[j] = 0.0;
            for (int64_t i = b0; i < b1; ++i) {
                uint64_t e = (uint64_t)r * m_total + row0 + (uint64_t)i;
                double z0, z1;
                gauss_pair(seed, e >> 1, 3u, &z0, &z1, NULL, NULL);
                zr[i - b0] = ((e & 1) ? z1 : z0) / d;
            }
            for (int64_t i = b0; i < b1; ++i)
                for (int j = 0; j < n; ++j) blk[j] += zr[i - b0] * V[i * ldv + j];
            for (int j = 0; j < n; ++j) tot[j] += blk[j];
        }
        for (int j = 0; j < n; ++j) W[(int64_t)r * n + j] = tot[j];
        free(tot); free(blk); free(zr);
    }
}

/* ------------------------------------------------------------------------------------
 * O4  R factor of the Householder QR of A (rows x n, rows >= n), "hhqr(W)".
 * Classical column-by-column Householder (Higham, Accuracy and Stability, ch. 19, the
 * model the paper's analysis uses):
 *   x = A[j:, j];  v = x + sign(x_1) ||x||_2 e_1;  H = I - 2 v v^T / (v^T v);
 *   A[j:, j:] = H A[j:, j:].
 * A is destroyed.  R = upper n x n of the result, strict lower part set to exact zero;
 * rows with a negative diagonal are multiplied by -1 so that diag(R) > 0 (reading S4 in
 * DESIGN.md; the paper does not fix the sign, Cholesky fixes it for R1).
 * If Qout != NULL (rows x n) the thin Q is accumulated by applying the reflectors to
 * [I_n; 0] in reverse order and the same sign flips to its columns: the brute-force
 * Householder QR used on tiny inputs.
 * ---------------------------------------------------------------------------------- */
int orc_hhqr(double *A, int64_t rows, int n, double *R /* n x n */, double *Qout)
{
    int info = ORC_OK;
    double *Vs = NULL;     /* reflector vectors, column j stored in Vs[j*rows + i], i >= j */
    double *beta = NULL;
    if (Qout) {
        Vs = (double *)calloc((size_t)rows * (size_t)n, sizeof(double));
        beta = (double *)calloc((size_t)n, sizeof(double));
    }
    double *v = (double *)malloc(sizeof(double) * (size_t)rows);
    for (int j = 0; j < n; ++j) {
        double nrm2 = 0.0;
        for (int64_t i = j; i < rows; ++i) nrm2 += A[i * n + j] * A[i * n + j];
        double nrm = sqrt(nrm2);
        if (!(nrm > 0.0) && info == ORC_OK) info = ORC_SINGULAR + j + 1;
        double x1 = A[(int64_t)j * n + j];
        double sgn = (x1 < 0.0) ? -1.0 : 1.0;
        for (int64_t i = j; i < rows; ++i) v[i] = A[i * n + j];
        v[j] = x1 + sgn * nrm;
        double vtv = 0.0;
        for (int64_t i = j; i < rows; ++i) vtv += v[i] * v[i];
        double b = (vtv > 0.0) ? 2.0 / vtv : 0.0;
        for (int c = j; c < n; ++c) {
            double w = 0.0;
            for (int64_t i = j; i < rows; ++i) w += v[i] * A[i * n + c];
            w *= b;
            for (int64_t i = j; i < rows; ++i) A[i * n + c] -= w * v[i];
        }
        if (Qout) {
            for (int64_t i = j; i < rows; ++i) Vs[(int64_t)j * rows + i] = v[i];
            beta[j] = b;
        }
    }
    for (int a = 0; a < n; ++a)
        for (int c = 0; c < n; ++c) R[a * n + c] = (c >= a) ? A[(int64_t)a * n + c] : 0.0;
    if (Qout) {
        for (int64_t i = 0; i < rows; ++i)
            for (int c = 0; c < n; ++c) Qout[i * n + c] = (i == c) ? 1.0 : 0.0;
        for (int j = n - 1; j >= 0; --j) {
            const double *vj = Vs + (int64_t)j * rows;
            for (int c = 0; c < n; ++c) {
                double w = 0.0;
                for (int64_t i = j; i < rows; ++i) w += vj[i] * Qout[i * n + c];
                w *= beta[j];
                for (int64_t i = j; i < rows; ++i) Qout[i * n + c] -= w * vj[i];
            }
        }
    }
    for (int a = 0; a < n; ++a)
        if (R[a * n + a] < 0.0) {
            for (int c = a; c < n; ++c) R[a * n + c] = -R[a * n + c];
            if (Qout) for (int64_t i = 0; i < rows; ++i) Qout[i * n + a] = -Qout[i * n + a];
        }
    free(v); free(Vs); free(beta);
    return info;
}

/* ------------------------------------------------------------------------------------
 * O5  X = V R^{-1}, R upper triangular: each row by forward substitution, the row-wise
 * model of PAPER.md:449-453 eq. (42) (Alg. 1 step 3 :115; Alg. 2 step 3 :198):
 *   x_j = (v_j - sum_{k<j} x_k R[k,j]) / R[j,j],   j = 0..n-1.
 * X may alias V.
 * ---------------------------------------------------------------------------------- */
void orc_trsm(const double *V, int64_t m, int n, int64_t ldv, const double *R,
              double *X, int64_t ldx)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < m; ++i) {
        const double *v = V + i * ldv;
        double *x = X + i * ldx;
        for (int j = 0; j < n; ++j) {
            double acc = v[j];
            for (int k = 0; k < j; ++k) acc -= x[k] * R[k * n + j];
            x[j] = acc / R[j * n + j];
        }
    }
}

/* ------------------------------------------------------------------------------------
 * O6  Gram matrix G = A^T A (Alg. 2 step 1), G[a,b] = sum_i A[i,a] A[i,b]
 * for a <= b, mirrored.  Rows are summed in blocks of ORC_SUM_BLOCK (see header).
 * ---------------------------------------------------------------------------------- */
void orc_gram(const double *A, int64_t m, int n, int64_t lda, double *G /* n x n */)
{
    int64_t nblk = (m + ORC_SUM_BLOCK - 1) / ORC_SUM_BLOCK;
    double *part = (double *)malloc(sizeof(double) * (size_t)(nblk > 0 ? nblk : 1) * (size_t)n * (size_t)n);
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < nblk; ++b) {
        double *P = part + b * (int64_t)n * n;
        for (int e = 0; e < n * n; ++e) P[e] = 0.0;
        int64_t i1 = (b + 1) * ORC_SUM_BLOCK < m ? (b + 1) * ORC_SUM_BLOCK : m;
        for (int64_t i = b * ORC_SUM_BLOCK; i < i1; ++i) {
            const double *r = A + i * lda;
            for (int a = 0; a < n; ++a)
                for (int c = a; c < n; ++c) P[a * n + c] += r[a] * r[c];
        }
    }
    for (int a = 0; a < n; ++a)
        for (int c = a; c < n; ++c) {
            double acc = 0.0;
            for (int64_t b = 0; b < nblk; ++b) acc += part[b * (int64_t)n * n + a * n + c];
            G[a * n + c] = acc;
            G[c * n + a] = acc;
        }
    free(part);
}

/* ------------------------------------------------------------------------------------
 * O7  Upper Cholesky factor, G + shift*I = R^T R (Alg. 2 step 2), row by
 * row.  Fails (status ORC_NOT_SPD + j) if a pivot is not > 0 (catches NaN).
 * ---------------------------------------------------------------------------------- */
int orc_chol(const double *G, int n, double shift, double *R /* n x n */)
{
    for (int e = 0; e < n * n; ++e) R[e] = 0.0;
    for (int j = 0; j < n; ++j) {
        double d = G[j * n + j] + shift;
        for (int k = 0; k < j; ++k) d -= R[k * n + j] * R[k * n + j];
        if (!(d > 0.0)) return ORC_NOT_SPD + j + 1;
        double rjj = sqrt(d);
        R[j * n + j] = rjj;
        for (int c = j + 1; c < n; ++c) {
            double s = G[j * n + c];
            for (int k = 0; k < j; ++k) s -= R[k * n + j] * R[k * n + c];
            R[j * n + c] = s / rjj;
        }
    }
    return ORC_OK;
}

/* O8  R = R1 R0, upper x upper (Alg. 3 step 3) */
void orc_triu_mul(const double *R1, const double *R0, int n, double *R)
{
    for (int a = 0; a < n; ++a)
        for (int c = 0; c < n; ++c) {
            double acc = 0.0;
            for (int k = a; k <= c; ++k) acc += R1[a * n + k] * R0[k * n + c];
            R[a * n + c] = (c >= a) ? acc : 0.0;
        }
}

/* Alg. 2 cholQR on A (m x n, ld n) -> Q (may alias A), R1 */
static int cholqr_step(const double *A, int64_t m, int n, double shift, double *Q, double *R1,
                       double *G)
{
    orc_gram(A, m, n, n, G);
    int info = orc_chol(G, n, shift, R1);
    if (info != ORC_OK) return info;
    orc_trsm(A, m, n, n, R1, Q, n);
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------
 * Alg. 3 rand_cholQR with Alg. 1 randQR using the
 * Count-Gauss multisketch:
 *   W1 = S1 V;  W = S2 W1;  R0 = hhqr(W).R;  V1 = V R0^{-1};      (randQR)
 *   G = V1^T V1;  R1 = chol(G);  Q = V1 R1^{-1};                    (cholQR of the STORED V1)
 *   R = R1 R0.
 * Optional outputs (may be NULL): R0out, R1out (n x n), V1out (m x n), W1out, Wout.
 * ---------------------------------------------------------------------------------- */
static int rand_cholqr_impl(const double *V, int64_t m, int n, int64_t s1, int s2, uint64_t seed,
                           double *Q, double *R, double *R0out, double *R1out, double *V1out,
                           double *W1out, double *Wout, int rademacher)
{
    double *W1 = (double *)malloc(sizeof(double) * (size_t)s1 * (size_t)n);
    double *W = (double *)malloc(sizeof(double) * (size_t)s2 * (size_t)n);
    double *R0 = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    double *R1 = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    double *G = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    int info;
    orc_countsketch(V, m, n, n, s1, seed, 0, W1);
    if (rademacher) orc_rademacher_sketch(W1, s1, n, s2, seed, W);
    else orc_gauss_sketch(W1, s1, n, s2, seed, W);
    if (W1out) memcpy(W1out, W1, sizeof(double) * (size_t)s1 * (size_t)n);
    if (Wout) memcpy(Wout, W, sizeof(double) * (size_t)s2 * (size_t)n);
    info = orc_hhqr(W, s2, n, R0, NULL);
    if (R0out) memcpy(R0out, R0, sizeof(double) * (size_t)n * (size_t)n);
    if (info == ORC_OK) {
        orc_trsm(V, m, n, n, R0, Q, n);                       /* V1, stored in Q */
        if (V1out) memcpy(V1out, Q, sizeof(double) * (size_t)m * (size_t)n);
        info = cholqr_step(Q, m, n, 0.0, Q, R1, G);
        if (R1out) memcpy(R1out, R1, sizeof(double) * (size_t)n * (size_t)n);
        if (info == ORC_OK) orc_triu_mul(R1, R0, n, R);
    }
    free(W1); free(W); free(R0); free(R1); free(G);
    return info;
}

int orc_rand_cholqr(const double *V, int64_t m, int n, int64_t s1, int s2, uint64_t seed,
                    double *Q, double *R, double *R0out, double *R1out, double *V1out,
                    double *W1out, double *Wout)
{
    return rand_cholqr_impl(V, m, n, s1, s2, seed, Q, R, R0out, R1out, V1out, W1out, Wout, 0);
}

/* the same with the Rademacher S2 of N4 (Count-Rademacher multisketch) */
int orc_rand_cholqr_rademacher(const double *V, int64_t m, int n, int64_t s1, int s2, uint64_t seed,
                               double *Q, double *R, double *R0out, double *R1out, double *V1out,
                               double *W1out, double *Wout)
{
    return rand_cholqr_impl(V, m, n, s1, s2, seed, Q, R, R0out, R1out, V1out, W1out, Wout, 1);
}

/* rand_cholQR with one dense Gaussian sketch S (s x m) in place of S2 S1
 * (PAPER.md:218-222, :234): W = S V, then as above. */
int orc_gauss_rand_cholqr(const double *V, int64_t m, int n, int s, uint64_t seed,
                          double *Q, double *R)
{
    double *W = (double *)malloc(sizeof(double) * (size_t)s * (size_t)n);
    double *R0 = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    double *R1 = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    double *G = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    orc_dense_gauss_sketch(V, m, n, n, s, seed, 0, (uint64_t)m, W);
    int info = orc_hhqr(W, s, n, R0, NULL);
    if (info == ORC_OK) {
        orc_trsm(V, m, n, n, R0, Q, n);
        info = cholqr_step(Q, m, n, 0.0, Q, R1, G);
        if (info == ORC_OK) orc_triu_mul(R1, R0, n, R);
    }
    free(W); free(R0); free(R1); free(G);
    return info;
}

/* Alg. 4 CholeskyQR2: cholQR twice, R = R1 R0.
 * Returns ORC_NOT_SPD + j if either Cholesky breaks down (kappa(V) >~ u^-1/2). */
int orc_cholqr2(const double *V, int64_t m, int n, double *Q, double *R)
{
    double *R0 = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    double *R1 = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    double *G = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    int info = cholqr_step(V, m, n, 0.0, Q, R0, G);
    if (info == ORC_OK) info = cholqr_step(Q, m, n, 0.0, Q, R1, G);
    if (info == ORC_OK) orc_triu_mul(R1, R0, n, R);
    free(R0); free(R1); free(G);
    return info;
}

/* ------------------------------------------------------------------------------------
 * Shifted CholeskyQR3.  The paper only cites it ([12] Fukaya et al.);
 * reading S9 in DESIGN.md restates the published method:
 *   G = V^T V;  shift = 11 (m n + n (n+1)) u ||V||_2^2, u = 2^-53, with ||V||_F^2 = tr(G)
 *   used as the bound on ||V||_2^2;  R0 = chol(G + shift I);  Q1 = V R0^{-1};
 *   [Q, R21] = cholQR2(Q1);  R = R21 R0.
 * ---------------------------------------------------------------------------------- */
int orc_scholqr3(const double *V, int64_t m, int n, double *Q, double *R, double *shift_out)
{
    double *R0 = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    double *R21 = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    double *G = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    orc_gram(V, m, n, n, G);
    double tr = 0.0;
    for (int j = 0; j < n; ++j) tr += G[j * n + j];
    double shift = 11.0 * ((double)m * n + (double)n * (n + 1)) * 0x1p-53 * tr;
    if (shift_out) *shift_out = shift;
    int info = orc_chol(G, n, shift, R0);
    if (info == ORC_OK) {
        orc_trsm(V, m, n, n, R0, Q, n);
        info = orc_cholqr2(Q, m, n, Q, R21);
        if (info == ORC_OK) orc_triu_mul(R21, R0, n, R);
    }
    free(R0); free(R21); free(G);
    return info;
}
