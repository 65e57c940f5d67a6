// rqr_gauss.cuh -- branch-free Box-Muller pair of the CUDA path (reading S3), built for instruction count:
// the single dense Gaussian sketch (B'', rqr_dense_mma.cu) draws s m Gaussians per factorization and is bound by the
// ISSUE rate of this routine.  Same definition as rqr_gauss_pair in rqr_common.cuh (which calls it):
//   out = philox(q, stream);  x1 = (out0:out1) >> 12, x2 = (out2:out3) >> 12;  u = (2x + 1) 2^-53;
//   rho = sqrt(-2 ln u1);  z_even = rho cos(2 pi u2),  z_odd = rho sin(2 pi u2).
// What differs from calling log / sincospi of the CUDA math library (~320 instructions per pair, two data-dependent
// branches) -- ~190 instructions, none of them a branch:
//   * u1 = k 2^-53 (k odd, < 2^53): mantissa m' in [sqrt(1/2), sqrt(2)) and exponent from the high word of (double)k
//     with 32-bit integer operations.
//   * ln m = ln c_i + log1p(r), c_i = i / 128 the grid point NEAREST to m (i = round(128 m), 91 entries, table
//     rqr_log_table.inc written by gen_log_table.py), r = m / c_i - 1 by one fma, |r| <= 2^-7.5; log1p by its Taylor
//     polynomial to r^7.  The entry of c = 1 is (1, 0) exactly and its bin reaches to both sides of 1, so arguments
//     next to 1 (rho -> 0) keep full RELATIVE accuracy without a special case.
//   * 2 pi u2 = (pi / 2)(k + f): quadrant k = round(4 u2) and f in [-1/2, 1/2] again from the integer (2 x2 + 1):
//     f is exact and never 0; sin and cos of (pi / 2) f by their Taylor polynomials to a^17 / a^16 (truncation
//     < 2^-58 for |a| <= pi / 4), quadrant rotation by selects and sign-bit flips.
// Measured against the CPU oracle (libm log / sin / cos, written independently): tests/test_gpu_steps.py
// test_gauss_entries_within_1e15 (north_star tolerance 1e-15 relative, absolute below 1).
#pragma once
#include <stdint.h>
#include <string.h>
#include <math.h>

#if defined(__CUDACC__)
#define RQR_HD __host__ __device__ __forceinline__
#else
#define RQR_HD static inline
#endif

struct RqrLogEntry {
    double invc, logc;
};
#define RQR_LOG_TAB_LO 91
#define RQR_LOG_TAB_N 91
#if defined(__CUDACC__)
static __device__ const RqrLogEntry d_rqr_log_tab[RQR_LOG_TAB_N] = {
#include "rqr_log_table.inc"
};
#endif
static const RqrLogEntry h_rqr_log_tab[RQR_LOG_TAB_N] = {
#include "rqr_log_table.inc"
};

RQR_HD double rqr_bits_to_double(uint64_t b)
{
#if defined(__CUDA_ARCH__)
    return __longlong_as_double((long long)b);
#else
    double d;
    memcpy(&d, &b, 8);
    return d;
#endif
}
RQR_HD uint64_t rqr_double_to_bits(double d)
{
#if defined(__CUDA_ARCH__)
    return (uint64_t)__double_as_longlong(d);
#else
    uint64_t b;
    memcpy(&b, &d, 8);
    return b;
#endif
}
RQR_HD uint32_t rqr_hi32(double d) { return (uint32_t)(rqr_double_to_bits(d) >> 32); }
RQR_HD double rqr_with_hi32(double d, uint32_t hi)
{
    return rqr_bits_to_double(((uint64_t)hi << 32) | (rqr_double_to_bits(d) & 0xFFFFFFFFull));
}

// one Philox4x32 round (Salmon et al., SC'11; reading S1) on (c0..c3) with round key (k0, k1)
RQR_HD void rqr_philox_round(uint32_t& c0, uint32_t& c1, uint32_t& c2, uint32_t& c3, uint32_t k0, uint32_t k1)
{
    // one 32 x 32 -> 64 product per multiplier (SASS IMAD.WIDE.U32): high and low word from one instruction
    uint32_t h0, l0, h1, l1;
#ifdef __CUDA_ARCH__
    asm("{\n\t.reg .b64 p;\n\tmul.wide.u32 p, %2, %3;\n\tmov.b64 {%0, %1}, p;\n\t}" : "=r"(l0), "=r"(h0) : "r"(c0), "r"(0xD2511F53u));
    asm("{\n\t.reg .b64 p;\n\tmul.wide.u32 p, %2, %3;\n\tmov.b64 {%0, %1}, p;\n\t}" : "=r"(l1), "=r"(h1) : "r"(c2), "r"(0xCD9E8D57u));
#else
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    h0 = (uint32_t)(p0 >> 32); l0 = (uint32_t)p0;
    h1 = (uint32_t)(p1 >> 32); l1 = (uint32_t)p1;
#endif
    const uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
    c0 = n0; c1 = l1; c2 = n2; c3 = l0;
}

// ------------------------------------------------------------------------------------------------------------------
// The pair as a sequence of NSTAGES short straight-line stages, so that a caller can place independent work (the
// DMMAs of rqr_dense_mma.cu) between them; run back to back they are the whole routine (rqr_gauss_pair).
//   stages 0..9   Philox rounds
//   stage 10      the two 53-bit odd integers; ln: mantissa / exponent / table entry; sincos: quadrant, a = (pi/2) f
//   stages 11..13 ln: r, w, hi, lo, the log1p polynomial; sin and cos polynomials (interleaved: independent chains)
//   stage 14      rho = sqrt(-2 ln u1); sin a, cos a
//   stage 15      quadrant rotation, z = rho (cos, sin)
// ln(k 2^-53), k odd < 2^53:  all decisions on the HIGH WORD of (double)k (32-bit integer operations; k converts
// exactly): m' in [0.7071066, 1.4142132), i = round(128 m') on the truncated mantissa, ln = kd ln 2 + ln c_i + log1p(r).
// cos / sin(2 pi N 2^-53), N odd < 2^53: quadrant qd = round(4 u) = (N + 2^50) >> 51 and f 2^51 = N - qd 2^51 on the
// high word (bit 51 is bit 19 of it); f is exact, odd, never 0.
// ------------------------------------------------------------------------------------------------------------------
struct RqrPairDraw {
    static constexpr int NSTAGES = 16;
    uint32_t c0, c1, c2, c3, k0, k1;
    uint32_t qd;
    double md, kd, invc, logc, r, r2, q, hi, lo, a, a2, ps, pc, rho, sa, ca;
    double z0, z1;                                     // results after stage 15: z_even, z_odd

    RQR_HD void begin(uint64_t seed, uint64_t idx, uint32_t stream)
    {
        c0 = (uint32_t)idx; c1 = (uint32_t)(idx >> 32); c2 = stream; c3 = 0u;
        k0 = (uint32_t)seed; k1 = (uint32_t)(seed >> 32);
    }
    template <int S>
    RQR_HD void stage(const RqrLogEntry* tab)
    {
        if constexpr (S < 10) {
            rqr_philox_round(c0, c1, c2, c3, k0, k1);
            k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
        } else if constexpr (S == 10) {
            // k = 2 x1 + 1, x1 = (c0:c1) >> 12:  k = ((c0:c1) >> 11) | 1
            const uint64_t k = ((((uint64_t)c0 << 32) | c1) >> 11) | 1ull;
            const uint64_t N = ((((uint64_t)c2 << 32) | c3) >> 11) | 1ull;
            const double d = (double)k;                        // exact
            const uint32_t h = rqr_hi32(d);
            const uint32_t mh = h & 0x000FFFFFu;               // top 20 mantissa bits: m = 1.mh... in [1, 2)
            const bool big = mh >= 0x6A09Eu;                   // m >= 1.41421318 (just below sqrt 2): m' = m / 2
            const int i = big ? 64 + (int)((mh + 0x2000u) >> 14) : 128 + (int)((mh + 0x1000u) >> 13);
            md = rqr_with_hi32(d, mh | (big ? 0x3FE00000u : 0x3FF00000u));
            kd = (double)((int)(h >> 20) - (1023 + 53) + (big ? 1 : 0));      // k 2^-53 = m' 2^kd
            const RqrLogEntry t = tab[i - RQR_LOG_TAB_LO];
            invc = t.invc; logc = t.logc;
            const uint32_t nh = (uint32_t)(N >> 32);
            qd = (nh + (1u << 18)) >> 19;                                      // 0 .. 4
            const int64_t fi = (int64_t)(((uint64_t)(nh - (qd << 19)) << 32) | (N & 0xFFFFFFFFull));
            a = (double)fi * 0x1.921fb54442d18p-51;            // (pi / 2) f, f = fi 2^-51 exact; |a| <= pi / 4
        } else if constexpr (S == 11) {
            r = fma(md, invc, -1.0);
            const double w = fma(kd, 0x1.62e42fefa39efp-1, logc);   // kd ln 2 + ln c (|kd| <= 53: the dropped low
                                                                    // part of ln 2 is below 2^-59 of the result)
            hi = w + r;
            lo = (w - hi) + r;
            r2 = r * r;
            a2 = a * a;
            // log1p(r) = r + r^2 (-1/2 + r/3 - r^2/4 + r^3/5 - r^4/6 + r^5/7)
            q = fma(1.0 / 7.0, r, -1.0 / 6.0);
            // Taylor coefficients of sin / cos: reciprocals of factorials below 2^53 (correctly rounded)
            ps = fma(-1.0 / 355687428096000.0, a2, 1.0 / 1307674368000.0);        // -1/17!, 1/15!
            pc = fma(1.0 / 20922789888000.0, a2, -1.0 / 87178291200.0);           //  1/16!, -1/14!
        } else if constexpr (S == 12) {
            q = fma(q, r, 1.0 / 5.0);
            q = fma(q, r, -0.25);
            ps = fma(ps, a2, -1.0 / 6227020800.0);         // -1/13!
            ps = fma(ps, a2, 1.0 / 39916800.0);            //  1/11!
            ps = fma(ps, a2, -1.0 / 362880.0);             // -1/9!
            pc = fma(pc, a2, 1.0 / 479001600.0);           //  1/12!
            pc = fma(pc, a2, -1.0 / 3628800.0);            // -1/10!
            pc = fma(pc, a2, 1.0 / 40320.0);               //  1/8!
        } else if constexpr (S == 13) {
            q = fma(q, r, 1.0 / 3.0);
            q = fma(q, r, -0.5);
            ps = fma(ps, a2, 1.0 / 5040.0);                //  1/7!
            ps = fma(ps, a2, -1.0 / 120.0);                // -1/5!
            ps = fma(ps, a2, 1.0 / 6.0);                   //  1/3!  (sin a = a - a^3 (1/6 - a^2/120 + ...))
            pc = fma(pc, a2, -1.0 / 720.0);                // -1/6!
            pc = fma(pc, a2, 1.0 / 24.0);                  //  1/4!
            pc = fma(pc, a2, -0.5);
        } else if constexpr (S == 14) {
            const double ln_u1 = fma(r2, q, lo) + hi;
            rho = sqrt(-2.0 * ln_u1);
            sa = fma(-(a * a2), ps, a);
            ca = fma(a2, pc, 1.0);
        } else {
            // rotate by qd quadrants: (cos, sin)(a + qd pi / 2)
            const bool swap = (qd & 1u) != 0;
            const double cc = swap ? sa : ca, ss = swap ? ca : sa;
            const uint64_t cneg = (uint64_t)(((qd + 1u) >> 1) & 1u) << 63;     // qd = 1, 2: cos negative
            const uint64_t sneg = (uint64_t)((qd >> 1) & 1u) << 63;           // qd = 2, 3: sin negative
            z0 = rho * rqr_bits_to_double(rqr_double_to_bits(cc) ^ cneg);
            z1 = rho * rqr_bits_to_double(rqr_double_to_bits(ss) ^ sneg);
        }
    }
};

template <int S>
RQR_HD void rqr_pair_draw_run(RqrPairDraw& d, const RqrLogEntry* tab)
{
    if constexpr (S < RqrPairDraw::NSTAGES) {
        d.template stage<S>(tab);
        rqr_pair_draw_run<S + 1>(d, tab);
    }
}
