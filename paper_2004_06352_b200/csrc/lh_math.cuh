// lh_math.cuh -- the FP64 primitives of the superposition kernel.
//
// The per-(pixel, lens) arithmetic of a dPIE needs two square roots with their
// reciprocals, four reciprocals, one atan and one atanh.  libdevice spends ~190 FP64
// instructions per evaluation on them.  On the B200 an FP64 warp instruction holds the
// dispatch port of its SM sub-partition for 2 cycles (3 when it reads three distinct vector
// registers) and every other instruction for 1, so both counts matter.
// These replacements all follow one pattern:
//
//   1. a 20-bit seed from the MUFU unit (MUFU.RCP64H / MUFU.RSQ64H: `rcp.approx.ftz.f64`,
//      `rsqrt.approx.ftz.f64`; relative error < 1e-6).
//   2. ONE third-order correction in FMAs: error e -> O(e^3) ~ 1e-18, i.e. the result is
//      good to a few ulp.  Several reciprocals share one seed and one correction through
//      the reciprocal of their product (rcp2 / rcp4).
//   3. for atan / atanh: range reduction against a shared-memory table indexed by the
//      exponent and the top 6 mantissa bits of the approximate quotient (seed x numerator;
//      the additive constants of the two index arguments ride in the FMA that forms them, so
//      that each index costs shift + biased unsigned min + address + LDS and nothing else),
//      with the quotient folded into the reduced argument so that each function needs ONE
//      refined reciprocal:
//        atan(n/d)  = atan(c) + atan( (|n| - c d)/(d + c |n|) ),  c = |n|/d rounded to 6 bits
//        atanh(n/d) = atanh(c') + atanh( (|n| - c' d)/(d - c' |n|) ),  c' = 1 - t_c with
//                     t_c = 1 - |n|/d rounded to 6 mantissa bits
//      and a two-term odd polynomial on |z| <= 2^-8 (truncation < 6e-16 relative).
//      No branch, no swap of numerator and denominator: large quotients are large table
//      indices.
//
// Every function is __host__ __device__ so that the CPU-only tests can pin the same source
// (lh_math_host_eval in include/lh.h); on the host the MUFU seeds are emulated by an exact
// quotient truncated to 20 mantissa bits.
#pragma once
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstring>

#define LH_HD __host__ __device__ __forceinline__

namespace lh {

// atan table, indexed by the exponent / 6-mantissa-bit code of q' = q + 2^-8 (q = |n|/d approximately):
//   entry 0                      q' in [2^-8, 2^-8 (1 + 1/64))  i.e. q < 2^-14: the identity, c = 0
//   entry 64 o + k (1..1023)     q' in 2^(o-8) [1 + k/64, 1 + (k+1)/64):  c = 2^(o-8) (1 + (k + 1/2)/64) - 2^-8
//   entry 1024                   q' >= 2^8:  c = 2^8  (z = (q - c)/(1 + c q) stays below 1/c)
// atanh table: entry 0 is the identity (c' = 0); see quot_index_down.
constexpr int TAB_PER_OCT = 64;
constexpr int ATAN_OCT_MIN = -8, ATAN_OCTAVES = 16;  // quotient in [2^-8, 2^8)
constexpr int ATAN_N = ATAN_OCTAVES * TAB_PER_OCT + 1;
constexpr int LN_OCTAVES = 16;                        // t = 1 - |n|/d in (2^-16, 1]
constexpr int LN_N = LN_OCTAVES * TAB_PER_OCT + 1;

struct MathTables {
    double2 at[ATAN_N];  // {c, atan c}
    double2 ah[LN_N];    // {c', atanh c'}, c' = 1 - t_c
};

// The three constants of the correction steps that have a non-zero low word or share an instruction with another
// constant (an FP64 instruction takes ONE immediate / uniform operand, so the second constant needs a vector
// register).  As literals ptxas rematerialises them inside the lens loop (two moves each per iteration, 8 in all);
// the kernel therefore hands them in as VALUES it read from its launch parameters -- loop-invariant registers the
// compiler cannot fold.  The defaults serve the host build and the stand-alone forms.
struct Consts {
    double third = 1.0 / 3.0, fifth = 0.2, c375 = 0.375;
};

// ---- bit access -------------------------------------------------------------------------------
LH_HD int hi32(double x) {
#ifdef __CUDA_ARCH__
    return __double2hiint(x);
#else
    int64_t b; std::memcpy(&b, &x, 8); return (int)(b >> 32);
#endif
}
LH_HD int lo32(double x) {
#ifdef __CUDA_ARCH__
    return __double2loint(x);
#else
    int64_t b; std::memcpy(&b, &x, 8); return (int)(b & 0xffffffff);
#endif
}
LH_HD double mk64(int hi, int lo) {
#ifdef __CUDA_ARCH__
    return __hiloint2double(hi, lo);
#else
    int64_t b = ((int64_t)hi << 32) | (uint32_t)lo; double x; std::memcpy(&x, &b, 8); return x;
#endif
}

// ---- MUFU seeds (relative error <= 2^-19.9) ---------------------------------------------------
LH_HD double rcp_seed(double x) {
#ifdef __CUDA_ARCH__
    double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y;
#else
    return mk64(hi32(1.0 / x), 0);
#endif
}
LH_HD double rsq_seed(double x) {
#ifdef __CUDA_ARCH__
    double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y;
#else
    return mk64(hi32(1.0 / std::sqrt(x)), 0);
#endif
}

// 1/x: seed + third-order step  y (1 + e + e^2), e = 1 - x y.          3 FP64 + 1 MUFU
LH_HD double rcp(double x) {
    const double y = rcp_seed(x);
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);
}

// 1/a and 1/b from one seed: r = 1/(a b), 1/a = r b, 1/b = r a.       6 FP64 + 1 MUFU
LH_HD void rcp2(double a, double b, double &ia, double &ib) {
    const double r = rcp(a * b);
    ia = r * b;
    ib = r * a;
}

// four reciprocals from one seed (product tree).                      12 FP64 + 1 MUFU
// The product a b c d must stay inside the double range (lh.h states the resulting range of lengths).
LH_HD void rcp4(double a, double b, double c, double d, double &ia, double &ib, double &ic, double &id) {
    const double ab = a * b, cd = c * d;
    const double r = rcp(ab * cd);
    const double rab = r * cd, rcd = r * ab;  // 1/(a b), 1/(c d)
    ia = rab * b;
    ib = rab * a;
    ic = rcd * d;
    id = rcd * c;
}

// w = sqrt(v) and iw = 1/sqrt(v), v > 0: seed + third-order step
//   (1 + h) y and (1 + h) v y,  h = e (1/2 + 3 e/8), e = 1 - v y^2.     6 FP64 + 1 MUFU
// (both closing FMAs read one register twice: two distinct registers each; a caller that
// drops iw pays 5)
LH_HD void rsqrt_sqrt(double v, double &w, double &iw, const Consts &K = Consts()) {
    const double y = rsq_seed(v);
    const double t = v * y;
    const double e = fma(-t, y, 1.0);
    const double h = fma(K.c375, e, 0.5) * e;
    iw = fma(y, h, y);
    w = fma(t, h, t);
}

// w = sqrt(v) alone (same seed and step as rsqrt_sqrt, without the closing FMA of 1/sqrt).   5 FP64 + 1 MUFU
LH_HD double sqrt_pos(double v, const Consts &K = Consts()) {
    const double y = rsq_seed(v);
    const double t = v * y;
    const double e = fma(-t, y, 1.0);
    const double h = fma(K.c375, e, 0.5) * e;
    return fma(t, h, t);
}

// copysign as ONE integer operation on the high word (1 dispatch cycle, not 2); mag >= 0
LH_HD double copysign_pos_i(double mag, double sgn) { return mk64(hi32(mag) | (hi32(sgn) & (int)0x80000000), lo32(mag)); }

// Table index of q' = q + 2^-8 >= 2^-8 (q >= 0 approximate quotient): exponent and top 6 mantissa bits,
// truncated, counted from the code of 2^-8.  No lower clamp is needed (q' >= 2^-8 by construction); the
// unsigned min sends everything at or above 2^8 -- and NaN / negative garbage -- to the last entry.
LH_HD unsigned quot_index_up(double qp, int n) {
    const unsigned j = (unsigned)((hi32(qp) >> 14) - ((1023 + ATAN_OCT_MIN) << 6));
#ifdef __CUDA_ARCH__
    return min(j, (unsigned)(n - 1));
#else
    return j > (unsigned)(n - 1) ? (unsigned)(n - 1) : j;
#endif
}

// Table index of t in (0, 1] counted DOWN from 1: entry 0 is t = 1 (c' = 0), entry 64 o + k,
// k = 0..63, is t_c = 2^-(o+1) (2 - k/64) ... i.e. the exponent/6-bit-mantissa code of t, rounded to
// nearest, subtracted from that of 1.0.  The caller guarantees t <= 1 (atanh_reduce forms it as
// 1 - an * seed), so the difference is never negative; t below the table -- and NaN / negative garbage,
// whose difference wraps to a large unsigned -- maps to the last entry.
LH_HD unsigned quot_index_down(double t, int n) {
    const unsigned j = (unsigned)(((1023 << 20) + 0x2000 - hi32(t))) >> 14;  // round((code(1.0) - code(t)) / 2^14)
#ifdef __CUDA_ARCH__
    return min(j, (unsigned)(n - 1));
#else
    return j > (unsigned)(n - 1) ? (unsigned)(n - 1) : j;
#endif
}

// ---- atan(n/d), d > 0 -------------------------------------------------------------------------
// Split in two so that the caller can share the reciprocal of the reduced denominator with
// other reciprocals (rcp2 / rcp4), and fed with an = |n| so that the caller can fold the
// absolute value into the instruction that produces n (|x| operand modifiers are free):
//   atan_reduce: pick c, return num = an - c d and den = d + c an (> 0)             3 FP64 + 1 MUFU
//   atan_finish: z = num/den given 1/den, atan c + z (1 - z^2/3 + z^4/5), sign of `sgn`  5 FP64
struct Reduced {
    double num, den, base;
};
LH_HD Reduced atan_reduce(double an, double d, const double2 *__restrict__ tab) {
    const double qp = fma(an, rcp_seed(d), 0x1p-8);  // |n|/d to 1e-6, + 2^-8: the index needs no lower clamp
    const double2 ca = tab[quot_index_up(qp, ATAN_N)];
    return Reduced{fma(-ca.x, d, an), fma(ca.x, an, d), ca.y};
}
LH_HD double atan_finish(const Reduced &r, double iden, double sgn, const Consts &K = Consts()) {
    const double z = r.num * iden;  // |z| <= 2^-8
    const double z2 = z * z;
    const double p = fma(z2, fma(z2, K.fifth, -K.third), 1.0);
    return copysign_pos_i(fma(z, p, r.base), sgn);
}

// ---- atanh(n/d), 0 <= an = |n| < d with 1 - an/d > 2^-16 --------------------------------------
// u = an/d; the bin is chosen on t = 1 - u = (d-an)/d, whose exponent follows the singularity
// of atanh at u = 1: bins are t_c = 2^-e (1 + k/64), c' = 1 - t_c, so that the reduced argument
//   s = (an - c' d)/(d - c' an) = (u - c')/(1 - c' u)
// stays below 2^-7.5 everywhere (|u - c'| <= t/128 and 1 - c'u >= 1 - u^2 ~ 2t near u = 1).
// Both FMAs see the exact an and d.  The host packer (lh_pack.cpp) routes every lens whose
// ellipticity could push u past the table into the CLS_EXTREME class, which does not come
// through here; the index is clamped all the same.
// t is formed as 1 - an * seed(d) (one FMA): its ABSOLUTE error is u * 2^-19.9, which against the bin
// half-width t/128 is negligible as long as t > 2^-8.6, i.e. eps <= EXTREME_EPS = 0.85 (lh_pack.h).
//   atanh_reduce  3 FP64 + 1 MUFU      atanh_finish  5 FP64
LH_HD Reduced atanh_reduce(double an, double d, const double2 *__restrict__ tab) {
    const double t0 = fma(-an, rcp_seed(d), 1.0);  // 1 - u, absolute error u 2^-19.9; never above 1
    const double2 ca = tab[quot_index_down(t0, LN_N)];
    return Reduced{fma(-ca.x, d, an), fma(-ca.x, an, d), ca.y};
}
LH_HD double atanh_finish(const Reduced &r, double iden, double sgn, const Consts &K = Consts()) {
    const double s = r.num * iden;
    const double s2 = s * s;
    const double p = fma(s2, fma(s2, K.fifth, K.third), 1.0);
    return copysign_pos_i(fma(s, p, r.base), sgn);
}

// Stand-alone forms (one reciprocal each), any sign of n
LH_HD double atan_nd(double n, double d, const double2 *__restrict__ tab) {
    const Reduced r = atan_reduce(fabs(n), d, tab);
    return atan_finish(r, rcp(r.den), n);
}
LH_HD double atanh_nd(double n, double d, const double2 *__restrict__ tab) {
    const Reduced r = atanh_reduce(fabs(n), d, tab);
    return atanh_finish(r, rcp(r.den), n);
}

// host: fill the tables (long-double libm: they are constants of the library)
inline void fill_math_tables(MathTables &T) {
    T.at[0] = make_double2(0.0, 0.0);
    for (int j = 1; j < ATAN_N - 1; ++j) {
        const int e = j / TAB_PER_OCT + ATAN_OCT_MIN, m = j % TAB_PER_OCT;
        const double c = std::ldexp(1.0 + ((double)m + 0.5) / TAB_PER_OCT, e) - std::ldexp(1.0, ATAN_OCT_MIN);  // exact
        T.at[j] = make_double2(c, (double)atanl((long double)c));
    }
    {
        const double c = std::ldexp(1.0, ATAN_OCT_MIN + ATAN_OCTAVES);
        T.at[ATAN_N - 1] = make_double2(c, (double)atanl((long double)c));
    }
    // entry j <-> code(1.0) - j: j = 64 o + k, k = 1..64  ->  t_c = 2^-(o+1) (2 - k/64)  (k = 64: 2^-(o+1))
    for (int j = 0; j < LN_N; ++j) {
        const int code = (1023 << 6) - j;  // exponent field and 6 mantissa bits of t_c
        const double tc = std::ldexp(1.0 + (double)(code & 63) / TAB_PER_OCT, (code >> 6) - 1023);
        const double cp = 1.0 - tc;  // exact
        T.ah[j] = make_double2(cp, (double)atanhl((long double)cp));
    }
}

}  // namespace lh
