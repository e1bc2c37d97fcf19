// lh_math.cuh -- the FP64 primitives of the superposition kernel.
//
// The per-(pixel, lens) arithmetic of a dPIE needs two square roots with their
// reciprocals, four reciprocals, one atan and one atanh.  libdevice spends ~190 FP64-pipe
// instructions per evaluation on them; the B200 FP64 pipe issues one warp instruction
// every two cycles per scheduler, so instruction count is the roofline.  These
// replacements all follow one pattern:
//
//   1. a 20-bit seed from the MUFU unit (MUFU.RCP64H / MUFU.RSQ64H: `rcp.approx.ftz.f64`,
//      `rsqrt.approx.ftz.f64`; measured max relative error 9.9e-7 and 9.3e-7 on B200 --
//      profiles/r01_mufu_probe.txt).  The XU pipe runs beside the FP64 pipe.
//   2. ONE third-order correction in FMAs: error e -> O(e^3) ~ 1e-18, i.e. the result is
//      good to a few ulp (measured 1.1e-16 / 1.7e-16).
//   3. for atan / atanh: range reduction against a shared-memory table indexed by the
//      approximate quotient (seed x numerator), with the quotient folded into the reduced
//      argument so that each function costs ONE refined reciprocal:
//        atan(n/d)  = atan(c) + atan( (n - c d)/(d + c n) )             c = i/128
//        atanh(n/d) = atanh(c') + atanh( (n - c' d)/(d - c' n) ),  c' = (c-1)/(c+1) with
//                     c = (d+|n|)/(d-|n|) rounded to 6 mantissa bits (atanh c' = 1/2 ln c)
//      and a two-term odd polynomial on |z| <= 2^-8 (truncation < 6e-16 relative).
//
// Every function is __host__ __device__ so that the same source can be exercised by the
// CPU-only unit tests of the host logic; on the host the MUFU seeds are emulated by an
// exact quotient truncated to 20 mantissa bits.
#pragma once
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstring>

#define LH_HD __host__ __device__ __forceinline__

namespace lh {

constexpr int ATAN_N = 128;                 // atan table: c_i = i/128, i = 0..128
constexpr int LN_OCTAVES = 16;              // atanh table: ratio c in [1, 2^16), 64 entries per octave
constexpr int LN_PER_OCT = 64;
constexpr int LN_N = LN_OCTAVES * LN_PER_OCT;

struct MathTables {
    double2 at[ATAN_N + 1];  // {c_i, atan(c_i)}
    double2 ah[LN_N];        // {c'_j, atanh(c'_j)}, c'_j = (c_j-1)/(c_j+1), c_j = 2^(j/64) (linear inside an octave)
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

// w = sqrt(v) and iw = 1/sqrt(v), v > 0: seed + third-order step
//   y (1 + e/2 + 3 e^2/8), e = 1 - v y^2.                              6 FP64 + 1 MUFU
LH_HD void rsqrt_sqrt(double v, double &w, double &iw) {
    const double y = rsq_seed(v);
    const double t = v * y;
    const double e = fma(-t, y, 1.0);
    const double c = fma(0.375, e, 0.5);
    iw = fma(y * e, c, y);
    w = v * iw;
}

// |x| and copysign as integer operations on the high word (ALU pipe, not the FP64 pipe)
LH_HD double fabs_i(double x) { return mk64(hi32(x) & 0x7fffffff, lo32(x)); }
LH_HD double copysign_i(double mag, double sgn) {
    return mk64((hi32(mag) & 0x7fffffff) | (hi32(sgn) & (int)0x80000000), lo32(mag));
}
// a > b for two non-negative doubles: their bit patterns order like 64-bit integers
LH_HD bool gt_nonneg(double a, double b) {
#ifdef __CUDA_ARCH__
    return __double_as_longlong(a) > __double_as_longlong(b);
#else
    int64_t x, y; std::memcpy(&x, &a, 8); std::memcpy(&y, &b, 8); return x > y;
#endif
}

// atan(n/d) for d > 0 and any finite n.  Branch-free.                  12 FP64 + 2 MUFU
LH_HD double atan_nd(double n, double d, const double2 *__restrict__ tab) {
    const double an = fabs_i(n);
    const bool swap = gt_nonneg(an, d);
    const double hi = swap ? an : d, lo = swap ? d : an;  // t = lo/hi in [0, 1]
    // index: round(128 t) from the seed quotient, read from the low word after adding 1.5 * 2^45
    const double kk = fma(lo, rcp_seed(hi), 52776558133248.0);
    const unsigned i = min((unsigned)lo32(kk), (unsigned)ATAN_N);
    const double2 ca = tab[i];  // {c, atan c}
    const double num = fma(-ca.x, hi, lo), den = fma(ca.x, lo, hi);
    const double z = num * rcp(den);  // |z| <= 2^-8
    const double z2 = z * z;
    const double p = fma(z2, fma(z2, 0.2, -1.0 / 3.0), 1.0);
    // swap: atan(t) = pi/2 - atan(1/t)  ->  res = base -+ (atan c + z p), one FMA either way
    const double sg = swap ? -1.0 : 1.0, base = swap ? 1.5707963267948966 : 0.0;
    const double r = fma(z, p, ca.y);
    return copysign_i(fma(sg, r, base), n);
}

// atanh(n/d) for |n| < d with (d+|n|)/(d-|n|) < 2^16.  Branch-free.   13 FP64 + 2 MUFU
// The bin is chosen in the ratio domain q = (d+|n|)/(d-|n|) (so that the exponent of q does the
// coarse part of the logarithm), the reduction is done in the u = n/d domain against
// c' = (c-1)/(c+1), atanh(c') = 1/2 ln(c): both FMAs below see the exact n and d.
// The host packer (lh_pack.cpp) routes every lens whose ellipticity could push q past the table
// into the CLS_EXTREME class, which does not come through here; the index is clamped all the same.
LH_HD double atanh_nd(double n, double d, const double2 *__restrict__ tab) {
    const double an = fabs_i(n);                        // odd symmetry: q >= 1
    const double a = d + an, b = d - an;
    const double q0 = a * rcp_seed(b);                  // q to 1e-6
    const int hr = hi32(q0) + 0x2000;                   // q rounded to 6 mantissa bits = c
    const int j = max(0, min((hr >> 14) - (1023 << 6), LN_N - 1));
    const double2 ca = tab[j];                          // {c', atanh c'}
    const double num = fma(-ca.x, d, an), den = fma(-ca.x, an, d);
    const double s = num * rcp(den);                    // |s| <= 2^-8
    const double s2 = s * s;
    const double p = fma(s2, fma(s2, 0.2, 1.0 / 3.0), 1.0);
    return copysign_i(fma(s, p, ca.y), n);
}

// host: fill the tables (libm, correctly rounded enough: they are constants of the library)
inline void fill_math_tables(MathTables &T) {
    for (int i = 0; i <= ATAN_N; ++i) {
        const double c = (double)i / ATAN_N;
        T.at[i] = make_double2(c, (double)atanl((long double)c));
    }
    for (int j = 0; j < LN_N; ++j) {
        const int e = j / LN_PER_OCT, m = j % LN_PER_OCT;
        const long double c = std::ldexp(1.0L + (long double)m / LN_PER_OCT, e);
        const double cp = (double)((c - 1.0L) / (c + 1.0L));
        T.ah[j] = make_double2(cp, (double)atanhl((long double)cp));
    }
}

}  // namespace lh
