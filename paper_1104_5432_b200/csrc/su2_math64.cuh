// su2_math64.cuh — fp64 elementary functions of the heat-bath draw, specialised to their
// arguments. CUDA path only; shares nothing with oracle/ (which calls libm).
//
// In the fp64 kernel the CUDA library's log, cospi, sincospi and rsqrt were ~450 of the 940
// instructions per link update: they are general (any double, specials, denormals, 1 ulp) and
// each materialises ~10 polynomial constants with two UMOVs apiece. The arguments here are
// much narrower: the logs and angles are functions of one 32-bit Philox word [R5], so the
// range reduction is exact integer arithmetic on that word, and the square roots act on
// normal numbers in [1e-300, 1e3]. Each function below is accurate to a few 1e-16 (absolute
// for sin/cos, relative for log and rsqrt); the link tolerance is 1e-12.
//
//   log_uniform(w)      ln((w + 1/2) 2^-32)      table (128 x {1/c, ln c}, L1-resident) + degree-7 log1p
//   cos2_2pi_uniform(w) cos^2(2 pi (w + 1/2) 2^-32)   fold to (0, pi/4), one sine polynomial
//   sincos_2pi_uniform  sin, cos of the same angle     octant fold, sine + cosine polynomial
//   rsqrt_n(x)          1/sqrt(x), x normal            MUFU.RSQ64H + one cubic iteration
//   sqrt0_n(x)          sqrt(x), x >= 0                 x * rsqrt_n(max(x, 1e-300))
//
// All are __host__ __device__ so that a host harness can check them against libm.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace su2 {
namespace m64 {

#if defined(__CUDA_ARCH__)
#define SU2_M64_FMA(a, b, c) fma((a), (b), (c))
__device__ __forceinline__ int hi_word(double x) { return __double2hiint(x); }
__device__ __forceinline__ int lo_word(double x) { return __double2loint(x); }
__device__ __forceinline__ double from_words(int hi, int lo) { return __hiloint2double(hi, lo); }
#else
#define SU2_M64_FMA(a, b, c) __builtin_fma((a), (b), (c))
inline int hi_word(double x)
{
    uint64_t b;
    memcpy(&b, &x, 8);
    return (int)(b >> 32);
}
inline int lo_word(double x)
{
    uint64_t b;
    memcpy(&b, &x, 8);
    return (int)(uint32_t)b;
}
inline double from_words(int hi, int lo)
{
    const uint64_t b = ((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo;
    double x;
    memcpy(&x, &b, 8);
    return x;
}
#endif

struct __align__(16) LogEntry {
    double cinv, logc;  // ~1/c_j and -ln(cinv) of that double
};
constexpr int kLogEntries = 128;

// Polynomial constants live in constant memory: ptxas then reads two of them with one
// LDCU.128 instead of building each from two 32-bit immediates.
struct Coef {
    double log1p_q[6];  // log1p(r) = r + r^2 (q0 + q1 r + ... + q5 r^5)
    double sin_c[7];    // sin(x) = x (1 + z (c0 + c1 z + ... + c6 z^6)), z = x^2, |x| < pi/4
    double cos_c[8];    // cos(x) = 1 + z (c0 + ... + c7 z^7)
    double ln2;
    double two_pi_2m32;  // 2 pi 2^-32
    double pi_2m32;      //   pi 2^-32
};
#define SU2_M64_COEF_INIT                                                                                        \
    {                                                                                                            \
        {-1.0 / 2, 1.0 / 3, -1.0 / 4, 1.0 / 5, -1.0 / 6, 1.0 / 7},                                               \
            {-1.0 / 6, 1.0 / 120, -1.0 / 5040, 1.0 / 362880, -1.0 / 39916800, 1.0 / 6227020800.0,                \
             -1.0 / 1307674368000.0},                                                                            \
            {-1.0 / 2, 1.0 / 24, -1.0 / 720, 1.0 / 40320, -1.0 / 3628800, 1.0 / 479001600, -1.0 / 87178291200.0, \
             1.0 / 20922789888000.0},                                                                            \
            0.693147180559945309417232121458, 6.283185307179586476925286766559 / 4294967296.0,                   \
            3.141592653589793238462643383279 / 4294967296.0                                                      \
    }
#if defined(__CUDACC__)
static __constant__ Coef kCoef = SU2_M64_COEF_INIT;
#endif
#if defined(__CUDA_ARCH__)
#define SU2_M64_K kCoef
#else
static const Coef kCoefHost = SU2_M64_COEF_INIT;
#define SU2_M64_K kCoefHost
#endif

// ln u, u = (w + 1/2) 2^-32 [R5], given as the double `u` (exact). u = 2^e m with
// m in [sqrt(1/2), sqrt(2)); m c_inv = 1 + r with |r| <= 2^-8 (exact in the FMA);
// ln u = e ln2 + ln c + log1p(r). For u -> 1: e = 0, c = 1, and the result is the
// polynomial alone (relative accuracy kept).
__host__ __device__ __forceinline__ double log_uniform(double u, const LogEntry* __restrict__ tab)
{
    const int t = hi_word(u) + (0x3FF00000 - 0x3FE6A09E);
    const int e = (t >> 20) - 0x3FF;
    const int frac = t & 0x000FFFFF;
    const double m = from_words(frac + 0x3FE6A09E, lo_word(u));
#if defined(__CUDA_ARCH__)
    // The 2 KB table is read through L1 (ld.global.nc, one 16-byte load): measured faster than
    // a per-CTA shared-memory copy, whose fill + barrier delays the CTA's first link loads
    // (profiles/r01d.md).
    const double2 le2 = __ldg((const double2*)(tab + (frac >> 13)));
    const LogEntry le = {le2.x, le2.y};
#else
    const LogEntry le = tab[frac >> 13];
#endif
    const double r = SU2_M64_FMA(m, le.cinv, -1.0);
    const double* q = SU2_M64_K.log1p_q;
    double p = SU2_M64_FMA(q[5], r, q[4]);
    p = SU2_M64_FMA(p, r, q[3]);
    p = SU2_M64_FMA(p, r, q[2]);
    p = SU2_M64_FMA(p, r, q[1]);
    p = SU2_M64_FMA(p, r, q[0]);
    const double big = SU2_M64_FMA((double)e, SU2_M64_K.ln2, le.logc);
    return SU2_M64_FMA(r * r, p, r) + big;
}

// sin(x)/x - 1 and cos(x) - 1 as z * polynomial(z), z = x^2, |x| <= pi/4 (Taylor; the first
// neglected terms are x^16/17! < 6e-17 and x^18/18! < 3e-18)
__host__ __device__ __forceinline__ double sin_poly(double x, double z)
{
    const double* c = SU2_M64_K.sin_c;
    double p = SU2_M64_FMA(c[6], z, c[5]);
    p = SU2_M64_FMA(p, z, c[4]);
    p = SU2_M64_FMA(p, z, c[3]);
    p = SU2_M64_FMA(p, z, c[2]);
    p = SU2_M64_FMA(p, z, c[1]);
    p = SU2_M64_FMA(p, z, c[0]);
    return SU2_M64_FMA(x * z, p, x);
}
__host__ __device__ __forceinline__ double cos_poly(double z)
{
    const double* c = SU2_M64_K.cos_c;
    double p = SU2_M64_FMA(c[7], z, c[6]);
    p = SU2_M64_FMA(p, z, c[5]);
    p = SU2_M64_FMA(p, z, c[4]);
    p = SU2_M64_FMA(p, z, c[3]);
    p = SU2_M64_FMA(p, z, c[2]);
    p = SU2_M64_FMA(p, z, c[1]);
    p = SU2_M64_FMA(p, z, c[0]);
    return SU2_M64_FMA(z, p, 1.0);
}

// cos^2(2 pi u), u = (w + 1/2) 2^-32. In units of 2^-32 turns the angle is w + 1/2:
// cos^2 has period 2^31 and is even about 0 and 2^30, and cos^2(2^30 - a) = sin^2(a):
// two mirror folds (bitwise complements, exact) leave a in (0, 2^29), i.e. x in (0, pi/4).
__host__ __device__ __forceinline__ double cos2_2pi_uniform(uint32_t w)
{
    const uint32_t m1 = (uint32_t)((int32_t)(w << 1) >> 31);           // all ones if bit 30
    const uint32_t v1 = (w ^ m1) & 0x3FFFFFFFu;                        // angle in (0, pi/2)
    const uint32_t m2 = (uint32_t)((int32_t)(v1 << 2) >> 31);          // all ones if bit 29: use sin^2(pi/2 - .)
    const uint32_t v2 = (v1 ^ m2) & 0x1FFFFFFFu;
    const double x = SU2_M64_FMA((double)v2, SU2_M64_K.two_pi_2m32, SU2_M64_K.pi_2m32);
    const double s = sin_poly(x, x * x);
    const double s2 = s * s;
    return m2 ? s2 : 1.0 - s2;
}

// sin and cos of 2 pi u: octant o = w >> 29; odd octants are mirrored; (s, c) of the
// reduced angle in (0, pi/4) are swapped and signed per octant.
__host__ __device__ __forceinline__ void sincos_2pi_uniform(uint32_t w, double* sn, double* cs)
{
    const uint32_t o = w >> 29;
    const uint32_t mm = 0u - (o & 1u);
    const uint32_t v = (w ^ mm) & 0x1FFFFFFFu;
    const double x = SU2_M64_FMA((double)v, SU2_M64_K.two_pi_2m32, SU2_M64_K.pi_2m32);
    const double z = x * x;
    const double s = sin_poly(x, z), c = cos_poly(z);
    const bool swap = ((o + 1u) & 2u) != 0u;       // octants 1, 2, 5, 6
    const double a = swap ? c : s, b = swap ? s : c;
    const int sneg = (int)((o & 4u) << 29);        // sin < 0 in octants 4..7
    const int cneg = (int)(((o + 2u) & 4u) << 29); // cos < 0 in octants 2..5
    *sn = from_words(hi_word(a) ^ sneg, lo_word(a));
    *cs = from_words(hi_word(b) ^ cneg, lo_word(b));
}

// 1/sqrt(x) for normal x (no zero, infinity, NaN, denormal): seed with ~20 good bits, then
// y (1 + e/2 + 3 e^2/8), e = 1 - x y^2: error O(e^3) < 1e-18, plus the rounding of 3 operations.
__host__ __device__ __forceinline__ double rsqrt_n(double x)
{
    double y;
#if defined(__CUDA_ARCH__)
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
#else
    y = from_words(hi_word(1.0 / __builtin_sqrt(from_words(hi_word(x), 0))), 0);  // stand-in for MUFU.RSQ64H
#endif
    const double e = SU2_M64_FMA(-(x * y), y, 1.0);
    const double t = SU2_M64_FMA(e, 0.375, 0.5);
    return SU2_M64_FMA(y * e, t, y);
}

// sqrt(x) for x >= 0 as x * rsqrt(x); the clamp keeps rsqrt_n's argument normal, so that
// sqrt0_n(0) = 0 exactly and a denormal x gives a value below 1e-150 instead of a NaN.
__host__ __device__ __forceinline__ double sqrt0_n(double x)
{
#if defined(__CUDA_ARCH__)
    return x * rsqrt_n(fmax(x, 1e-300));
#else
    return x * rsqrt_n(x > 1e-300 ? x : 1e-300);
#endif
}

}  // namespace m64
}  // namespace su2
