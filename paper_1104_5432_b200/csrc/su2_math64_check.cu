// su2_math64_check.cu — host harness for su2_math64.cuh (built and run by
// tests/test_math64_cpu.py; not part of libsu2hb.so). Compares each function with the
// C library in long double over the edge words and a stream of pseudo-random words and
// prints the worst errors as one line of "name value" pairs.
#include <cmath>
#include <cstdio>
#include <cstdlib>

#include "su2_math64.cuh"
using namespace su2::m64;

static const LogEntry tab[kLogEntries] = {
#include "su2_log_table.inc"
};

int main(int argc, char** argv)
{
    const long n = argc > 1 ? atol(argv[1]) : 4000000L;
    const long double PI = 3.141592653589793238462643383279502884L;
    double log_rel = 0, cos2_abs = 0, sincos_abs = 0, rsqrt_rel = 0, sqrt0_rel = 0;
    uint64_t st = 88172645463325252ull;  // xorshift64: test inputs only
    for (long i = 0; i < n; ++i) {
        st ^= st << 13; st ^= st >> 7; st ^= st << 17;
        uint32_t w = (uint32_t)(st >> 16);
        if (i < 64) w = (i < 32) ? (uint32_t)i : 0xFFFFFFFFu - (uint32_t)(i - 32);        // both ends of (0,1)
        else if (i < 4096) w = ((uint32_t)(i & 7) << 29) + (uint32_t)(((i >> 3) & 1) ? -(int)(i >> 4) : (i >> 4));  // octant edges
        const double u = fma((double)w, 1.0 / 4294967296.0, 1.0 / 8589934592.0);
        const long double lu = logl((long double)u);
        log_rel = fmax(log_rel, fabs((double)((log_uniform(u, tab) - lu) / lu)));
        const long double ang = 2 * PI * (long double)u;
        const long double c2 = cosl(ang) * cosl(ang);
        cos2_abs = fmax(cos2_abs, fabs((double)(cos2_2pi_uniform(w) - c2)));
        double s, c;
        sincos_2pi_uniform(w, &s, &c);
        sincos_abs = fmax(sincos_abs, fmax(fabs((double)(s - sinl(ang))), fabs((double)(c - cosl(ang)))));
        const double x = ldexp(1.0 + u, (int)(w % 80) - 60);
        const long double rr = 1.0L / sqrtl((long double)x);
        rsqrt_rel = fmax(rsqrt_rel, fabs((double)((rsqrt_n(x) - rr) / rr)));
        // sqrt0_n over the arguments the kernel gives it: delta (2 - delta) and 1 - cos^2(theta), both in [0, 1],
        // down to the smallest positive values (u^2 ~ 1e-20) - the function M<double>::sqrt0 calls
        const double y0 = (i & 1) ? u * u : u * (2.0 - u) * 0.5;
        const long double sr = sqrtl((long double)y0);
        sqrt0_rel = fmax(sqrt0_rel, fabs((double)((sqrt0_n(y0) - sr) / sr)));
    }
    printf("log_rel %.3e cos2_abs %.3e sincos_abs %.3e rsqrt_rel %.3e sqrt0_rel %.3e sqrt0_zero %.3e sqrt0_denormal %.3e "
           "sqrt_tiny %.17g\n",
           log_rel, cos2_abs, sincos_abs, rsqrt_rel, sqrt0_rel, sqrt0_n(0.0), sqrt0_n(4.9e-324), sqrt0_n(1e-300));
    return 0;
}
