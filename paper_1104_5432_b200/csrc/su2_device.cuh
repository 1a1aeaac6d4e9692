// su2_device.cuh — device-side building blocks of the SU(2) heat-bath path (sm_100a).
//
// Written from DESIGN.md §3 (readings [R1]..[R14]); shares nothing with oracle/.
//   [R1] quaternion algebra          [R5] Philox4x32-10 keying + uniform rules
//   [R3] staple sum                  [R6] Kennedy-Pendleton draw
//   [R7] direction + composition     [R9] Shoemake hot start
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "su2_math64.cuh"

namespace su2 {

// ---------------------------------------------------------------- geometry
// Device layout: array (p,mu) holds the V/2 links U_mu(x) of the
// sites with parity p, element h = s>>1 = hx + nxh*(y + Ny*(z + Nz*t)), hx = x>>1.
struct Geom {
    int n[4];        // Nx, Ny, Nz, Nt
    int nxh;         // Nx/2
    int sy, sz, st;  // strides of y, z, t in half-index units: nxh, nxh*Ny, nxh*Ny*Nz
    uint32_t vh;     // V/2
    int tile;        // tiled launch: which tile shape (su2_launch.h kTiles), -1 = linear launch
    int nb[4];       // tiled launch: number of tiles along hx, y, z, t
    int wup[4];      // half-index delta of +mu at the upper boundary: -(N-1)*stride  (x: -(nxh-1))
    uint32_t zmagic; // ceil(2^32 / nb[2]): blockIdx.z -> (bz, bt) without a division
    int tloop;       // heat-bath tiled launch: consecutive t-tiles one CTA walks through (divides nb[3])
    // time slab of a lattice split over GPUs: only the slices t_lo <= t < t_lo + nt_upd
    // are updated and measured, the others are halo copies. Whole lattice: t_lo = 0, nt_upd = Nt.
    int t_lo, nt_upd;
};

// ---------------------------------------------------------------- sites and neighbours
struct Site {
    int hx, y, z, t;  // hx = x>>1
};

// half-index deltas of the 8 neighbours; r = low bit of x
struct Nbr {
    int up[4], dn[4];
};
__device__ __forceinline__ Nbr neighbours(const Geom& g, const Site& c, int r)
{
    Nbr d;
    d.up[0] = r ? ((c.hx + 1 == g.nxh) ? g.wup[0] : 1) : 0;
    d.dn[0] = r ? 0 : ((c.hx == 0) ? -g.wup[0] : -1);
    d.up[1] = (c.y + 1 == g.n[1]) ? g.wup[1] : g.sy;
    d.dn[1] = (c.y == 0) ? -g.wup[1] : -g.sy;
    d.up[2] = (c.z + 1 == g.n[2]) ? g.wup[2] : g.sz;
    d.dn[2] = (c.z == 0) ? -g.wup[2] : -g.sz;
    d.up[3] = (c.t + 1 == g.n[3]) ? g.wup[3] : g.st;
    d.dn[3] = (c.t == 0) ? -g.wup[3] : -g.st;
    return d;
}

// Tiled launch: one CTA = 2^LHX x 2^LY x 2^LZ x 2^LT threads of a 4-D tile; grid =
// (nb0[*k], nb1, nb2*nb3), dispatched x fastest, then y, then z, then t: roughly memory
// order. (Sweeping z-slabs through all t first, to shorten the t-neighbour reuse
// distance in L2, was measured and made no difference: profiles/r01b.md.)
template <int LHX, int LY, int LZ, int LT>
__device__ __forceinline__ Site tile_site(const Geom& g, uint32_t bzt, uint32_t bx = blockIdx.x)
{
    const uint32_t bt = (g.nb[2] == 1) ? bzt : __umulhi(bzt, g.zmagic);
    const uint32_t bz = bzt - bt * (uint32_t)g.nb[2];
    const int tid = threadIdx.x;
    Site c;
    c.hx = (int)(bx << LHX) + (tid & ((1 << LHX) - 1));
    c.y = (int)(blockIdx.y << LY) + ((tid >> LHX) & ((1 << LY) - 1));
    c.z = (int)(bz << LZ) + ((tid >> (LHX + LY)) & ((1 << LZ) - 1));
    c.t = (int)(bt << LT) + (tid >> (LHX + LY + LZ));
    return c;
}

// ---------------------------------------------------------------- quaternions
template <typename Real>
struct Quat {
    Real a0, a1, a2, a3;
};

template <typename Real>
struct LinkPtr;  // storage element type of one link
template <>
struct LinkPtr<float> {
    typedef float4 type;
};
struct __align__(32) double4a {
    double x, y, z, w;
};
template <>
struct LinkPtr<double> {
    typedef double4a type;
};

// Load path of the link reads: ".nc" (read-only data path, L1-cached), "" (plain ld.global)
// or ".cg" (L2 only) - the sm_100a analogue of the paper's texture-vs-global-memory study
// (PAPER.md:97); measured in profiles/r01c.md, ".nc" kept.
#ifndef HB_LD
#define HB_LD ".nc"
#endif
// Loads go through the non-coherent path: within one sub-step no array that is
// read is written, and L1 is invalidated at every launch.
__device__ __forceinline__ Quat<float> ldq(const float4* p)
{
    Quat<float> q;
    // volatile: keeps the 18 staple loads of a thread in program order, ahead of the arithmetic
    asm volatile("ld.global" HB_LD ".v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(q.a0), "=f"(q.a1), "=f"(q.a2), "=f"(q.a3)
                 : "l"(p));
    return q;
}
__device__ __forceinline__ Quat<double> ldq(const double4a* p)
{
    Quat<double> q;
    // one 256-bit load per link (sm_100+)
    asm volatile("ld.global" HB_LD ".v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(q.a0), "=d"(q.a1), "=d"(q.a2), "=d"(q.a3)
                 : "l"(p));
    return q;
}
// The updated link is not read again in its own sub-step: streaming store (evict-first in L2).
#ifndef HB_ST
#define HB_ST ".cs"
#endif
// L2-only loads (no L1 allocation): streams that are read once (the Polyakov lines).
__device__ __forceinline__ Quat<float> ldq_cg(const float4* p)
{
    Quat<float> q;
    asm volatile("ld.global.cg.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(q.a0), "=f"(q.a1), "=f"(q.a2), "=f"(q.a3)
                 : "l"(p)
                 : "memory");
    return q;
}
__device__ __forceinline__ Quat<double> ldq_cg(const double4a* p)
{
    Quat<double> q;
    asm volatile("ld.global.cg.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(q.a0), "=d"(q.a1), "=d"(q.a2), "=d"(q.a3)
                 : "l"(p)
                 : "memory");
    return q;
}
// Loads of the links the PRECEDING sub-step wrote, issued after griddepcontrol.wait: ordinary
// (coherent, L1-allocating) ld.global, not the read-only .nc path - the array was written while this kernel's
// CTAs were already being scheduled. An ordinary load after the wait observes the primary grid's flushed
// writes; no earlier kernel's copy can linger in L1, which is invalidated at every launch, and the kernel
// launched in between never reads that array. U_mu on the other parity is the most re-used operand of a tile
// (6 reads per link): through L2 only (.cg, round 1) these loads cost 14 % more L2 -> SM traffic per launch
// (ncu: 2.24 against 1.93 GB at 64^4 fp32, profiles/r02b.md).
__device__ __forceinline__ Quat<float> ldq_dep(const float4* p)
{
    Quat<float> q;
    asm volatile("ld.global.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(q.a0), "=f"(q.a1), "=f"(q.a2), "=f"(q.a3)
                 : "l"(p)
                 : "memory");
    return q;
}
__device__ __forceinline__ Quat<double> ldq_dep(const double4a* p)
{
    Quat<double> q;
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(q.a0), "=d"(q.a1), "=d"(q.a2), "=d"(q.a3)
                 : "l"(p)
                 : "memory");
    return q;
}
// Programmatic dependent launch: wait for the preceding kernel of the
// stream to finish and flush; then allow the next kernel's CTAs to be scheduled.
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ void stq(float4* p, const Quat<float>& q)
{
    asm volatile("st.global" HB_ST ".v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(q.a0), "f"(q.a1), "f"(q.a2), "f"(q.a3)
                 : "memory");
}
__device__ __forceinline__ void stq(double4a* p, const Quat<double>& q)
{
    asm volatile("st.global" HB_ST ".v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(q.a0), "d"(q.a1), "d"(q.a2), "d"(q.a3)
                 : "memory");
}

// [R1] c = op(a) * op(b), op = dagger when DA / DB:
//   c0 = a0 b0 - a.b ; cvec = a0 b + b0 a - a x b ; dagger flips the vector part.
// Written as FMA chains (4 mul + 12 fma, sign flips ride on the FMA operands).
__device__ __forceinline__ float fmad(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fmad(double a, double b, double c) { return fma(a, b, c); }

template <bool DA, bool DB, typename Real>
__device__ __forceinline__ Quat<Real> qmul(const Quat<Real>& a, const Quat<Real>& b)
{
    const Real a1 = DA ? -a.a1 : a.a1, a2 = DA ? -a.a2 : a.a2, a3 = DA ? -a.a3 : a.a3;
    const Real b1 = DB ? -b.a1 : b.a1, b2 = DB ? -b.a2 : b.a2, b3 = DB ? -b.a3 : b.a3;
    Quat<Real> c;
    c.a0 = fmad(-a3, b3, fmad(-a2, b2, fmad(-a1, b1, a.a0 * b.a0)));
    c.a1 = fmad(a3, b2, fmad(-a2, b3, fmad(b.a0, a1, a.a0 * b1)));
    c.a2 = fmad(a1, b3, fmad(-a3, b1, fmad(b.a0, a2, a.a0 * b2)));
    c.a3 = fmad(a2, b1, fmad(-a1, b2, fmad(b.a0, a3, a.a0 * b3)));
    return c;
}
// acc += op(a) * op(b)   (16 fma)
template <bool DA, bool DB, typename Real>
__device__ __forceinline__ void qmac(Quat<Real>& acc, const Quat<Real>& a, const Quat<Real>& b)
{
    const Real a1 = DA ? -a.a1 : a.a1, a2 = DA ? -a.a2 : a.a2, a3 = DA ? -a.a3 : a.a3;
    const Real b1 = DB ? -b.a1 : b.a1, b2 = DB ? -b.a2 : b.a2, b3 = DB ? -b.a3 : b.a3;
    acc.a0 = fmad(-a3, b3, fmad(-a2, b2, fmad(-a1, b1, fmad(a.a0, b.a0, acc.a0))));
    acc.a1 = fmad(a3, b2, fmad(-a2, b3, fmad(b.a0, a1, fmad(a.a0, b1, acc.a1))));
    acc.a2 = fmad(a1, b3, fmad(-a3, b1, fmad(b.a0, a2, fmad(a.a0, b2, acc.a2))));
    acc.a3 = fmad(a2, b1, fmad(-a1, b2, fmad(b.a0, a3, fmad(a.a0, b3, acc.a3))));
}
// scalar part only of a * b^dagger  ( = 4-vector dot product )
template <typename Real>
__device__ __forceinline__ Real qdot(const Quat<Real>& a, const Quat<Real>& b)
{
    return a.a0 * b.a0 + a.a1 * b.a1 + a.a2 * b.a2 + a.a3 * b.a3;
}

// ---------------------------------------------------------------- Philox4x32-10 [R5]
struct Words {
    uint32_t w0, w1, w2, w3;
};
__device__ __forceinline__ Words philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                               uint32_t k1)
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return {c0, c1, c2, c3};
}
// counter = (site, sweep_idx, (purpose<<8)|(parity<<2)|mu, call n), key = seed
__device__ __forceinline__ Words draw(uint64_t seed, uint32_t s, uint32_t sweep, uint32_t tag, uint32_t n)
{
    return philox4x32_10(s, sweep, tag, n, (uint32_t)seed, (uint32_t)(seed >> 32));
}
// The 10 round keys depend on the seed only: the launcher expands them once on the
// host (same Weyl sequence as above) so that the hot kernel reads them as constants.
struct __align__(16) RoundKeys {
    uint32_t k[20];  // k[2r] = key word 0 of round r, k[2r+1] = key word 1
};
__host__ __device__ inline RoundKeys expand_keys(uint64_t seed)
{
    RoundKeys rk;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        rk.k[2 * r] = k0;
        rk.k[2 * r + 1] = k1;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return rk;
}
__device__ __forceinline__ Words philox_keyed(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const RoundKeys& rk)
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        c0 = hi1 ^ c1 ^ rk.k[2 * r];
        c1 = lo1;
        c2 = hi0 ^ c3 ^ rk.k[2 * r + 1];
        c3 = lo0;
    }
    return {c0, c1, c2, c3};
}

// ---------------------------------------------------------------- per-precision math
template <typename Real>
struct M;
template <>
struct M<float> {
    // fp32 rule: u = (2*(w>>9)+1) * 2^-24, exact, strictly inside (0,1).
    // Built from the bits: f = 1.m in [1,2) with m = w>>9, then u = f - (1 - 2^-24) (exact).
    static __device__ __forceinline__ float one_two(uint32_t w) { return __uint_as_float(0x3F800000u | (w >> 9)); }
    static __device__ __forceinline__ float uniform(uint32_t w) { return one_two(w) - 0.99999994f; }
    static __device__ __forceinline__ float log(float x) { return logf(x); }
    static __device__ __forceinline__ float exp(float x) { return expf(x); }
    static __device__ __forceinline__ float sqrt(float x) { return sqrtf(x); }
    static __device__ __forceinline__ float rcp(float x) { return 1.0f / x; }
    // MUFU approximations (<= 2 ulp): the fp32 link tolerance is 1e-5
    static __device__ __forceinline__ float rsqrt(float x)
    {
        float r;
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
        return r;
    }
    static __device__ __forceinline__ float sqrt0(float x)  // x >= 0
    {
        float r;
        asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
        return r;
    }
    static __device__ __forceinline__ float lg2(float x)
    {
        float r;
        asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
        return r;
    }
    // angle 2 pi u - pi in (-pi, pi): (f - 1.5) is exact, one rounding in the FMA
    static __device__ __forceinline__ float angle(uint32_t w)
    {
        return fmaf(one_two(w) - 1.5f, 6.2831855f, 3.7450704e-7f);  // 2 pi (u - 1/2), 2 pi 2^-24
    }
    static __device__ __forceinline__ float cos2pi(float x) { return cospif(2.0f * x); }
    static __device__ __forceinline__ void sincos2pi(float x, float* s, float* c) { sincospif(2.0f * x, s, c); }
    // sin, cos of 2 pi u(w) by MUFU on the reduced angle: sin(2 pi u) = -sin(2 pi u - pi)
    static __device__ __forceinline__ void sincos2pi_word(uint32_t w, float* s, float* c)
    {
        const float x = angle(w);
        *s = -__sinf(x);
        *c = -__cosf(x);
    }
    // [R6] delta of one KP trial, MUFU lg2/cos (abs. error of delta <= ~4e-7/alpha)
    static __device__ __forceinline__ float kp_delta(const Words& w, float inv_alpha, const m64::LogEntry*)
    {
        const float cs = __cosf(angle(w.w1));  // cos(2 pi R' - pi); only its square is used
        const float g2 = fmaf(cs * cs, lg2(uniform(w.w2)), lg2(uniform(w.w0)));
        return g2 * (-0.6931472f * inv_alpha);
    }
    // The radius sqrt(delta(2-delta)) amplifies the absolute error of delta by 1/radius:
    // where that would exceed ~1e-6 (radius^2 < 0.12/alpha^2, probability ~1e-4) the
    // accepted trial is recomputed with the accurate logf/cospif. So is
    // every accepted trial at alpha < 2, where the error of delta itself (~4e-7/alpha,
    // and |ln R''| times the MUFU cosine error) is no longer small against 1e-5.
    static __device__ __forceinline__ float kp_delta_refined(const Words& w, float inv_alpha, float delta)
    {
        if (delta * (2.0f - delta) < 0.12f * inv_alpha * inv_alpha || inv_alpha > 0.5f) {
            const float cs = cospif(2.0f * uniform(w.w1));
            delta = -(logf(uniform(w.w0)) + cs * cs * logf(uniform(w.w2))) * inv_alpha;
        }
        return delta;
    }
    static __device__ __forceinline__ float tiny() { return 1e-20f; }
};
template <>
struct M<double> {
    // fp64 rule: u = (w + 0.5) * 2^-32, exact
    static __device__ __forceinline__ double uniform(uint32_t w)
    {
        return fma((double)w, 1.0 / 4294967296.0, 1.0 / 8589934592.0);
    }
    static __device__ __forceinline__ double log(double x) { return ::log(x); }
    static __device__ __forceinline__ double exp(double x) { return ::exp(x); }
    static __device__ __forceinline__ double sqrt(double x) { return ::sqrt(x); }
    static __device__ __forceinline__ double rcp(double x) { return 1.0 / x; }
    // su2_math64.cuh: functions specialised to the arguments of this path
    static __device__ __forceinline__ double rsqrt(double x) { return m64::rsqrt_n(x); }  // x normal
    static __device__ __forceinline__ double sqrt0(double x) { return m64::sqrt0_n(x); }  // x >= 0
    static __device__ __forceinline__ double cos2pi(double x) { return cospi(2.0 * x); }
    static __device__ __forceinline__ void sincos2pi(double x, double* s, double* c) { sincospi(2.0 * x, s, c); }
    static __device__ __forceinline__ void sincos2pi_word(uint32_t w, double* s, double* c)
    {
        m64::sincos_2pi_uniform(w, s, c);
    }
    // [R6] delta of one KP trial; `tab` = the log table in shared memory
    static __device__ __forceinline__ double kp_delta(const Words& w, double inv_alpha, const m64::LogEntry* tab)
    {
        const double c2 = m64::cos2_2pi_uniform(w.w1);
        const double l0 = m64::log_uniform(uniform(w.w0), tab), l2 = m64::log_uniform(uniform(w.w2), tab);
        return -fma(c2, l2, l0) * inv_alpha;
    }
    static __device__ __forceinline__ double kp_delta_refined(const Words&, double, double delta) { return delta; }
    static __device__ __forceinline__ double tiny() { return 1e-30; }
};

// Device-resident loop state of su2_run: a captured CUDA graph of one
// step is replayed n times without touching its kernel parameters, so what changes from
// step to step lives here. Written by set_run_state_kernel and advanced by the last
// kernel of every step.
struct __align__(32) RunState {
    double inv_beta;
    uint32_t sweep;   // sweep_idx of the current step
    uint32_t index;   // step number: results go to out[2*index], out[2*index+1]
    double* out;      // [device] 2 doubles per step
    uint64_t pad;
};
// Every thread of a sub-step reads (inv_beta, sweep). With one copy the 2^18 warps of a 64^4
// launch would all address a single L2 sector, so the state is replicated: a CTA reads copy (CTA id mod kRunCopies), the last kernel
// of a step advances all copies. Copy 0 is the one whose `out` and `index` are used.
constexpr int kRunCopies = 1024;
__device__ __forceinline__ const RunState* run_state_copy(const RunState* base)
{
    return base + ((blockIdx.x + 37u * blockIdx.y + 101u * blockIdx.z) & (uint32_t)(kRunCopies - 1));
}
// (inv_beta, sweep) in one 16-byte L2 load
__device__ __forceinline__ void ld_run_state(const RunState* p, double& inv_beta, uint32_t& sweep)
{
    uint64_t a, b;
    asm volatile("ld.global.cg.v2.u64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
    inv_beta = __longlong_as_double((long long)a);
    sweep = (uint32_t)b;
}
// per-replica inputs of a batched launch
struct __align__(16) RepParams {
    double inv_beta;
    uint64_t seed;
};
// what a thread needs to know about its replica; all zero for a single lattice
struct RepCtx {
    uint32_t rep;   // replica index
    uint32_t hoff;  // rep * rep_stride: added to every link index
    uint32_t k0, k1;  // Philox key words when the keys are not the launch's expanded ones
};

// per-launch constants of the heat-bath kernels. The array bases are resolved on the
// host so that a link address is base + 16*(32-bit index): one IMAD.WIDE per load.
template <typename Real>
struct __align__(16) HbParams {
    RoundKeys rk;
    const typename LinkPtr<Real>::type* same[4];  // U_nu on the parity being updated
    const typename LinkPtr<Real>::type* oppo[4];  // U_nu on the other parity
    typename LinkPtr<Real>::type* out;            // U_mu on the parity being updated
    double* epart;                                // fused plaquette: one partial per CTA (MEAS kernels)
    const RunState* state;                        // non-null inside su2_run: sweep and 1/beta come from here
    Real inv_beta;
    uint32_t sweep;
    Real creutz_below;  // [R15] ALT kernels: Creutz's draw where alpha < this (0 = never, +inf = always)
    // replica batch (ALT kernels only): R configurations of the same geometry, one after
    // the other in memory, updated by one launch; replica index = leading part of the grid
    const RepParams* reps;  // [device] per-replica 1/beta and seed; NULL = single lattice
    uint32_t rep_stride;    // links of one configuration: 8 * V/2
    uint32_t nzt;           // tiled launch: CTAs along grid z per replica (nb2 * nb3)
    uint32_t epart_stride;  // fused-plaquette partials per replica (3 * CTAs of one replica)
    // time slab (ALT kernels only): Philox is keyed by the GLOBAL site, and the links of
    // the first / last interior slice are also stored into the neighbouring slab's halo (peer memory)
    uint32_t s_off;                        // global site index - local site index
    typename LinkPtr<Real>::type* peer_lo;  // array (p,mu) of the slab below (NULL = not a slab)
    typename LinkPtr<Real>::type* peer_hi;  // array (p,mu) of the slab above
    int d_lo, d_hi;                        // own link index -> index of its halo copy in peer_lo / peer_hi
    int t_first, t_last;                   // first / last interior slice (-1 = not a slab)
};

// [R9] Shoemake: uniform unit quaternion from three uniforms
template <typename Real>
__device__ __forceinline__ Quat<Real> haar_from_words(const Words& w)
{
    const Real u1 = M<Real>::uniform(w.w0), u2 = M<Real>::uniform(w.w1), u3 = M<Real>::uniform(w.w2);
    const Real r1 = M<Real>::sqrt((Real)1 - u1), r2 = M<Real>::sqrt(u1);
    Real s2, c2, s3, c3;
    M<Real>::sincos2pi(u2, &s2, &c2);
    M<Real>::sincos2pi(u3, &s3, &c3);
    return {r1 * s2, r1 * c2, r2 * s3, r2 * c3};
}

// ---------------------------------------------------------------- block reduction
// warp shuffle + fixed-order block tree in fp64; valid result in thread 0.
// `red` must hold blockDim.x/32 doubles.
__device__ __forceinline__ double block_sum(double v, double* red)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double tot = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < nw; ++i) tot += red[i];
    __syncthreads();
    return tot;
}

// Same without the trailing barrier: for one use at the end of a kernel. The per-thread value is converted
// to fp64 BEFORE the first shuffle (north_star: reductions "accumulated in fp64"; round 1 summed the 32 lanes
// of an fp32 kernel in fp32 - 5 shuffles fewer in 3 of the 8 kernels of a sweep, not measurable).
__device__ __forceinline__ double block_sum_end(double v, double* red)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double tot = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < nw; ++i) tot += red[i];
    return tot;
}

}  // namespace su2
