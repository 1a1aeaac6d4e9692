// su2_heatbath.cu — init and heat-bath sub-step kernels (rows 1-6 of SURVEY.md §8(a)).
//
// One thread updates one link U_mu(x) of the sub-step's parity:
//   neighbour addressing (row 2) -> 18 vector loads + 12 quaternion products (row 3)
//   -> k, alpha (row 4) -> Philox (row 5) -> Kennedy-Pendleton loop, compose, store (row 6).
// Formulas: DESIGN.md §3 [R1]-[R9]. The paper's own kernels (texture vs global
// memory) are prior art for GT200/Fermi; here link reads are
// 128/256-bit non-coherent loads and the 2.4x neighbour reuse is served by L1
// through a compact 4-D CTA tile.
#include "su2_launch.h"

namespace su2 {

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

// The 18 links of the staple are all requested before the first product: one
// round trip to L2/HBM per thread instead of one per product.
// Array bases are uniform 64-bit pointers, element indices 32-bit (h + delta < V/2).
template <typename Real, int MU>
__device__ __forceinline__ void heatbath_site(const Geom& g, const Site& c, const HbParams<Real>& hp,
                                              int* __restrict__ err)
{
    typedef typename LinkPtr<Real>::type L;
    const int r = (c.y + c.z + c.t + hp.parity) & 1;
    const int h = c.hx + g.sy * c.y + g.sz * c.z + g.st * c.t;
    const Nbr d = neighbours(g, c, r);
    const L* o_mu = hp.oppo[MU];  // U_mu on the other parity
    const uint32_t h_up = (uint32_t)(h + d.up[MU]);

    Quat<Real> a[3], b[3], cc[3], a2[3], b2[3], c2[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const int nu = i + (i >= MU ? 1 : 0);
        const L* s_nu = hp.same[nu];
        const L* o_nu = hp.oppo[nu];
        const uint32_t h_dn = (uint32_t)(h + d.dn[nu]);
        a[i] = ldq(o_nu + h_up);                               // U_nu(x+mu)
        b[i] = ldq(o_mu + (uint32_t)(h + d.up[nu]));           // U_mu(x+nu)
        cc[i] = ldq(s_nu + (uint32_t)h);                       // U_nu(x)
        a2[i] = ldq(s_nu + (uint32_t)((int)h_up + d.dn[nu]));  // U_nu(x+mu-nu)
        b2[i] = ldq(o_mu + h_dn);                              // U_mu(x-nu)
        c2[i] = ldq(o_nu + h_dn);                              // U_nu(x-nu)
    }

    // [R5] counter = (s, sweep, (p<<2)|mu, n); the n = 0 draw does not depend on the links
    const uint32_t s = 2u * (uint32_t)h + (uint32_t)r;
    const uint32_t tag = hp.tag;
    const Words wd = philox_keyed(s, hp.sweep, tag, 0u, hp.rk);

    // [R3] staple sum, nu ascending, forward then backward, products left to right;
    // the second product of every term accumulates straight into v (FMA chains).
    Quat<Real> v = {0, 0, 0, 0};
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        qmac<false, true>(v, qmul<false, true>(a[i], b[i]), cc[i]);    // (a b^+) c^+
        qmac<false, false>(v, qmul<true, true>(a2[i], b2[i]), c2[i]);  // (a2^+ b2^+) c2
    }

    const Real k2 = v.a0 * v.a0 + v.a1 * v.a1 + v.a2 * v.a2 + v.a3 * v.a3;
    Quat<Real> u;
    if (k2 < M<Real>::tiny()) {  // [R8]
        u = haar_from_words<Real>(wd);
    } else {
        const Real rk = M<Real>::rsqrt(k2);       // 1/k
        const Real inv_alpha = rk * hp.inv_beta;  // 1/(beta k)
        // [R6] Kennedy-Pendleton
        Real delta = 0;
        uint32_t n = 1;
        for (;;) {
            const Words w = philox_keyed(s, hp.sweep, tag, n, hp.rk);
            delta = M<Real>::kp_delta(w, inv_alpha);
            const Real Rppp = M<Real>::uniform(w.w3);
            if (Rppp * Rppp <= (Real)1 - (Real)0.5 * delta) {
                delta = M<Real>::kp_delta_refined(w, inv_alpha, delta);
                break;
            }
            if (++n > 10000u) {  // unreachable for alpha >~ 1e-4; flag, keep x0 = 1
                atomicOr(err, 1);
                delta = 0;
                break;
            }
        }
        // [R7] direction on the sphere of radius sqrt(delta(2-delta)), compose with Vbar^dagger
        const Real x0 = (Real)1 - delta;
        const Real rad = M<Real>::sqrt0(fmax(delta * ((Real)2 - delta), (Real)0));
        const Real cth = (Real)1 - (Real)2 * M<Real>::uniform(wd.w0);
        const Real sth = M<Real>::sqrt0(fmax((Real)1 - cth * cth, (Real)0));
        Real sphi, cphi;
        M<Real>::sincos2pi_word(wd.w1, &sphi, &cphi);
        const Real rs = rad * sth;
        const Quat<Real> X = {x0, rs * cphi, rs * sphi, rad * cth};
        u = qmul<false, true>(X, v);  // X * v^dagger = k * (X * Vbar^dagger); k drops out below
    }
    const Real inv = M<Real>::rsqrt(u.a0 * u.a0 + u.a1 * u.a1 + u.a2 * u.a2 + u.a3 * u.a3);
    u.a0 *= inv; u.a1 *= inv; u.a2 *= inv; u.a3 *= inv;
    stq(hp.out + (uint32_t)h, u);
}

// Resident CTAs per SM that ptxas must allow: this is the register budget that lets it
// keep all 18 link loads of a thread in flight at once.
#ifndef HB_MINB_F32
#define HB_MINB_F32 8
#endif
#ifndef HB_MINB_F64
#define HB_MINB_F64 8
#endif
template <typename Real>
struct MinBlocks {
    static constexpr int value = HB_MINB_F32;
};
template <>
struct MinBlocks<double> {
    static constexpr int value = HB_MINB_F64;
};

// tiled launch: one CTA = 2^LHX x 2^LY x 2^LZ x 2^LT threads of a 4-D tile;
// grid = (nb0, nb1, nb2*nb3): x fastest, so CTAs are scheduled roughly in memory order.
template <typename Real, int MU, int LHX, int LY, int LZ, int LT>
__global__ void __launch_bounds__(1 << (LHX + LY + LZ + LT), MinBlocks<Real>::value)
    heatbath_tiled_kernel(const Geom g, const HbParams<Real> hp, int* __restrict__ err)
{
    const uint32_t bzt = blockIdx.z;
    const uint32_t bt = (g.nb[2] == 1) ? bzt : __umulhi(bzt, g.zmagic);
    const uint32_t bz = bzt - bt * (uint32_t)g.nb[2];
    const int tid = threadIdx.x;
    Site c;
    c.hx = (int)(blockIdx.x << LHX) + (tid & ((1 << LHX) - 1));
    c.y = (int)(blockIdx.y << LY) + ((tid >> LHX) & ((1 << LY) - 1));
    c.z = (int)(bz << LZ) + ((tid >> (LHX + LY)) & ((1 << LZ) - 1));
    c.t = (int)(bt << LT) + (tid >> (LHX + LY + LZ));
    heatbath_site<Real, MU>(g, c, hp, err);
}

// linear launch: thread i <-> half-index h = i; any even extents
template <typename Real, int MU>
__global__ void __launch_bounds__(kBlock)
    heatbath_linear_kernel(const Geom g, const HbParams<Real> hp, int* __restrict__ err)
{
    const uint32_t h = blockIdx.x * (uint32_t)kBlock + threadIdx.x;
    if (h >= g.vh) return;
    Site c;
    uint32_t q = h / (uint32_t)g.nxh;
    c.hx = (int)(h - q * (uint32_t)g.nxh);
    uint32_t q2 = q / (uint32_t)g.n[1];
    c.y = (int)(q - q2 * (uint32_t)g.n[1]);
    c.t = (int)(q2 / (uint32_t)g.n[2]);
    c.z = (int)(q2 - (uint32_t)c.t * (uint32_t)g.n[2]);
    heatbath_site<Real, MU>(g, c, hp, err);
}

// [R9] init: one thread per link of the device layout
template <typename Real>
__global__ void __launch_bounds__(kBlock)
    init_kernel(typename LinkPtr<Real>::type* __restrict__ links, const Geom g, int start, uint64_t seed)
{
    const uint32_t h = blockIdx.x * (uint32_t)kBlock + threadIdx.x;
    if (h >= g.vh) return;
    const int arr = blockIdx.y;  // p*4 + mu
    const int p = arr >> 2, mu = arr & 3;
    Quat<Real> u = {1, 0, 0, 0};
    if (start == 1) {
        uint32_t q = h / (uint32_t)g.nxh;
        uint32_t q2 = q / (uint32_t)g.n[1];
        const uint32_t y = q - q2 * (uint32_t)g.n[1];
        const uint32_t t = q2 / (uint32_t)g.n[2];
        const uint32_t z = q2 - t * (uint32_t)g.n[2];
        const uint32_t r = (y + z + t + (uint32_t)p) & 1u;
        const uint32_t s = 2u * h + r;
        const Words w = draw(seed, s, 0u, (1u << 8) | ((uint32_t)p << 2) | (uint32_t)mu, 0u);
        u = haar_from_words<Real>(w);
    }
    stq(links + (size_t)arr * g.vh + h, u);
}

bool tiled_ok(const Geom& g)
{
    // grid limits (y, z <= 65535) and exactness of the zmagic split: nb2^2 * nb3 < 2^32
    const uint64_t t0 = g.nxh >> kTileLog2[0], t1 = g.n[1] >> kTileLog2[1], t2 = g.n[2] >> kTileLog2[2],
                   t3 = g.n[3] >> kTileLog2[3];
    if (t1 > 65535 || t2 * t3 > 65535 || t0 == 0) return false;
    return g.nxh % (1 << kTileLog2[0]) == 0 && g.n[1] % (1 << kTileLog2[1]) == 0 &&
           g.n[2] % (1 << kTileLog2[2]) == 0 && g.n[3] % (1 << kTileLog2[3]) == 0;
}

template <typename Real, int MU>
static int launch_substep_t(void* links, const Geom& g, int parity, double beta, uint64_t seed, uint32_t sweep,
                            int* err, cudaStream_t st)
{
    typedef typename LinkPtr<Real>::type L;
    HbParams<Real> hp;
    hp.inv_beta = (Real)(1.0 / beta);
    hp.sweep = sweep;
    hp.rk = expand_keys(seed);
    hp.tag = ((uint32_t)parity << 2) | (uint32_t)MU;
    hp.parity = parity;
    for (int nu = 0; nu < 4; ++nu) {
        hp.same[nu] = (const L*)links + (size_t)(parity * 4 + nu) * g.vh;
        hp.oppo[nu] = (const L*)links + (size_t)((1 - parity) * 4 + nu) * g.vh;
    }
    hp.out = (L*)links + (size_t)(parity * 4 + MU) * g.vh;
    if (tiled_ok(g)) {
        constexpr int T = 1 << (kTileLog2[0] + kTileLog2[1] + kTileLog2[2] + kTileLog2[3]);
        const dim3 grid((unsigned)g.nb[0], (unsigned)g.nb[1], (unsigned)(g.nb[2] * g.nb[3]));
        heatbath_tiled_kernel<Real, MU, kTileLog2[0], kTileLog2[1], kTileLog2[2], kTileLog2[3]>
            <<<grid, T, 0, st>>>(g, hp, err);
    } else {
        const unsigned grid = (g.vh + kBlock - 1) / kBlock;
        heatbath_linear_kernel<Real, MU><<<grid, kBlock, 0, st>>>(g, hp, err);
    }
    return 1;
}

template <typename Real>
static int launch_substep_p(void* links, const Geom& g, int mu, int parity, double beta, uint64_t seed,
                            uint32_t sweep, int* err, cudaStream_t st)
{
    switch (mu) {
        case 0: return launch_substep_t<Real, 0>(links, g, parity, beta, seed, sweep, err, st);
        case 1: return launch_substep_t<Real, 1>(links, g, parity, beta, seed, sweep, err, st);
        case 2: return launch_substep_t<Real, 2>(links, g, parity, beta, seed, sweep, err, st);
        default: return launch_substep_t<Real, 3>(links, g, parity, beta, seed, sweep, err, st);
    }
}

int launch_heatbath_substep(void* links, const Geom& g, int precision, int mu, int parity, double beta,
                            uint64_t seed, uint32_t sweep, int* err, cudaStream_t st)
{
    return precision == 32 ? launch_substep_p<float>(links, g, mu, parity, beta, seed, sweep, err, st)
                           : launch_substep_p<double>(links, g, mu, parity, beta, seed, sweep, err, st);
}

int launch_init(void* links, const Geom& g, int precision, int start, uint64_t seed, cudaStream_t st)
{
    const dim3 grid((g.vh + kBlock - 1) / kBlock, 8);
    if (precision == 32)
        init_kernel<float><<<grid, kBlock, 0, st>>>((float4*)links, g, start, seed);
    else
        init_kernel<double><<<grid, kBlock, 0, st>>>((double4a*)links, g, start, seed);
    return 1;
}

}  // namespace su2
