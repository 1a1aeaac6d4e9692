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

// The 18 links of the staple are all requested before the first product: one
// round trip to L2/HBM per thread instead of one per product.
// Array bases are uniform 64-bit pointers, element indices 32-bit (h + delta < V/2).
//
// Overlap with the preceding sub-step. In the canonical order [R4] the
// kernel before (MU,P) wrote exactly one array that this one reads:
//   P = 1: U_MU on parity 0        = hp.oppo[MU]            (the b, b2 loads)
//   P = 0: U_{MU-1} on parity 1    = hp.oppo[(MU+3)%4]      (the a, c2 loads of that nu)
// With programmatic dependent launch the CTA is scheduled, decodes its site and computes
// its neighbour indices in the predecessor's tail, then waits (griddepcontrol.wait) before
// its first load; loads issued ahead of the wait were measured to cost more (an extra
// dependent round trip, or spills) than they hide. The predecessor's output is read
// through L2 (ld.global.cg): its lines may not be taken from an L1 that an overlapping
// launch did not invalidate. Launched without the attribute the wait is a no-op.
//
// Fused plaquette. MEAS is used only for P = 1, MU >= 1: the return value
// is 1/2 Tr(U' w), w = the staple terms of the directions nu < MU, i.e. the sum of the
// plaquettes of the planes (nu, MU), nu < MU, through the new link. Those planes are not
// touched by any later sub-step of the sweep and each of their plaquettes holds exactly
// one odd-parity mu-link, so the three kernels (1,1), (2,1), (3,1) together sum every
// plaquette of the final configuration exactly once.
// log table of su2_math64.cuh (fp64 kernels; 2 KB, stays in L1)
__device__ const m64::LogEntry kLogTab[m64::kLogEntries] = {
#include "su2_log_table.inc"
};
template <typename Real>
struct Staple18 {  // the 18 links of one staple sum, per direction nu != mu (i = 0..2)
    Quat<Real> a[3], b[3], cc[3], a2[3], b2[3], c2[3];
};
struct SiteIdx {
    int h;   // half-index of the site
    int r;   // low bit of x
    int ha;  // h + the replica's offset: index into the link arrays
    int t;   // time slice (a slab's edge slices are also stored to its neighbours)
};

// STATE: 0 = sweep index and 1/beta are launch parameters, 1 = they come from su2_run's device loop state, 2 = decided at
// run time by hp.state. The hot-path tiled kernels are instantiated for 0 and 1 (the run-time form costs every
// launch the ~12 instructions of the other one); the ALT and linear kernels use 2.
template <int STATE, typename Real>
__device__ __forceinline__ void run_state(const HbParams<Real>& hp, uint32_t& sweep, Real& inv_beta)
{
    sweep = hp.sweep;
    inv_beta = hp.inv_beta;
    if (STATE == 1 || (STATE == 2 && hp.state)) {  // su2_run: the captured graph's parameters are frozen, the loop state is not
        double ib;
        ld_run_state(run_state_copy(hp.state), ib, sweep);
        inv_beta = (Real)ib;
    }
}


// Checked build (-DHB_BOUNDS_CHECK; compute-sanitizer is not available on the GPU pool): every link index of a
// heat-bath thread is tested against its array, [hoff, hoff + V/2); a miss sets bit 1 of the error word, which
// su2_synchronize reports, and the access is redirected to the array's first element.
#ifdef HB_BOUNDS_CHECK
__device__ __forceinline__ uint32_t hb_check(uint32_t idx, uint32_t hoff, uint32_t vh, int* err)
{
    if (idx - hoff >= vh) {
        atomicOr(err, 2);
        return hoff;
    }
    return idx;
}
#define HB_CK(idx) hb_check((uint32_t)(idx), hoff, g.vh, err)
#else
#define HB_CK(idx) ((uint32_t)(idx))
#endif

// neighbour addressing (row 2) and the 18 loads (row 3, first half) of one site
template <typename Real, int MU, int P, int STATE>
__device__ __forceinline__ SiteIdx load18(const Geom& g, const Site& c, const HbParams<Real>& hp, Staple18<Real>& q,
                                          uint32_t& sweep, Real& inv_beta, uint32_t hoff, int* __restrict__ err)
{
    typedef typename LinkPtr<Real>::type L;
    constexpr int DEP_NU = (P == 0) ? (MU + 3) % 4 : -1;
    constexpr bool DEP_MU = (P == 1);
    SiteIdx ix;
    ix.r = (c.y + c.z + c.t + P) & 1;
    ix.h = c.hx + g.sy * c.y + g.sz * c.z + g.st * c.t;
    ix.ha = ix.h + (int)hoff;
    ix.t = c.t;
    const int h = ix.ha;
    const Nbr d = neighbours(g, c, ix.r);
    const L* o_mu = hp.oppo[MU];  // U_mu on the other parity
    const uint32_t h_up = HB_CK(h + d.up[MU]);
    // First-touch loads first. CTAs sweep the lattice x fastest, then y, z, t; of the reads of one array in a
    // sub-step the one that reaches furthest ahead in that order misses L2, the others find the line the
    // earlier CTA brought in: U_nu(x+mu) is always ahead of U_nu(x-nu); U_nu(x+mu-nu) is ahead of U_nu(x)
    // iff mu > nu; of the six reads of U_mu the one at x+nu with the largest nu. Those 7 go out as the first
    // batch, so that the later batches wait for cache hits only.
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const int nu = i + (i >= MU ? 1 : 0);
        q.a[i] = (nu == DEP_NU) ? ldq_dep(hp.oppo[nu] + h_up) : ldq(hp.oppo[nu] + h_up);  // U_nu(x+mu)
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const int nu = i + (i >= MU ? 1 : 0);
        if (MU > nu) q.a2[i] = ldq(hp.same[nu] + HB_CK((int)h_up + d.dn[nu]));  // U_nu(x+mu-nu)
        else q.cc[i] = ldq(hp.same[nu] + HB_CK(h));                             // U_nu(x)
    }
    {
        constexpr int nu = (MU == 3) ? 2 : 3;
        const uint32_t h_upnu = HB_CK(h + d.up[nu]);
        q.b[2] = DEP_MU ? ldq_dep(o_mu + h_upnu) : ldq(o_mu + h_upnu);  // U_mu(x+nu), largest nu
    }
    run_state<STATE>(hp, sweep, inv_beta);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const int nu = i + (i >= MU ? 1 : 0);
        const uint32_t h_dn = HB_CK(h + d.dn[nu]);
        if (i < 2) {
            const uint32_t h_upnu = HB_CK(h + d.up[nu]);
            q.b[i] = DEP_MU ? ldq_dep(o_mu + h_upnu) : ldq(o_mu + h_upnu);  // U_mu(x+nu)
        }
        if (MU > nu) q.cc[i] = ldq(hp.same[nu] + HB_CK(h));
        else q.a2[i] = ldq(hp.same[nu] + HB_CK((int)h_up + d.dn[nu]));
        q.b2[i] = DEP_MU ? ldq_dep(o_mu + h_dn) : ldq(o_mu + h_dn);                         // U_mu(x-nu)
        q.c2[i] = (nu == DEP_NU) ? ldq_dep(hp.oppo[nu] + h_dn) : ldq(hp.oppo[nu] + h_dn);  // U_nu(x-nu)
    }
    return ix;
}

// Hot-path kernels read the launch's expanded round keys (uniform registers); the ALT kernels key
// Philox from two words per thread (a batched launch has one seed per replica)
template <bool ALT>
__device__ __forceinline__ Words philox_sel(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const RoundKeys& rk,
                                            const RepCtx& rc)
{
    if (ALT) return philox4x32_10(c0, c1, c2, c3, rc.k0, rc.k1);
    return philox_keyed(c0, c1, c2, c3, rk);
}

// rows 3 (products) to 6: staple sum, Philox, Kennedy-Pendleton, compose, store
template <typename Real, int MU, int P, bool MEAS, bool ALT>
__device__ __forceinline__ Real update_link(const Staple18<Real>& q, const SiteIdx ix, uint32_t sweep, Real inv_beta,
                                            const HbParams<Real>& hp, const m64::LogEntry* tab,
                                            const RepCtx& rc, int* __restrict__ err)
{
    const Quat<Real>*a = q.a, *b = q.b, *cc = q.cc, *a2 = q.a2, *b2 = q.b2, *c2 = q.c2;
    const int h = ix.h, r = ix.r;
    // [R5] counter = (s, sweep, (p<<2)|mu, n); the n = 0 draw does not depend on the links
    uint32_t s = 2u * (uint32_t)h + (uint32_t)r;
    if (ALT) s += hp.s_off;  // slab: the global site keys the draws
    const uint32_t tag = ((uint32_t)P << 2) | (uint32_t)MU;
    const Words wd = philox_sel<ALT>(s, sweep, tag, 0u, hp.rk, rc);

    // [R3] staple sum, nu ascending, forward then backward, products left to right;
    // the second product of every term accumulates straight into v (FMA chains).
    Quat<Real> v = {0, 0, 0, 0}, w = {0, 0, 0, 0};
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        qmac<false, true>(v, qmul<false, true>(a[i], b[i]), cc[i]);    // (a b^+) c^+
        qmac<false, false>(v, qmul<true, true>(a2[i], b2[i]), c2[i]);  // (a2^+ b2^+) c2
        if (MEAS && i == MU - 1) w = v;  // nu = 0..MU-1 are the first MU terms
    }

    const Real k2 = v.a0 * v.a0 + v.a1 * v.a1 + v.a2 * v.a2 + v.a3 * v.a3;
    Quat<Real> u;
    if (k2 < M<Real>::tiny()) {  // [R8]
        u = haar_from_words<Real>(wd);
    } else {
        const Real rk = M<Real>::rsqrt(k2);       // 1/k
        const Real inv_alpha = rk * inv_beta;  // 1/(beta k)
        Real delta = 0;
        uint32_t n = 1;
        if (ALT && inv_alpha * hp.creutz_below > (Real)1) {
            // [R15] Creutz: propose x0 ~ exp(alpha x0) by inversion, accept with sqrt(1 - x0^2).
            // The rare small-alpha path: accurate library exp/log in both precisions.
            const Real E = M<Real>::exp((Real)-2 / inv_alpha);
            for (;;) {
                const Words w = philox_sel<ALT>(s, sweep, tag, n, hp.rk, rc);
                const Real R = M<Real>::uniform(w.w0), Rp = M<Real>::uniform(w.w1);
                delta = -M<Real>::log(R + ((Real)1 - R) * E) * inv_alpha;
                if (Rp * Rp <= delta * ((Real)2 - delta)) break;
                if (++n > 10000u) {
                    atomicOr(err, 1);
                    delta = 0;
                    break;
                }
            }
        } else {
            // [R6] Kennedy-Pendleton
            for (;;) {
                const Words w = philox_sel<ALT>(s, sweep, tag, n, hp.rk, rc);
                delta = M<Real>::kp_delta(w, inv_alpha, tab);
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
    stq(hp.out + (uint32_t)ix.ha, u);
    if (ALT && hp.peer_lo) {  // slab: the edge slices are the neighbours' halos
        if (ix.t == hp.t_first) stq(hp.peer_lo + (ix.ha + hp.d_lo), u);
        if (ix.t == hp.t_last) stq(hp.peer_hi + (ix.ha + hp.d_hi), u);
    }
    return MEAS ? u.a0 * w.a0 - u.a1 * w.a1 - u.a2 * w.a2 - u.a3 * w.a3 : (Real)0;  // 1/2 Tr(U' w)
}

template <typename Real, int MU, int P, bool MEAS, bool ALT, int STATE>
__device__ __forceinline__ Real heatbath_site(const Geom& g, const Site& c, const HbParams<Real>& hp, uint32_t rep,
                                              int* __restrict__ err)
{
    grid_dep_wait();    // the preceding kernel of the stream has finished and flushed
    grid_dep_launch();  // ... so the next one may be scheduled behind this CTA
    uint32_t sweep;
    Real inv_beta;
    Staple18<Real> q;
    RepCtx rc = {0u, 0u, hp.rk.k[0], hp.rk.k[1]};
    if (ALT) rc = {rep, rep * hp.rep_stride, hp.rk.k[0], hp.rk.k[1]};
    const SiteIdx ix = load18<Real, MU, P, STATE>(g, c, hp, q, sweep, inv_beta, rc.hoff, err);
    if (ALT && hp.reps) {  // batched launch: this replica's coupling and seed
        const RepParams rp = hp.reps[rep];
        inv_beta = (Real)rp.inv_beta;
        rc.k0 = (uint32_t)rp.seed;
        rc.k1 = (uint32_t)(rp.seed >> 32);
    }
    return update_link<Real, MU, P, MEAS, ALT>(q, ix, sweep, inv_beta, hp, kLogTab, rc, err);
}

// Resident CTAs per SM that ptxas must allow: this is the register budget that lets it
// keep all 18 link loads of a thread in flight at once.
#ifndef HB_MINB_F32
#define HB_MINB_F32 8
#endif
#ifndef HB_MINB_F64
#define HB_MINB_F64 6
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
// TLOOP: consecutive t-tiles one CTA walks through (kTLoop for the hot-path kernels of large lattices, where a
// quarter of the CTA launches and drains is worth 4-5 % in fp32 and 2 % in fp64; 0 = g.tloop at run time, the
// ALT kernels).
#ifndef HB_TLOOP
#define HB_TLOOP 4
#endif

constexpr int kTLoop = HB_TLOOP;
template <typename Real, int MU, int P, bool MEAS, bool ALT, int LHX, int LY, int LZ, int LT, int TLOOP, int STATE>
__global__ void __launch_bounds__(1 << (LHX + LY + LZ + LT), (MinBlocks<Real>::value << 7) >> (LHX + LY + LZ + LT))
    heatbath_tiled_kernel(const Geom g, const HbParams<Real> hp, int* __restrict__ err)
{
    uint32_t rep = 0, bzt = blockIdx.z;
    if (ALT && hp.reps) {  // batched launch: grid z = (replica, z-t tile)
        rep = bzt / hp.nzt;
        bzt -= rep * hp.nzt;
    }
    Site c = tile_site<LHX, LY, LZ, LT>(g, bzt);
    // One CTA walks through `tloop` consecutive t-tiles: 65536 CTAs of 3.5 us each leave the
    // SMs' CTA slots empty 6 % of the time between a drain and the next launch (ncu: 44 % warps active of 50 %).
    const int tloop = TLOOP ? TLOOP : g.tloop;
    const int tt = c.t & ((1 << LT) - 1);
    c.t = (c.t - tt) * tloop + tt;
    if (ALT) c.t += g.t_lo;  // slab: the grid covers the interior slices only
    Real e = 0;
    if (TLOOP == 1) {
        e = heatbath_site<Real, MU, P, MEAS, ALT, STATE>(g, c, hp, rep, err);
    } else {
#pragma unroll 1
        for (int it = 0; it < tloop; ++it, c.t += 1 << LT)
            e += heatbath_site<Real, MU, P, MEAS, ALT, STATE>(g, c, hp, rep, err);
    }
    if (MEAS) {  // one fp64 partial per CTA, fixed order
        __shared__ double red[kBlock / 32];
        const double tot = block_sum_end((double)e, red);
        if (threadIdx.x == 0)
            hp.epart[(size_t)rep * hp.epart_stride + blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * bzt)] = tot;
    }
}

// linear launch: thread i <-> half-index h = i; any even extents
template <typename Real, int MU, int P, bool MEAS, bool ALT>
__global__ void __launch_bounds__(kBlock)
    heatbath_linear_kernel(const Geom g, const HbParams<Real> hp, int* __restrict__ err)
{
    uint32_t h = blockIdx.x * (uint32_t)kBlock + threadIdx.x;
    Real e = 0;
    if (h < (ALT ? (uint32_t)g.st * (uint32_t)g.nt_upd : g.vh)) {
        if (ALT) h += (uint32_t)g.st * (uint32_t)g.t_lo;  // slab: interior slices only
        Site c;
        uint32_t q = h / (uint32_t)g.nxh;
        c.hx = (int)(h - q * (uint32_t)g.nxh);
        uint32_t q2 = q / (uint32_t)g.n[1];
        c.y = (int)(q - q2 * (uint32_t)g.n[1]);
        c.t = (int)(q2 / (uint32_t)g.n[2]);
        c.z = (int)(q2 - (uint32_t)c.t * (uint32_t)g.n[2]);
        e = heatbath_site<Real, MU, P, MEAS, ALT, 2>(g, c, hp, blockIdx.y, err);  // grid y = replica
    }
    if (MEAS) {
        __shared__ double red[kBlock / 32];
        const double tot = block_sum_end((double)e, red);
        if (threadIdx.x == 0) hp.epart[(size_t)blockIdx.y * hp.epart_stride + blockIdx.x] = tot;
    }
}

// [R9] init: one thread per link of the device layout
template <typename Real>
__global__ void __launch_bounds__(kBlock)
    init_kernel(typename LinkPtr<Real>::type* __restrict__ links, const Geom g, int start, uint64_t seed, int t_shift,
                int nt_glob)
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
        // slab: slice t holds the global slice (t + t_shift) mod Nt (t_shift even), whose site keys the draw
        int tg = ((int)t + t_shift) % nt_glob;
        if (tg < 0) tg += nt_glob;
        const uint32_t s = 2u * h + r + 2u * (uint32_t)g.st * (uint32_t)(tg - (int)t);
        const Words w = draw(seed, s, 0u, (1u << 8) | ((uint32_t)p << 2) | (uint32_t)mu, 0u);
        u = haar_from_words<Real>(w);
    }
    stq(links + (size_t)arr * g.vh + h, u);
}

void choose_tiling(Geom& g, int nrep, int precision)
{
    (void)precision;  // both precisions use the same tiling (the fp64 kernels took no walk until r02)
    g.tile = -1;
    g.tloop = 1;
    g.nb[0] = g.nb[1] = g.nb[2] = g.nb[3] = 0;
    g.zmagic = 0;
    for (int k = 0; k < kNumTiles; ++k) {
        const int* t = kTiles[k];
        const int ext[4] = {g.nxh, g.n[1], g.n[2], g.nt_upd};
        bool ok = true;
        for (int d = 0; d < 4; ++d) ok = ok && ext[d] % (1 << t[d]) == 0;
        if (!ok) continue;
        const uint64_t nb1 = g.n[1] >> t[1], nb2 = g.n[2] >> t[2], nb3 = g.nt_upd >> t[3];
        // grid limits (y, z <= 65535) and exactness of the zmagic split: nb2^2 * nb3 < 2^32
        // (a batch carries the replica in grid z as well)
        if (nb1 > 65535 || nb2 * nb3 * (uint64_t)nrep > 65535) continue;
        g.tile = k;
        g.nb[0] = g.nxh >> t[0];
        g.nb[1] = (int)nb1;
        g.nb[2] = (int)nb2;
        g.nb[3] = (int)nb3;
        // walk (see heatbath_tiled_kernel): first tile shape, and at least 4 CTA waves of 148 x 8 left
        if (k == 0 && nb3 % kTLoop == 0 && (uint64_t)g.nb[0] * nb1 * nb2 * (nb3 / kTLoop) >= 4736)
            g.tloop = kTLoop;
        g.zmagic = (uint32_t)(((1ull << 32) + nb2 - 1) / nb2);  // unused if nb2 == 1
        return;
    }
}

template <typename Real, int MU, int P, bool MEAS, bool ALT>
static int launch_substep_t(void* links, const Geom& g, double beta, double creutz_below, uint64_t seed,
                            uint32_t sweep, int* err, double* epart, const RunState* state, const RepParams* reps,
                            int nrep, bool overlap, cudaStream_t st, const SlabCtx* slab)
{
    typedef typename LinkPtr<Real>::type L;
    HbParams<Real> hp;
    hp.s_off = 0;
    hp.peer_lo = hp.peer_hi = nullptr;
    hp.d_lo = hp.d_hi = 0;
    hp.t_first = hp.t_last = -1;
    if (slab) {  // ALT kernels
        hp.s_off = slab->s_off;
        hp.peer_lo = (L*)slab->peer_lo + (size_t)(P * 4 + MU) * slab->vh_lo;
        hp.peer_hi = (L*)slab->peer_hi + (size_t)(P * 4 + MU) * slab->vh_hi;
        hp.d_lo = slab->d_lo;
        hp.d_hi = slab->d_hi;
        hp.t_first = g.t_lo;
        hp.t_last = g.t_lo + g.nt_upd - 1;
    }
    hp.inv_beta = (Real)(1.0 / beta);
    hp.sweep = sweep;
    hp.creutz_below = (Real)creutz_below;
    hp.rk = expand_keys(seed);
    for (int nu = 0; nu < 4; ++nu) {
        hp.same[nu] = (const L*)links + (size_t)(P * 4 + nu) * g.vh;
        hp.oppo[nu] = (const L*)links + (size_t)((1 - P) * 4 + nu) * g.vh;
    }
    hp.out = (L*)links + (size_t)(P * 4 + MU) * g.vh;
    hp.epart = epart;
    hp.state = state;
    hp.reps = reps;
    hp.rep_stride = 8u * g.vh;
    hp.nzt = (uint32_t)(g.nb[2] * (g.nb[3] / g.tloop));
    hp.epart_stride = (uint32_t)(3 * heatbath_ctas(g));
    const dim3 grid((unsigned)g.nb[0], (unsigned)g.nb[1], (unsigned)(g.nb[2] * (g.nb[3] / g.tloop) * nrep));
    // hot-path kernels: the walk length (1, or kTLoop on the first tile shape) and the source of the loop state are
    // template parameters; the ALT kernels read both at run time
    const dim3 block0(1 << (kTiles[0][0] + kTiles[0][1] + kTiles[0][2] + kTiles[0][3]));
    const dim3 block1(1 << (kTiles[1][0] + kTiles[1][1] + kTiles[1][2] + kTiles[1][3]));
#define SU2_TILED(K_, TL_, ST_)                                                                                       \
    launch_ex(heatbath_tiled_kernel<Real, MU, P, MEAS, ALT, kTiles[K_][0], kTiles[K_][1], kTiles[K_][2], kTiles[K_][3], \
                                    TL_, ST_>,                                                                        \
              grid, K_ == 0 ? block0 : block1, st, overlap, g, hp, err)
    if constexpr (ALT) {
        if (g.tile == 0) SU2_TILED(0, 0, 2);
        else if (g.tile == 1) SU2_TILED(1, 0, 2);
    } else {
        if (g.tile == 0 && g.tloop == kTLoop) {
            if (state) SU2_TILED(0, kTLoop, 1);
            else SU2_TILED(0, kTLoop, 0);
        } else if (g.tile == 0) {
            if (state) SU2_TILED(0, 1, 1);
            else SU2_TILED(0, 1, 0);
        } else if (g.tile == 1) {
            if (state) SU2_TILED(1, 1, 1);
            else SU2_TILED(1, 1, 0);
        }
    }
#undef SU2_TILED
    if (g.tile < 0) {
        launch_ex(heatbath_linear_kernel<Real, MU, P, MEAS, ALT>, dim3((unsigned)heatbath_ctas(g), (unsigned)nrep),
                  dim3(kBlock), st, overlap, g, hp, err);
    }
    return 1;
}

// number of CTAs (= fused-plaquette partials) of one heat-bath launch
size_t heatbath_ctas(const Geom& g)
{
    if (g.tile >= 0) return (size_t)g.nb[0] * g.nb[1] * g.nb[2] * (g.nb[3] / g.tloop);
    return ((size_t)g.st * g.nt_upd + kBlock - 1) / kBlock;
}

template <typename Real, bool ALT>
static int launch_substep_p(void* links, const Geom& g, int mu, int parity, double beta, double cb, uint64_t seed,
                            uint32_t sweep, int* err, double* epart, const RunState* state, const RepParams* reps,
                            int nrep, bool overlap, cudaStream_t st, const SlabCtx* slab)
{
#define SU2_HB(MU_, P_, MEAS_, EP_)                                                                               \
    return launch_substep_t<Real, MU_, P_, MEAS_, ALT>(links, g, beta, cb, seed, sweep, err, EP_, state, reps, nrep, \
                                                       overlap, st, slab)
    if (epart && parity == 1 && mu >= 1) {  // the three measuring kernels
        switch (mu) {
            case 1: SU2_HB(1, 1, true, epart);
            case 2: SU2_HB(2, 1, true, epart);
            default: SU2_HB(3, 1, true, epart);
        }
    }
    switch (mu * 2 + parity) {
        case 0: SU2_HB(0, 0, false, nullptr);
        case 1: SU2_HB(0, 1, false, nullptr);
        case 2: SU2_HB(1, 0, false, nullptr);
        case 3: SU2_HB(1, 1, false, nullptr);
        case 4: SU2_HB(2, 0, false, nullptr);
        case 5: SU2_HB(2, 1, false, nullptr);
        case 6: SU2_HB(3, 0, false, nullptr);
        default: SU2_HB(3, 1, false, nullptr);
    }
#undef SU2_HB
}

// `overlap` may be true only if the launch before this one on `st` was the canonical
// predecessor sub-step [R4] of the same lattice (see heatbath_site). `epart` (nullable):
// where the sub-steps (mu >= 1, parity 1) store their heatbath_ctas(g) fused-plaquette
// partials; ignored by the other sub-steps.
// `creutz_below` [R15]: 0 = Kennedy-Pendleton everywhere (the hot-path kernels); otherwise the ALT
// kernels, which use Creutz's draw on links with alpha < creutz_below (+inf = on every link).
// `reps` (nullable, [device]): batched launch over `nrep` configurations stored one after the other
// from `links`, each with its own 1/beta and seed (beta and seed arguments are then unused); `epart`
// then holds nrep * 3 * heatbath_ctas(g) partials, replica-major. Batched launches use the ALT kernels.
int launch_heatbath_substep(void* links, const Geom& g, int precision, int mu, int parity, double beta,
                            double creutz_below, uint64_t seed, uint32_t sweep, int* err, double* epart,
                            const RunState* state, bool overlap, cudaStream_t st, const RepParams* reps, int nrep,
                            const SlabCtx* slab)
{
    const bool alt = creutz_below > 0.0 || reps != nullptr || slab != nullptr;
    if (!reps) nrep = 1;
#define SU2_HB(REAL_, ALT_)                                                                                      \
    launch_substep_p<REAL_, ALT_>(links, g, mu, parity, beta, creutz_below, seed, sweep, err, epart, state, reps, \
                                  nrep, overlap, st, slab)
    if (precision == 32) return alt ? SU2_HB(float, true) : SU2_HB(float, false);
    return alt ? SU2_HB(double, true) : SU2_HB(double, false);
#undef SU2_HB
}

int launch_init(void* links, const Geom& g, int precision, int start, uint64_t seed, cudaStream_t st, int t_shift,
                int nt_glob)
{
    const dim3 grid((g.vh + kBlock - 1) / kBlock, 8);
    if (nt_glob <= 0) nt_glob = g.n[3];
    if (precision == 32)
        init_kernel<float><<<grid, kBlock, 0, st>>>((float4*)links, g, start, seed, t_shift, nt_glob);
    else
        init_kernel<double><<<grid, kBlock, 0, st>>>((double4a*)links, g, start, seed, t_shift, nt_glob);
    return 1;
}

}  // namespace su2
