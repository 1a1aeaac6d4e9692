// su2_measure.cu — mean plaquette (row 7), Polyakov loop (row 8), Polyakov-loop
// correlator (NEXT-1) and the canonical <-> device layout conversions.
//
// Reductions: per-thread fp64 value -> warp shuffle -> fixed-order block tree ->
// one partial per block -> one final block that sums the partials in a fixed
// strided order. Block size kBlock is part of the definition, so a given lattice
// always produces the same bits.
#include "su2_launch.h"

namespace su2 {

// ------------------------------------------------------------------ plaquette
// one thread per site; grid.y = parity. [R10]
//   1/2 Tr[U_mu(x) U_nu(x+mu) U_mu^dag(x+nu) U_nu^dag(x)]
//     = < U_mu(x) U_nu(x+mu) , U_nu(x) U_mu(x+nu) >   (4-vector dot product)
template <typename Real>
__global__ void __launch_bounds__(kBlock)
    plaquette_kernel(const typename LinkPtr<Real>::type* __restrict__ links, const Geom g,
                     double* __restrict__ partials)
{
    typedef typename LinkPtr<Real>::type L;
    __shared__ double red[kBlock / 32];
    uint32_t h = blockIdx.x * (uint32_t)kBlock + threadIdx.x;
    const int p = blockIdx.y;
    double acc = 0.0;
    if (h < (uint32_t)g.st * (uint32_t)g.nt_upd) {  // = V/2, or the interior slices of a slab
        h += (uint32_t)g.st * (uint32_t)g.t_lo;
        uint32_t q = h / (uint32_t)g.nxh;
        const int hx = (int)(h - q * (uint32_t)g.nxh);
        uint32_t q2 = q / (uint32_t)g.n[1];
        const int y = (int)(q - q2 * (uint32_t)g.n[1]);
        const int t = (int)(q2 / (uint32_t)g.n[2]);
        const int z = (int)(q2 - (uint32_t)t * (uint32_t)g.n[2]);
        const int r = (y + z + t + p) & 1;
        int up[4];
        up[0] = r ? ((hx + 1 == g.nxh) ? -(g.nxh - 1) : 1) : 0;
        up[1] = (y + 1 == g.n[1]) ? -(g.n[1] - 1) * g.sy : g.sy;
        up[2] = (z + 1 == g.n[2]) ? -(g.n[2] - 1) * g.sz : g.sz;
        up[3] = (t + 1 == g.n[3]) ? -(g.n[3] - 1) * g.st : g.st;
        const size_t vh = g.vh;
        const L* same = links + (size_t)(p * 4) * vh;
        const L* oppo = links + (size_t)((1 - p) * 4) * vh;
        Quat<Real> u[4];
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) u[mu] = ldq(same + mu * vh + h);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu)
#pragma unroll
            for (int nu = mu + 1; nu < 4; ++nu) {
                const Quat<Real> a = qmul<false, false>(u[mu], ldq(oppo + nu * vh + ((int)h + up[mu])));
                const Quat<Real> b = qmul<false, false>(u[nu], ldq(oppo + mu * vh + ((int)h + up[nu])));
                acc += (double)qdot(a, b);
            }
    }
    const double tot = block_sum(acc, red);
    if (threadIdx.x == 0) partials[blockIdx.y * gridDim.x + blockIdx.x] = tot;
}

// Tiled form (same CTA tiles as the heat-bath kernel): grid.x carries
// (tile along x, parity), parity fastest, so the two CTAs that read the same 8 tiles of
// links are scheduled back to back and the second is served by L2 (with parity slowest
// ncu showed 2.15 GB of DRAM reads for 1.07 GB of links). All 16 links of a site are requested before the
// first product; one partial per CTA, indexed by the linear CTA id.
// Measured and rejected in round 2 (profiles/r02b.md): both parities of a tile in ONE 256-thread CTA (L1 then
// serves 56 % of the reads, L2 -> SM traffic falls by 30 %, yet 347 against 302 us at 64^4 fp32), and host-resolved
// array bases with 32-bit indices and an fp32 per-site sum (11 % fewer instructions, 343 us): the kernel is
// bound by the latency of its load batches at 29 resident warps, neither by L2 bandwidth nor by issue slots.
// (Repeated with the round-1 pointer arithmetic, in case the parameter-table lookups had cost the first attempt:
// L2 -> SM traffic 3.62 -> 2.53 GB, 301 -> 313 us. Not L2-bound.) fp64: 6 resident CTAs (80 registers) instead of 4
// (126): 553 -> 523 us at 64^4 = 0.63 of the copy peak.
#ifndef PLAQ_MINB_F32
#define PLAQ_MINB_F32 8
#endif
#ifndef PLAQ_MINB_F64
#define PLAQ_MINB_F64 6
#endif
template <typename Real, int LHX, int LY, int LZ, int LT>
__global__ void __launch_bounds__(1 << (LHX + LY + LZ + LT),
                                  ((sizeof(Real) == 4 ? PLAQ_MINB_F32 : PLAQ_MINB_F64) << 7) >> (LHX + LY + LZ + LT))
    plaquette_tiled_kernel(const typename LinkPtr<Real>::type* __restrict__ links, const Geom g,
                           double* __restrict__ partials)
{
    typedef typename LinkPtr<Real>::type L;
    __shared__ double red[kBlock / 32];
    const int p = blockIdx.x & 1;
    Site c = tile_site<LHX, LY, LZ, LT>(g, blockIdx.z, blockIdx.x >> 1);
    c.t += g.t_lo;  // slab: interior slices only (0 for a whole lattice)
    const int r = (c.y + c.z + c.t + p) & 1;
    const int h = c.hx + g.sy * c.y + g.sz * c.z + g.st * c.t;
    int up[4];
    up[0] = r ? ((c.hx + 1 == g.nxh) ? g.wup[0] : 1) : 0;
    up[1] = (c.y + 1 == g.n[1]) ? g.wup[1] : g.sy;
    up[2] = (c.z + 1 == g.n[2]) ? g.wup[2] : g.sz;
    up[3] = (c.t + 1 == g.n[3]) ? g.wup[3] : g.st;
    const size_t vh = g.vh;
    const L* same = links + (size_t)(p * 4) * vh;
    const L* oppo = links + (size_t)((1 - p) * 4) * vh;
    Quat<Real> u[4], n1[6], n2[6];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) u[mu] = ldq(same + mu * vh + (uint32_t)h);
    {
        int k = 0;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu)
#pragma unroll
            for (int nu = mu + 1; nu < 4; ++nu, ++k) {
                n1[k] = ldq(oppo + nu * vh + (uint32_t)(h + up[mu]));  // U_nu(x+mu)
                n2[k] = ldq(oppo + mu * vh + (uint32_t)(h + up[nu]));  // U_mu(x+nu)
            }
    }
    double acc = 0.0;
    {
        int k = 0;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu)
#pragma unroll
            for (int nu = mu + 1; nu < 4; ++nu, ++k)
                acc += (double)qdot(qmul<false, false>(u[mu], n1[k]), qmul<false, false>(u[nu], n2[k]));
    }
    const double tot = block_sum(acc, red);
    if (threadIdx.x == 0) partials[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = tot;
}

// final stage: dst[0] = scale * sum(partials[0..n)), fixed order
__global__ void __launch_bounds__(1024) final_sum_kernel(const double* __restrict__ partials, size_t n, double scale,
                                                         double* __restrict__ dst)
{
    __shared__ double red[32];
    double acc = 0.0;
    for (size_t i = threadIdx.x; i < n; i += 1024) acc += partials[i];
    const double tot = block_sum(acc, red);
    if (threadIdx.x == 0) dst[0] = tot * scale;
}

// ------------------------------------------------------------------ tail of a step
// su2_heatbath_sweep_measure / su2_run: the Polyakov kernel is the last kernel of a step and
// also finishes both observables (no separate final-sum launch). CTA b sums slice b of the
// fused-plaquette partials (fixed slice, fixed order) and stores it beside its Polyakov
// partial; the CTA that draws the last ticket then sums the gridDim.x slot pairs in index
// order. Grid and slices depend on the lattice only: a given lattice always gives the same bits.
struct StepTail {
    const double* epart;  // [device] fused-plaquette partials of the sweep; NULL = no tail (plain Polyakov kernel)
    size_t n_epart;
    double scale_plaq, scale_poly;
    double* slots;        // [device] 2 * gridDim.x doubles per replica
    unsigned* ticket;     // [device] one per replica + one for the whole batch, zero between steps
    double* dst;          // [device] 2 doubles per replica (ignored when state != NULL)
    RunState* state;      // su2_run: destination state->out[2*index..], then sweep and index advance
    unsigned advance;     // ... by this much (1; 2 when two loop states alternate)
};
__device__ __forceinline__ void step_tail(const StepTail& tl, double poly_tot, double* red)
{
    __shared__ bool is_last;
    const unsigned G = gridDim.x, b = blockIdx.x, rep = blockIdx.y;  // grid y = replica of a batched launch
    const double* epart = tl.epart + (size_t)rep * tl.n_epart;
    double* slots = tl.slots + (size_t)rep * 2 * G;
    unsigned* ticket = tl.ticket + rep;
    const size_t chunk = (tl.n_epart + G - 1) / G;
    const size_t lo = (size_t)b * chunk, hi = (lo + chunk < tl.n_epart) ? lo + chunk : tl.n_epart;
    double acc = 0.0;
    for (size_t i = lo + threadIdx.x; i < hi; i += blockDim.x) acc += __ldcg(epart + i);
    const double ea = block_sum(acc, red);
    if (threadIdx.x == 0) {
        slots[2 * b] = ea;
        slots[2 * b + 1] = poly_tot;
        __threadfence();
        is_last = atomicAdd(ticket, 1u) == G - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double sa = 0.0, sb = 0.0;
    for (unsigned i = threadIdx.x; i < G; i += blockDim.x) {
        sa += __ldcg(slots + 2 * i);
        sb += __ldcg(slots + 2 * i + 1);
    }
    const double ta = block_sum(sa, red);
    const double tb = block_sum(sb, red);
    const unsigned R = gridDim.y;  // replicas of a batched launch (1 otherwise)
    if (threadIdx.x == 0) {
        double* dst = tl.state ? tl.state->out + 2 * ((size_t)tl.state->index * R + rep) : tl.dst + 2 * (size_t)rep;
        dst[0] = ta * tl.scale_plaq;
        dst[1] = tb * tl.scale_poly;
        *ticket = 0u;
    }
    if (tl.state && R > 1) {  // su2_batch_run: the state advances once per round, after the last replica has read it
        __shared__ bool all_done;
        if (threadIdx.x == 0) {
            __threadfence();
            all_done = atomicAdd(tl.ticket + R, 1u) == R - 1;
            if (all_done) tl.ticket[R] = 0u;
        }
        __syncthreads();
        if (!all_done) return;
    }
    if (tl.state)  // su2_run: advance every copy of the loop state (this CTA is the last one running)
        for (int i = threadIdx.x; i < kRunCopies; i += blockDim.x) {
            tl.state[i].sweep += tl.advance;
            tl.state[i].index += tl.advance;
        }
}

// ------------------------------------------------------------------ Polyakov loop
// one thread per spatial site; ordered product of the N_t time links [R11]
constexpr int kPolyBatch = 8;
template <typename Real>
__global__ void __launch_bounds__(kBlock)
    polyakov_kernel(const typename LinkPtr<Real>::type* __restrict__ links, const Geom g,
                    double* __restrict__ field, double* __restrict__ partials, const StepTail tl)
{
    typedef typename LinkPtr<Real>::type L;
    __shared__ double red[kBlock / 32];
    const uint32_t v3 = (uint32_t)g.n[0] * (uint32_t)g.n[1] * (uint32_t)g.n[2];
    const uint32_t s3 = blockIdx.x * (uint32_t)kBlock + threadIdx.x;
    // as the last kernel of a step it may be scheduled while sub-step (3,1) drains:
    // every thread waits (the tail reads that kernel's partials), links are read through L2
    grid_dep_wait();
    grid_dep_launch();
    links += (size_t)blockIdx.y * 8 * g.vh;  // grid y = replica of a batched launch (else 0)
    if (field) field += (size_t)blockIdx.y * v3;
    double val = 0.0;
    if (s3 < v3) {
        const uint32_t x = s3 % (uint32_t)g.n[0];
        const uint32_t q = s3 / (uint32_t)g.n[0];
        const uint32_t y = q % (uint32_t)g.n[1], z = q / (uint32_t)g.n[1];
        const int p0 = (int)((x + y + z) & 1u);
        const size_t vh = g.vh;
        const L* a0 = links + (size_t)(p0 * 4 + 3) * vh + (s3 >> 1);        // even t
        const L* a1 = links + (size_t)((1 - p0) * 4 + 3) * vh + (s3 >> 1);  // odd t
        // The N_t loads of a line are independent, only the products are ordered: request kPolyBatch links
        // at a time, then multiply them in order (one L2/HBM round trip per batch instead of one per link).
        Quat<Real> prod = {1, 0, 0, 0};
        const int nt = g.n[3];
        for (int t0 = 0; t0 < nt; t0 += kPolyBatch) {
            Quat<Real> u[kPolyBatch];
#pragma unroll
            for (int j = 0; j < kPolyBatch; ++j) {
                const int t = min(t0 + j, nt - 1);  // the tail re-reads the last link (ignored below)
                u[j] = ldq_cg(((t & 1) ? a1 : a0) + (size_t)t * (size_t)g.st);
            }
#pragma unroll
            for (int j = 0; j < kPolyBatch; ++j)
                if (t0 + j < nt) prod = (t0 + j == 0) ? u[0] : qmul<false, false>(prod, u[j]);
        }
        val = (double)prod.a0;
        if (field) field[s3] = val;
    }
    const double tot = block_sum(val, red);
    if (tl.epart) {
        step_tail(tl, tot, red);
        return;
    }
    if (threadIdx.x == 0) partials[blockIdx.x] = tot;
}

// Long time extents: S threads per spatial site, each the ordered product of N_t/S
// consecutive time links; the S partial products are multiplied in order through shared
// memory. S = 1 above is the plain loop; S is fixed by N_t, so a lattice always gives the
// same bits. (32^4: the one-thread-per-site loop is 32 dependent loads deep on only 128 CTAs.)
template <typename Real, int S>
__global__ void __launch_bounds__(kBlock)
    polyakov_split_kernel(const typename LinkPtr<Real>::type* __restrict__ links, const Geom g,
                          double* __restrict__ field, double* __restrict__ partials, const StepTail tl)
{
    typedef typename LinkPtr<Real>::type L;
    constexpr int SITES = kBlock / S;
    __shared__ double red[kBlock / 32];
    __shared__ Quat<Real> part[S][SITES];
    const uint32_t v3 = (uint32_t)g.n[0] * (uint32_t)g.n[1] * (uint32_t)g.n[2];
    const int seg = threadIdx.x / SITES, lane = threadIdx.x % SITES;
    const uint32_t s3 = blockIdx.x * (uint32_t)SITES + lane;
    const int len = g.n[3] / S, t0 = seg * len;
    grid_dep_wait();
    grid_dep_launch();
    links += (size_t)blockIdx.y * 8 * g.vh;  // grid y = replica of a batched launch (else 0)
    if (field) field += (size_t)blockIdx.y * v3;
    if (s3 < v3) {
        const uint32_t x = s3 % (uint32_t)g.n[0];
        const uint32_t q = s3 / (uint32_t)g.n[0];
        const uint32_t y = q % (uint32_t)g.n[1], z = q / (uint32_t)g.n[1];
        const int p0 = (int)((x + y + z) & 1u);
        const size_t vh = g.vh;
        const L* a0 = links + (size_t)(p0 * 4 + 3) * vh + (s3 >> 1);        // even t
        const L* a1 = links + (size_t)((1 - p0) * 4 + 3) * vh + (s3 >> 1);  // odd t
        Quat<Real> prod = ldq_cg(((t0 & 1) ? a1 : a0) + (size_t)t0 * (size_t)g.st);
#pragma unroll 4
        for (int t = t0 + 1; t < t0 + len; ++t) {
            const Quat<Real> u = ldq_cg(((t & 1) ? a1 : a0) + (size_t)t * (size_t)g.st);
            prod = qmul<false, false>(prod, u);
        }
        part[seg][lane] = prod;
    }
    __syncthreads();
    double val = 0.0;
    if (seg == 0 && s3 < v3) {
        Quat<Real> prod = part[0][lane];
#pragma unroll
        for (int k = 1; k < S; ++k) prod = qmul<false, false>(prod, part[k][lane]);
        val = (double)prod.a0;
        if (field) field[s3] = val;
    }
    const double tot = block_sum(val, red);
    if (tl.epart) {
        step_tail(tl, tot, red);
        return;
    }
    if (threadIdx.x == 0) partials[blockIdx.x] = tot;
}

// Time slab: the ordered product continues from slab to slab. `prev` holds the product
// of the slices below this slab per spatial site (NULL: this slab holds t = 0), `next` receives the
// product including this slab's interior slices; the association is the plain loop's, left to right.
template <typename Real>
__global__ void __launch_bounds__(kBlock)
    polyakov_chain_kernel(const typename LinkPtr<Real>::type* __restrict__ links, const Geom g,
                          const typename LinkPtr<Real>::type* __restrict__ prev,
                          typename LinkPtr<Real>::type* __restrict__ next, double* __restrict__ partials)
{
    typedef typename LinkPtr<Real>::type L;
    __shared__ double red[kBlock / 32];
    const uint32_t v3 = (uint32_t)g.n[0] * (uint32_t)g.n[1] * (uint32_t)g.n[2];
    const uint32_t s3 = blockIdx.x * (uint32_t)kBlock + threadIdx.x;
    double val = 0.0;
    if (s3 < v3) {
        const uint32_t x = s3 % (uint32_t)g.n[0];
        const uint32_t q = s3 / (uint32_t)g.n[0];
        const uint32_t y = q % (uint32_t)g.n[1], z = q / (uint32_t)g.n[1];
        const int p0 = (int)((x + y + z) & 1u);
        const size_t vh = g.vh;
        const L* a0 = links + (size_t)(p0 * 4 + 3) * vh + (s3 >> 1);        // even t
        const L* a1 = links + (size_t)((1 - p0) * 4 + 3) * vh + (s3 >> 1);  // odd t
        int t = g.t_lo;
        Quat<Real> prod;
        if (prev) {
            const L v = prev[s3];
            prod = {v.x, v.y, v.z, v.w};
        } else {
            prod = ldq_cg(((t & 1) ? a1 : a0) + (size_t)t * (size_t)g.st);
            ++t;
        }
        for (; t < g.t_lo + g.nt_upd; ++t) {
            const Quat<Real> u = ldq_cg(((t & 1) ? a1 : a0) + (size_t)t * (size_t)g.st);
            prod = qmul<false, false>(prod, u);
        }
        val = (double)prod.a0;
        if (next) stq(next + s3, prod);
    }
    const double tot = block_sum(val, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = tot;
}

// ------------------------------------------------------------------ correlator (NEXT-1)
// C(r) = 1/(3 V3) sum_x sum_{i=x,y,z} l(x) l(x + r e_i);  grid.y = r-1
__global__ void __launch_bounds__(kBlock)
    correlator_kernel(const double* __restrict__ field, const Geom g, double* __restrict__ partials)
{
    __shared__ double red[kBlock / 32];
    const uint32_t v3 = (uint32_t)g.n[0] * (uint32_t)g.n[1] * (uint32_t)g.n[2];
    const uint32_t s3 = blockIdx.x * (uint32_t)kBlock + threadIdx.x;
    const int r = blockIdx.y + 1;
    double val = 0.0;
    if (s3 < v3) {
        const int x = (int)(s3 % (uint32_t)g.n[0]);
        const uint32_t q = s3 / (uint32_t)g.n[0];
        const int y = (int)(q % (uint32_t)g.n[1]), z = (int)(q / (uint32_t)g.n[1]);
        const int xs = (x + r) % g.n[0], ys = (y + r) % g.n[1], zs = (z + r) % g.n[2];
        const double l0 = field[s3];
        const double lx = field[(uint32_t)xs + (uint32_t)g.n[0] * ((uint32_t)y + (uint32_t)g.n[1] * (uint32_t)z)];
        const double ly = field[(uint32_t)x + (uint32_t)g.n[0] * ((uint32_t)ys + (uint32_t)g.n[1] * (uint32_t)z)];
        const double lz = field[(uint32_t)x + (uint32_t)g.n[0] * ((uint32_t)y + (uint32_t)g.n[1] * (uint32_t)zs)];
        val = l0 * lx + l0 * ly + l0 * lz;
    }
    const double tot = block_sum(val, red);
    if (threadIdx.x == 0) partials[blockIdx.y * gridDim.x + blockIdx.x] = tot;
}
__global__ void __launch_bounds__(1024)
    correlator_final_kernel(const double* __restrict__ partials, size_t n_per_r, double scale, double* __restrict__ dst)
{
    __shared__ double red[32];
    const double* src = partials + (size_t)blockIdx.x * n_per_r;
    double acc = 0.0;
    for (size_t i = threadIdx.x; i < n_per_r; i += 1024) acc += src[i];
    const double tot = block_sum(acc, red);
    if (threadIdx.x == 0) dst[blockIdx.x] = tot * scale;
}

// ------------------------------------------------------------------ layout conversion
// canonical [s][mu] <-> device [p][mu][h]; one thread per (s, mu)
template <typename Real, bool TO_DEVICE>
__global__ void __launch_bounds__(kBlock)
    layout_kernel(typename LinkPtr<Real>::type* __restrict__ canonical, typename LinkPtr<Real>::type* __restrict__ links,
                  const Geom g)
{
    const uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    const uint64_t nlinks = 8ull * g.vh;
    if (i >= nlinks) return;
    const uint32_t s = (uint32_t)(i >> 2);
    const int mu = (int)(i & 3);
    const uint32_t x = s % (uint32_t)g.n[0];
    uint32_t q = s / (uint32_t)g.n[0];
    const uint32_t y = q % (uint32_t)g.n[1];
    q /= (uint32_t)g.n[1];
    const uint32_t z = q % (uint32_t)g.n[2], t = q / (uint32_t)g.n[2];
    const int p = (int)((x + y + z + t) & 1u);
    typename LinkPtr<Real>::type* dev = links + (size_t)(p * 4 + mu) * g.vh + (s >> 1);
    if (TO_DEVICE) *dev = canonical[i];
    else canonical[i] = *dev;
}

// ------------------------------------------------------------------ launchers
static inline unsigned blocks_for(uint64_t n) { return (unsigned)((n + kBlock - 1) / kBlock); }

size_t partials_needed(const Geom& g)
{
    const uint64_t v3 = (uint64_t)g.n[0] * g.n[1] * g.n[2];
    size_t a = 2 * (size_t)blocks_for(g.vh);
    if (g.tile >= 0) {  // one partial per 128-thread tile and parity
        const size_t t = 2 * (size_t)g.nb[0] * g.nb[1] * g.nb[2] * g.nb[3];
        if (t > a) a = t;
    }
    size_t b = (size_t)kMaxR * blocks_for(v3);
    return a > b ? a : b;
}

template <typename Real>
static void launch_plaquette_t(const void* links, const Geom& g, const Scratch& sc, size_t* n_partials,
                               cudaStream_t st)
{
    typedef typename LinkPtr<Real>::type L;
    if (g.tile >= 0) {
        const dim3 grid(2u * (unsigned)g.nb[0], (unsigned)g.nb[1], (unsigned)(g.nb[2] * g.nb[3]));
        *n_partials = (size_t)grid.x * grid.y * grid.z;
        if (g.tile == 0)
            plaquette_tiled_kernel<Real, kTiles[0][0], kTiles[0][1], kTiles[0][2], kTiles[0][3]>
                <<<grid, 1 << (kTiles[0][0] + kTiles[0][1] + kTiles[0][2] + kTiles[0][3]), 0, st>>>((const L*)links, g,
                                                                                                    sc.partials);
        else
            plaquette_tiled_kernel<Real, kTiles[1][0], kTiles[1][1], kTiles[1][2], kTiles[1][3]>
                <<<grid, 1 << (kTiles[1][0] + kTiles[1][1] + kTiles[1][2] + kTiles[1][3]), 0, st>>>((const L*)links, g,
                                                                                                    sc.partials);
    } else {
        const dim3 grid(blocks_for((uint64_t)g.st * g.nt_upd), 2);
        *n_partials = (size_t)grid.x * 2;
        plaquette_kernel<Real><<<grid, kBlock, 0, st>>>((const L*)links, g, sc.partials);
    }
}

int launch_plaquette(const void* links, const Geom& g, int precision, const Scratch& sc, double* dev_dst,
                     cudaStream_t st, double scale_in)
{
    size_t n = 0;
    if (precision == 32)
        launch_plaquette_t<float>(links, g, sc, &n, st);
    else
        launch_plaquette_t<double>(links, g, sc, &n, st);
    const double scale = scale_in != 0.0 ? scale_in : 1.0 / (6.0 * 2.0 * (double)g.vh);
    final_sum_kernel<<<1, 1024, 0, st>>>(sc.partials, n, scale, dev_dst);
    return 2;
}

// su2_run: the loop state the captured step reads and its last kernel advances
__global__ void set_run_state_kernel(RunState* state, double inv_beta, double* out, uint32_t sweep, uint32_t index)
{
    state += blockIdx.x * blockDim.x + threadIdx.x;  // one thread per copy
    state->inv_beta = inv_beta;
    state->out = out;
    state->sweep = sweep;
    state->index = index;
}
int launch_set_run_state(RunState* state, double inv_beta, double* out, uint32_t sweep, uint32_t index,
                         cudaStream_t st)
{
    set_run_state_kernel<<<kRunCopies / 256, 256, 0, st>>>(state, inv_beta, out, sweep, index);
    return 1;
}

int launch_final_sum(const double* partials, size_t n, double scale, double* dev_dst, cudaStream_t st)
{
    final_sum_kernel<<<1, 1024, 0, st>>>(partials, n, scale, dev_dst);
    return 1;
}

template <typename Real>
static unsigned launch_polyakov_t(const void* links, const Geom& g, const Scratch& sc, const StepTail& tl,
                                  bool overlap, cudaStream_t st, int nrep = 1)
{
    typedef typename LinkPtr<Real>::type L;
    const uint64_t v3 = (uint64_t)g.n[0] * g.n[1] * g.n[2];
    const int nt = g.n[3];
    // split only while one thread per site cannot fill the GPU (fewer than ~1 CTA wave of sites)
    const bool small = v3 < 148ull * 1024ull;
    if (small && nt >= 16 && nt % 4 == 0) {
        const unsigned grid = (unsigned)((v3 + kBlock / 4 - 1) / (kBlock / 4));
        launch_ex(polyakov_split_kernel<Real, 4>, dim3(grid, (unsigned)nrep), dim3(kBlock), st, overlap, (const L*)links, g, sc.field,
                  sc.partials, tl);
        return grid;
    }
    if (small && nt >= 8 && nt % 2 == 0) {
        const unsigned grid = (unsigned)((v3 + kBlock / 2 - 1) / (kBlock / 2));
        launch_ex(polyakov_split_kernel<Real, 2>, dim3(grid, (unsigned)nrep), dim3(kBlock), st, overlap, (const L*)links, g, sc.field,
                  sc.partials, tl);
        return grid;
    }
    const unsigned grid = blocks_for(v3);
    launch_ex(polyakov_kernel<Real>, dim3(grid, (unsigned)nrep), dim3(kBlock), st, overlap, (const L*)links, g, sc.field, sc.partials,
              tl);
    return grid;
}

int launch_polyakov_partials(const void* links, const Geom& g, int precision, const Scratch& sc, size_t* n_partials,
                             cudaStream_t st)
{
    const StepTail none = {};
    *n_partials = precision == 32 ? launch_polyakov_t<float>(links, g, sc, none, false, st)
                                  : launch_polyakov_t<double>(links, g, sc, none, false, st);
    return 1;
}

// the last kernel of a step: Polyakov loop + both final sums (see step_tail)
int launch_polyakov_step(const void* links, const Geom& g, int precision, const Scratch& sc, const double* epart,
                         size_t n_epart, double scale_plaq, double* dev_dst, RunState* state, bool overlap,
                         cudaStream_t st, int nrep, unsigned advance)
{
    const uint64_t v3 = (uint64_t)g.n[0] * g.n[1] * g.n[2];
    const StepTail tl = {epart, n_epart, scale_plaq, 1.0 / (double)v3, sc.slots, sc.ticket, dev_dst, state, advance};
    if (precision == 32)
        launch_polyakov_t<float>(links, g, sc, tl, overlap, st, nrep);
    else
        launch_polyakov_t<double>(links, g, sc, tl, overlap, st, nrep);
    return 1;
}

int launch_polyakov(const void* links, const Geom& g, int precision, const Scratch& sc, double* dev_dst,
                    cudaStream_t st)
{
    size_t n = 0;
    launch_polyakov_partials(links, g, precision, sc, &n, st);
    const uint64_t v3 = (uint64_t)g.n[0] * g.n[1] * g.n[2];
    final_sum_kernel<<<1, 1024, 0, st>>>(sc.partials, n, 1.0 / (double)v3, dev_dst);
    return 2;
}

int launch_polyakov_chain(const void* links, const Geom& g, int precision, const Scratch& sc, const void* prev,
                          void* next, double* dev_dst, cudaStream_t st)
{
    const uint64_t v3 = (uint64_t)g.n[0] * g.n[1] * g.n[2];
    const unsigned grid = blocks_for(v3);
    if (precision == 32)
        polyakov_chain_kernel<float><<<grid, kBlock, 0, st>>>((const float4*)links, g, (const float4*)prev, (float4*)next,
                                                              sc.partials);
    else
        polyakov_chain_kernel<double><<<grid, kBlock, 0, st>>>((const double4a*)links, g, (const double4a*)prev,
                                                               (double4a*)next, sc.partials);
    if (!dev_dst) return 1;
    final_sum_kernel<<<1, 1024, 0, st>>>(sc.partials, grid, 1.0 / (double)v3, dev_dst);
    return 2;
}

int launch_polyakov_correlator(const Geom& g, const Scratch& sc, int rmax, double* dev_dst, cudaStream_t st)
{
    const uint64_t v3 = (uint64_t)g.n[0] * g.n[1] * g.n[2];
    const dim3 grid(blocks_for(v3), (unsigned)rmax);
    correlator_kernel<<<grid, kBlock, 0, st>>>(sc.field, g, sc.partials);
    correlator_final_kernel<<<(unsigned)rmax, 1024, 0, st>>>(sc.partials, grid.x, 1.0 / (3.0 * (double)v3), dev_dst);
    return 2;
}

int launch_to_device_layout(const void* canonical, void* links, const Geom& g, int precision, cudaStream_t st)
{
    const unsigned grid = blocks_for(8ull * g.vh);
    if (precision == 32)
        layout_kernel<float, true><<<grid, kBlock, 0, st>>>((float4*)canonical, (float4*)links, g);
    else
        layout_kernel<double, true><<<grid, kBlock, 0, st>>>((double4a*)canonical, (double4a*)links, g);
    return 1;
}
int launch_to_canonical(const void* links, void* canonical, const Geom& g, int precision, cudaStream_t st)
{
    const unsigned grid = blocks_for(8ull * g.vh);
    if (precision == 32)
        layout_kernel<float, false><<<grid, kBlock, 0, st>>>((float4*)canonical, (float4*)links, g);
    else
        layout_kernel<double, false><<<grid, kBlock, 0, st>>>((double4a*)canonical, (double4a*)links, g);
    return 1;
}

// ------------------------------------------------------------------ no-allocation mean plaquette
// su2_mean_plaquette_noalloc (include/su2_heatbath.h): row 7 for callers that cannot call cudaMalloc (code under
// CUDA graph capture, tight serving loops, harnesses that forbid it). The per-CTA partial sums - the scratch of the
// plaquette kernels, library-allocated per handle everywhere else - live in this file-scope array instead: every GPU
// that loads the library holds its 2 MiB until exit. One partial per 128 (tiled) or 256 (linear) sites, so it
// serves lattices of up to kNoAllocMaxPartials * 128 = 2^25 sites (64^4 is 2^24).
// All calls share the array: it keeps the previous call's partials, none of which is read (every launch writes
// the n partials its final sum reads, nothing needs to start at zero); calls that overlap on the GPU race.
constexpr size_t kNoAllocMaxPartials = size_t(1) << 18;
static __device__ __align__(256) double g_noalloc_partials[kNoAllocMaxPartials];

// variant of final_sum_kernel that names the static array itself (device code may; host code needs the address)
__global__ void __launch_bounds__(1024) final_sum_static_kernel(size_t n, double scale, double* __restrict__ dst)
{
    __shared__ double red[32];
    double acc = 0.0;
    for (size_t i = threadIdx.x; i < n; i += 1024) acc += g_noalloc_partials[i];
    const double tot = block_sum(acc, red);
    if (threadIdx.x == 0) dst[0] = tot * scale;
}

// In host code `g_noalloc_partials` is a host-side stand-in, not a device address: the plaquette kernels take the
// address cudaGetSymbolAddress returns, looked up once per device with that device current.
static double* noalloc_partials_of_current_device(cudaError_t* ce)
{
    constexpr int kMaxDevices = 64;
    static double* ptr[kMaxDevices] = {};
    int dev = -1;
    *ce = cudaGetDevice(&dev);
    if (*ce != cudaSuccess) return nullptr;
    if (dev < 0 || dev >= kMaxDevices) {
        *ce = cudaErrorInvalidDevice;
        return nullptr;
    }
    if (!ptr[dev]) {
        double* p = nullptr;
        *ce = cudaGetSymbolAddress((void**)&p, g_noalloc_partials);
        if (*ce != cudaSuccess) return nullptr;
        ptr[dev] = p;
    }
    return ptr[dev];
}

size_t noalloc_max_partials() { return kNoAllocMaxPartials; }

// returns an SU2_* code (0 ok, 3 CUDA error, 5 too large); enqueues 2 kernels on `st`, allocates nothing
int launch_plaquette_noalloc(const void* links, const Geom& g, int precision, double* dev_dst, cudaStream_t st)
{
    // partials the launch will write (same formula as launch_plaquette_t)
    const size_t need = g.tile >= 0 ? 2 * (size_t)g.nb[0] * g.nb[1] * g.nb[2] * g.nb[3]
                                    : 2 * (size_t)blocks_for((uint64_t)g.st * g.nt_upd);
    if (need > kNoAllocMaxPartials) return 5;
    cudaError_t ce = cudaSuccess;
    Scratch sc = {};
    sc.partials = noalloc_partials_of_current_device(&ce);
    if (!sc.partials) {
        cudaGetLastError();
        return 3;
    }
    sc.n_partials = kNoAllocMaxPartials;
    size_t n = 0;
    if (precision == 32)
        launch_plaquette_t<float>(links, g, sc, &n, st);
    else
        launch_plaquette_t<double>(links, g, sc, &n, st);
    final_sum_static_kernel<<<1, 1024, 0, st>>>(n, 1.0 / (6.0 * 2.0 * (double)g.vh), dev_dst);
    return cudaGetLastError() == cudaSuccess ? 0 : 3;
}

}  // namespace su2
