/*
 * su2_oracle.c — plain serial CPU oracle for the SU(2) heat-bath path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT. Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may build, load or call this
 * file. It shares no code, header, table or helper with the CUDA path under
 * paper_1104_5432_b200/csrc/; both are written from DESIGN.md §3 (the written
 * readings), which restates SURVEY.md §8(c).
 *
 * What the paper fixes: the workload — "random SU(2) matrix initialization
 * followed by 100 iterations of the heat bath method and the calculation of
 * the mean average plaquette at each iteration" (§2.1) — and the
 * Polyakov loop as order parameter (eq. 1). The paper prints
 * no formula for the action, the staple or the draw (it defers to its ref. [1],
 * PAPER.md:23); those follow BASELINE.json north_star and the textbook
 * definitions it names (Wilson action; Kennedy–Pendleton 1985). Every such
 * reading is tagged [R<n>] below and listed in DESIGN.md §3.
 *
 * Style: no blocking, fusion or reordering; a site loop, a direction loop and
 * the formulas in the order DESIGN.md states them. General dimension D = 2..4
 * at run time (D = 2 is needed for the exact I2/I1 pin).
 *
 * Compiled three times into one shared object (see oracle/build.py):
 *   -DORC_SFX=f64  REAL=double AREAL=double   fp64 mode
 *   -DORC_SFX=f32  REAL=float  AREAL=float    fp32 mode (float arithmetic)
 *   -DORC_SFX=f32x REAL=float  AREAL=double   fp32 storage + fp32 uniform rule,
 *                                             fp64 arithmetic (reference precision,
 *                                             DESIGN.md §3 [R12])
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors and
 * ATen's host engine; quaternion algebra vs 2x2 complex matrices; staple vs sum
 * of plaquettes; KP law vs I2/I1 and the closed-form acceptance; single-link
 * heat bath on 2^4 vs brute-force quadrature; cold plaquette = 1; gauge
 * invariance; Polyakov centre flip; D=2 equilibrium plaquette = I2(b)/I1(b);
 * D=4 Schwinger–Dyson identity; visiting-order independence; Creutz draw [R15]
 * vs I2/I1, (pi/2) I1/sinh and the quadrature CDF; the staple norm k returned
 * beside the margin vs the norm of the (pinned) staple; Polyakov-loop correlator:
 * cold C(r) = 1, a field with one non-trivial line, gauge invariance,
 * C(r) = C(N - r), factorisation on x-independent configurations.
 * Unpinned: D=4 <L> values across the N_t=4 transition (the paper prints none).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef ORC_REAL
#define ORC_REAL double
#endif
#ifndef ORC_AREAL
#define ORC_AREAL double
#endif
#ifndef ORC_SFX
#define ORC_SFX f64
#endif
#ifndef ORC_UNIFORM_BITS
#define ORC_UNIFORM_BITS 64 /* which uniform rule: 64 -> fp64 rule, 32 -> fp32 rule */
#endif

#define ORC_CAT2(a, b) a##_##b
#define ORC_CAT(a, b) ORC_CAT2(a, b)
#define FN(name) ORC_CAT(name, ORC_SFX)

typedef ORC_REAL REAL;   /* storage type of the links */
typedef ORC_AREAL AREAL; /* arithmetic type */

#define ORC_MAXD 4
#define ORC_OK 0
#define ORC_EARG 1
#define ORC_ETRIALS 5

/* ---- math in the arithmetic type ------------------------------------- */
#if defined(ORC_AREAL_IS_FLOAT)
#define A_SQRT sqrtf
#define A_LOG logf
#define A_EXP expf
#define A_COS cosf
#define A_SIN sinf
#define A_TWO_PI 6.28318530717958647692f
#else
#define A_SQRT sqrt
#define A_LOG log
#define A_EXP exp
#define A_COS cos
#define A_SIN sin
#define A_TWO_PI 6.28318530717958647692
#endif

/* ====================================================================== */
/* Philox4x32-10 [R5]: Salmon, Moraes, Dror, Shaw, SC'11. 128-bit counter,   */
/* 64-bit key, 10 rounds; round multipliers 0xD2511F53, 0xCD9E8D57; key      */
/* increments (Weyl) 0x9E3779B9, 0xBB67AE85.                                 */
/* Emitted once (from the f64 translation unit).                             */
/* ====================================================================== */
#ifdef ORC_EMIT_COMMON
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
#else
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
#endif

/* Counter layout [R5]: (site s, sweep_idx, tag, call n); key = seed.        */
/* tag = (purpose<<8) | (parity<<2) | mu; purpose 0 heat bath, 1 init,       */
/* 2 test gauge transformation.                                              */
static void draw_words(uint64_t seed, uint32_t s, uint32_t sweep, uint32_t purpose,
                       uint32_t parity, uint32_t mu, uint32_t n, uint32_t w[4])
{
    uint32_t ctr[4], key[2];
    ctr[0] = s;
    ctr[1] = sweep;
    ctr[2] = (purpose << 8) | (parity << 2) | mu;
    ctr[3] = n;
    key[0] = (uint32_t)(seed & 0xFFFFFFFFu);
    key[1] = (uint32_t)(seed >> 32);
    orc_philox4x32_10(ctr, key, w);
}

/* Uniform in (0,1), exact in the mode's precision [R5]:                     */
/*   fp64 rule: u = (w + 0.5) * 2^-32                                        */
/*   fp32 rule: u = (2*(w>>9) + 1) * 2^-24   (23 random bits, odd numerator) */
static AREAL uniform_from_word(uint32_t w)
{
#if ORC_UNIFORM_BITS == 64
    return (AREAL)(((double)w + 0.5) * (1.0 / 4294967296.0));
#else
    return (AREAL)((float)(2u * (w >> 9) + 1u) * (1.0f / 16777216.0f));
#endif
}
AREAL FN(orc_uniform)(uint32_t w) { return uniform_from_word(w); }

/* ====================================================================== */
/* Quaternion algebra [R1]: U = a0 + i(a1 s1 + a2 s2 + a3 s3).               */
/*   (ab)0 = a0 b0 - a.b ;  (ab)vec = a0 b + b0 a - a x b ;  dagger = (a0,-a) */
/* ====================================================================== */
static void qmul(const AREAL a[4], const AREAL b[4], AREAL c[4])
{
    c[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
    c[1] = a[0] * b[1] + b[0] * a[1] - (a[2] * b[3] - a[3] * b[2]);
    c[2] = a[0] * b[2] + b[0] * a[2] - (a[3] * b[1] - a[1] * b[3]);
    c[3] = a[0] * b[3] + b[0] * a[3] - (a[1] * b[2] - a[2] * b[1]);
}
static void qdag(const AREAL a[4], AREAL d[4])
{
    d[0] = a[0]; d[1] = -a[1]; d[2] = -a[2]; d[3] = -a[3];
}
void FN(orc_qmul)(const REAL *a, const REAL *b, REAL *c)
{
    AREAL x[4], y[4], z[4];
    for (int i = 0; i < 4; ++i) { x[i] = a[i]; y[i] = b[i]; }
    qmul(x, y, z);
    for (int i = 0; i < 4; ++i) c[i] = (REAL)z[i];
}

/* ====================================================================== */
/* Geometry: site s = x0 + N0 (x1 + N1 (x2 + ...)), x0 fastest; periodic.    */
/* Canonical storage: links[(s*D + mu)*4 + c].                               */
/* ====================================================================== */
typedef struct {
    int D;
    int n[ORC_MAXD];
    int64_t stride[ORC_MAXD];
    int64_t V;
} geom_t;

static int geom_init(geom_t *g, int D, const int *dims)
{
    if (D < 2 || D > ORC_MAXD || !dims) return ORC_EARG;
    g->D = D;
    g->V = 1;
    for (int d = 0; d < D; ++d) {
        if (dims[d] < 2 || (dims[d] & 1)) return ORC_EARG; /* even extents: checkerboard [R4] */
        g->n[d] = dims[d];
        g->stride[d] = g->V;
        g->V *= dims[d];
    }
    if (g->V >= ((int64_t)1 << 32)) return ORC_EARG; /* s is a 32-bit Philox word */
    return ORC_OK;
}
static void site_coords(const geom_t *g, int64_t s, int x[ORC_MAXD])
{
    for (int d = 0; d < g->D; ++d) { x[d] = (int)(s % g->n[d]); s /= g->n[d]; }
}
static int64_t site_index(const geom_t *g, const int x[ORC_MAXD])
{
    int64_t s = 0;
    for (int d = 0; d < g->D; ++d) s += g->stride[d] * x[d];
    return s;
}
static int site_parity(const geom_t *g, const int x[ORC_MAXD])
{
    int p = 0;
    for (int d = 0; d < g->D; ++d) p += x[d];
    return p & 1;
}
/* neighbour of x shifted by +1 (dir>0) or -1 (dir<0) along d, periodic */
static void shifted(const geom_t *g, const int x[ORC_MAXD], int d, int dir, int y[ORC_MAXD])
{
    for (int e = 0; e < g->D; ++e) y[e] = x[e];
    y[d] = (x[d] + dir + g->n[d]) % g->n[d];
}
static void load_link(const geom_t *g, const REAL *links, const int x[ORC_MAXD], int mu, AREAL u[4])
{
    const REAL *p = links + (site_index(g, x) * g->D + mu) * 4;
    for (int c = 0; c < 4; ++c) u[c] = (AREAL)p[c];
}

/* ====================================================================== */
/* Init [R9] ("random SU(2) matrix initialization").             */
/* cold: (1,0,0,0). hot: Shoemake's uniform unit quaternion from 3 uniforms: */
/*   a = (sqrt(1-u1) sin 2pi u2, sqrt(1-u1) cos 2pi u2,                      */
/*        sqrt(u1) sin 2pi u3,   sqrt(u1) cos 2pi u3)                        */
/* counter (s, 0, (1<<8)|(p<<2)|mu, 0).                                      */
/* ====================================================================== */
static void haar_from_words(const uint32_t w[4], AREAL a[4])
{
    AREAL u1 = uniform_from_word(w[0]);
    AREAL u2 = uniform_from_word(w[1]);
    AREAL u3 = uniform_from_word(w[2]);
    AREAL r1 = A_SQRT((AREAL)1 - u1);
    AREAL r2 = A_SQRT(u1);
    a[0] = r1 * A_SIN(A_TWO_PI * u2);
    a[1] = r1 * A_COS(A_TWO_PI * u2);
    a[2] = r2 * A_SIN(A_TWO_PI * u3);
    a[3] = r2 * A_COS(A_TWO_PI * u3);
}

int FN(orc_init)(int D, const int *dims, int start, uint64_t seed, REAL *links)
{
    geom_t g;
    if (geom_init(&g, D, dims) || !links || (start != 0 && start != 1)) return ORC_EARG;
    for (int64_t s = 0; s < g.V; ++s) {
        int x[ORC_MAXD];
        site_coords(&g, s, x);
        int p = site_parity(&g, x);
        for (int mu = 0; mu < D; ++mu) {
            REAL *u = links + (s * D + mu) * 4;
            if (start == 0) {
                u[0] = 1; u[1] = 0; u[2] = 0; u[3] = 0;
            } else {
                uint32_t w[4];
                AREAL a[4];
                draw_words(seed, (uint32_t)s, 0u, 1u, (uint32_t)p, (uint32_t)mu, 0u, w);
                haar_from_words(w, a);
                for (int c = 0; c < 4; ++c) u[c] = (REAL)a[c];
            }
        }
    }
    return ORC_OK;
}

/* ====================================================================== */
/* Staple sum [R3] for the link U_mu(x): over the D-1 directions nu != mu,   */
/* nu ascending, forward term then backward term, products left to right:    */
/*   fwd = U_nu(x+mu) . U_mu^dag(x+nu) . U_nu^dag(x)                         */
/*   bwd = U_nu^dag(x+mu-nu) . U_mu^dag(x-nu) . U_nu(x-nu)                   */
/* so that sum over the 2(D-1) plaquettes through the link of 1/2 Tr U_P     */
/* equals 1/2 Tr( U_mu(x) v ).                                               */
/* ====================================================================== */
static void staple_sum(const geom_t *g, const REAL *links, const int x[ORC_MAXD], int mu, AREAL v[4])
{
    v[0] = v[1] = v[2] = v[3] = 0;
    int xpmu[ORC_MAXD];
    shifted(g, x, mu, +1, xpmu);
    for (int nu = 0; nu < g->D; ++nu) {
        if (nu == mu) continue;
        int xpnu[ORC_MAXD], xmnu[ORC_MAXD], xpmumnu[ORC_MAXD];
        shifted(g, x, nu, +1, xpnu);
        shifted(g, x, nu, -1, xmnu);
        shifted(g, xpmu, nu, -1, xpmumnu);
        AREAL a[4], b[4], c[4], bd[4], cd[4], ad[4], t[4], f[4];

        /* forward */
        load_link(g, links, xpmu, nu, a);
        load_link(g, links, xpnu, mu, b);
        load_link(g, links, x, nu, c);
        qdag(b, bd);
        qdag(c, cd);
        qmul(a, bd, t);
        qmul(t, cd, f);
        for (int i = 0; i < 4; ++i) v[i] += f[i];

        /* backward */
        load_link(g, links, xpmumnu, nu, a);
        load_link(g, links, xmnu, mu, b);
        load_link(g, links, xmnu, nu, c);
        qdag(a, ad);
        qdag(b, bd);
        qmul(ad, bd, t);
        qmul(t, c, f);
        for (int i = 0; i < 4; ++i) v[i] += f[i];
    }
}

int FN(orc_staple)(int D, const int *dims, const REAL *links, int64_t s, int mu, REAL *v_out)
{
    geom_t g;
    if (geom_init(&g, D, dims) || s < 0 || s >= g.V || mu < 0 || mu >= D) return ORC_EARG;
    int x[ORC_MAXD];
    AREAL v[4];
    site_coords(&g, s, x);
    staple_sum(&g, links, x, mu, v);
    for (int i = 0; i < 4; ++i) v_out[i] = (REAL)v[i];
    return ORC_OK;
}

/* Norms k of the staple sums of all links, k_out[s*D+mu] (for the
 * Schwinger–Dyson pin 6<P> = <k I2(bk)/I1(bk)>, evaluated in the test). */
int FN(orc_staple_norms)(int D, const int *dims, const REAL *links, double *k_out)
{
    geom_t g;
    if (geom_init(&g, D, dims)) return ORC_EARG;
    for (int64_t s = 0; s < g.V; ++s) {
        int x[ORC_MAXD];
        site_coords(&g, s, x);
        for (int mu = 0; mu < D; ++mu) {
            AREAL v[4];
            staple_sum(&g, links, x, mu, v);
            k_out[s * D + mu] = sqrt((double)(v[0] * v[0] + v[1] * v[1] + v[2] * v[2] + v[3] * v[3]));
        }
    }
    return ORC_OK;
}

/* ====================================================================== */
/* Kennedy–Pendleton draw of x0 with density ~ sqrt(1-x0^2) exp(alpha x0)    */
/* [R6]. Trial n = 1,2,...: (R,R',R'',R''') = u(words of Philox(..., n));     */
/*   delta = -( ln R + cos^2(2 pi R') ln R'' ) / alpha                       */
/*   accept iff R'''^2 <= 1 - delta/2 ;  x0 = 1 - delta.                     */
/* Returns delta (not x0) so the caller can form sqrt(delta(2-delta)).       */
/* *margin = smallest |R'''^2 - (1 - delta/2)| over the trials made.         */
/* ====================================================================== */
#define ORC_MAX_TRIALS 10000
static int kp_delta(AREAL alpha, uint64_t seed, uint32_t s, uint32_t sweep, uint32_t parity,
                    uint32_t mu, AREAL *delta_out, int *trials_out, AREAL *margin_out)
{
    AREAL margin = (AREAL)1e30;
    for (int n = 1; n <= ORC_MAX_TRIALS; ++n) {
        uint32_t w[4];
        draw_words(seed, s, sweep, 0u, parity, mu, (uint32_t)n, w);
        AREAL R = uniform_from_word(w[0]);
        AREAL Rp = uniform_from_word(w[1]);
        AREAL Rpp = uniform_from_word(w[2]);
        AREAL Rppp = uniform_from_word(w[3]);
        AREAL c = A_COS(A_TWO_PI * Rp);
        AREAL delta = -(A_LOG(R) + c * c * A_LOG(Rpp)) / alpha;
        AREAL lhs = Rppp * Rppp;
        AREAL rhs = (AREAL)1 - delta / (AREAL)2;
        AREAL m = lhs - rhs;
        if (m < 0) m = -m;
        if (m < margin) margin = m;
        if (lhs <= rhs) {
            *delta_out = delta;
            if (trials_out) *trials_out = n;
            if (margin_out) *margin_out = margin;
            return ORC_OK;
        }
    }
    return ORC_ETRIALS;
}

/* Stand-alone KP draw for the x0-law pins: returns x0 = 1 - delta. */
int FN(orc_kp_x0)(double alpha, uint64_t seed, uint32_t s, uint32_t sweep, double *x0_out, int *trials_out)
{
    AREAL delta;
    int rc = kp_delta((AREAL)alpha, seed, s, sweep, 0u, 0u, &delta, trials_out, NULL);
    if (rc) return rc;
    *x0_out = (double)((AREAL)1 - delta);
    return ORC_OK;
}

/* ====================================================================== */
/* Creutz's original draw [R15] (Creutz 1980; north_star "Creutz/Kennedy-     */
/* Pendleton"): propose x0 with density ~ exp(alpha x0) on [-1,1] by          */
/* inversion, accept with probability sqrt(1 - x0^2). Trial n = 1,2,...:      */
/*   (R, R', ., .) = u(words of Philox(..., n))                               */
/*   delta = 1 - x0 = -ln( R + (1 - R) exp(-2 alpha) ) / alpha                */
/*   accept iff R'^2 <= 1 - x0^2 = delta (2 - delta).                         */
/* Same target law as [R6]; acceptance (pi/2) I1(alpha)/sinh(alpha), which    */
/* beats KP's below alpha_c = 1.6847 (where the two are equal).               */
/* *margin = smallest |R'^2 - delta(2-delta)| over the trials made.           */
/* ====================================================================== */
#define ORC_DRAW_KP 0
#define ORC_DRAW_AUTO 1   /* per link: Creutz iff alpha < ORC_ALPHA_C */
#define ORC_DRAW_CREUTZ 2 /* always Creutz */
#define ORC_ALPHA_C 1.6847
static int g_draw_method = ORC_DRAW_KP;

int FN(orc_set_draw)(int method)
{
    if (method < 0 || method > 2) return ORC_EARG;
    g_draw_method = method;
    return ORC_OK;
}

static int creutz_delta(AREAL alpha, uint64_t seed, uint32_t s, uint32_t sweep, uint32_t parity,
                        uint32_t mu, AREAL *delta_out, int *trials_out, AREAL *margin_out)
{
    AREAL margin = (AREAL)1e30;
    AREAL E = A_EXP(-(AREAL)2 * alpha);
    for (int n = 1; n <= ORC_MAX_TRIALS; ++n) {
        uint32_t w[4];
        draw_words(seed, s, sweep, 0u, parity, mu, (uint32_t)n, w);
        AREAL R = uniform_from_word(w[0]);
        AREAL Rp = uniform_from_word(w[1]);
        AREAL delta = -A_LOG(R + ((AREAL)1 - R) * E) / alpha;
        AREAL lhs = Rp * Rp;
        AREAL rhs = delta * ((AREAL)2 - delta);
        AREAL m = lhs - rhs;
        if (m < 0) m = -m;
        if (m < margin) margin = m;
        if (lhs <= rhs) {
            *delta_out = delta;
            if (trials_out) *trials_out = n;
            if (margin_out) *margin_out = margin;
            return ORC_OK;
        }
    }
    return ORC_ETRIALS;
}

/* Stand-alone Creutz draw for the x0-law pins: returns x0 = 1 - delta. */
int FN(orc_creutz_x0)(double alpha, uint64_t seed, uint32_t s, uint32_t sweep, double *x0_out, int *trials_out)
{
    AREAL delta;
    int rc = creutz_delta((AREAL)alpha, seed, s, sweep, 0u, 0u, &delta, trials_out, NULL);
    if (rc) return rc;
    *x0_out = (double)((AREAL)1 - delta);
    return ORC_OK;
}

/* ====================================================================== */
/* Heat-bath update of one link [R2][R4][R6][R7][R8]. Local weight           */
/* exp(beta 1/2 Tr(U v)) = exp(beta k 1/2 Tr(U Vbar)), k = |v|, Vbar = v/k.  */
/* X = U Vbar has density ~ exp(alpha x0) dHaar, alpha = beta k; U' = X Vbar^dag. */
/* The new link does not depend on the old one.                              */
/* ====================================================================== */
#if defined(ORC_AREAL_IS_FLOAT)
#define DEGENERATE_K2 1e-20f
#else
#define DEGENERATE_K2 1e-30
#endif

/* *knorm (nullable) = the staple norm k of this link as the update saw it: the draw divides the
 * staple by it (Vbar = v/k), so 1/k is the factor by which a perturbation of the neighbouring
 * links reaches the new link - the parity harness classifies ill-conditioned links with it
 * (DESIGN.md 3 [R13b]). *delta (nullable) = the accepted delta = 1 - x0 of the draw: the vector part of X
 * lives on a sphere of radius sqrt(delta (2 - delta)), which amplifies a rounding of delta by
 * |1 - delta| / radius (same use). */
static int heatbath_link(const geom_t *g, const REAL *links, double beta, uint64_t seed,
                         uint32_t sweep, int64_t s, int mu, AREAL unew[4], int *trials, AREAL *margin,
                         double *knorm, double *delta_out)
{
    int x[ORC_MAXD];
    site_coords(g, s, x);
    int p = site_parity(g, x);
    AREAL v[4];
    staple_sum(g, links, x, mu, v);
    AREAL k2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2] + v[3] * v[3];

    uint32_t wd[4];
    draw_words(seed, (uint32_t)s, sweep, 0u, (uint32_t)p, (uint32_t)mu, 0u, wd); /* n = 0: direction */

    if (k2 < DEGENERATE_K2) { /* [R8] measure-zero case: Haar-uniform new link */
        haar_from_words(wd, unew);
        if (trials) *trials = 0;
        if (margin) *margin = (AREAL)1;
        if (knorm) *knorm = 0.0;
        if (delta_out) *delta_out = 1.0;
        return ORC_OK;
    }
    AREAL k = A_SQRT(k2);
    if (knorm) *knorm = (double)k;
    AREAL alpha = (AREAL)beta * k;

    AREAL delta;
    int rc;
    if (g_draw_method == ORC_DRAW_CREUTZ || (g_draw_method == ORC_DRAW_AUTO && alpha < (AREAL)ORC_ALPHA_C))
        rc = creutz_delta(alpha, seed, (uint32_t)s, sweep, (uint32_t)p, (uint32_t)mu, &delta, trials, margin); /* [R15] */
    else
        rc = kp_delta(alpha, seed, (uint32_t)s, sweep, (uint32_t)p, (uint32_t)mu, &delta, trials, margin);
    if (rc) return rc;
    if (g_draw_method == ORC_DRAW_AUTO && margin) { /* a rounding-decided choice of method is excusable too */
        AREAL mc = alpha - (AREAL)ORC_ALPHA_C;
        if (mc < 0) mc = -mc;
        if (mc < *margin) *margin = mc;
    }

    if (delta_out) *delta_out = (double)delta;

    /* [R7] direction uniform on the sphere of radius sqrt(1-x0^2) = sqrt(delta(2-delta)) */
    AREAL x0 = (AREAL)1 - delta;
    AREAL r2 = delta * ((AREAL)2 - delta);
    AREAL r = A_SQRT(r2 > 0 ? r2 : 0);
    AREAL cth = (AREAL)1 - (AREAL)2 * uniform_from_word(wd[0]);
    AREAL phi = A_TWO_PI * uniform_from_word(wd[1]);
    AREAL s2 = (AREAL)1 - cth * cth;
    AREAL sth = A_SQRT(s2 > 0 ? s2 : 0);
    AREAL X[4];
    X[0] = x0;
    X[1] = r * sth * A_COS(phi);
    X[2] = r * sth * A_SIN(phi);
    X[3] = r * cth;

    AREAL vbd[4]; /* Vbar^dagger */
    vbd[0] = v[0] / k; vbd[1] = -v[1] / k; vbd[2] = -v[2] / k; vbd[3] = -v[3] / k;
    AREAL u[4];
    qmul(X, vbd, u);
    AREAL nrm = A_SQRT(u[0] * u[0] + u[1] * u[1] + u[2] * u[2] + u[3] * u[3]);
    for (int c = 0; c < 4; ++c) unew[c] = u[c] / nrm;
    return ORC_OK;
}

/* one link, result returned, lattice untouched (single-link pins) */
int FN(orc_heatbath_link)(int D, const int *dims, const REAL *links, double beta, uint64_t seed,
                          uint32_t sweep, int64_t s, int mu, REAL *u_out, int *trials, double *margin,
                          double *knorm, double *delta)
{
    geom_t g;
    if (geom_init(&g, D, dims) || s < 0 || s >= g.V || mu < 0 || mu >= D || !(beta > 0)) return ORC_EARG;
    AREAL u[4], m;
    int rc = heatbath_link(&g, links, beta, seed, sweep, s, mu, u, trials, &m, knorm, delta);
    if (rc) return rc;
    for (int c = 0; c < 4; ++c) u_out[c] = (REAL)u[c];
    if (margin) *margin = (double)m;
    return ORC_OK;
}

/* One sub-step (mu, parity) [R4]: every U_mu(x) with parity(x) = parity, in
 * place. `order` (nullable) is a permutation of 0..V-1 giving the visiting
 * order of the sites (order-independence pin); NULL = ascending s.
 * trials/margin/knorm/delta (nullable) are indexed [s*D+mu]. */
int FN(orc_heatbath_substep)(int D, const int *dims, REAL *links, double beta, uint64_t seed,
                             uint32_t sweep, int mu, int parity, const int64_t *order,
                             int32_t *trials, double *margin, double *knorm, double *delta)
{
    geom_t g;
    if (geom_init(&g, D, dims) || mu < 0 || mu >= D || (parity != 0 && parity != 1) || !(beta > 0) ||
        !isfinite(beta))
        return ORC_EARG;
    for (int64_t i = 0; i < g.V; ++i) {
        int64_t s = order ? order[i] : i;
        int x[ORC_MAXD];
        site_coords(&g, s, x);
        if (site_parity(&g, x) != parity) continue;
        AREAL u[4], m;
        int tr;
        double kn, dl;
        int rc = heatbath_link(&g, links, beta, seed, sweep, s, mu, u, &tr, &m, &kn, &dl);
        if (rc) return rc;
        REAL *dst = links + (s * D + mu) * 4;
        for (int c = 0; c < 4; ++c) dst[c] = (REAL)u[c];
        if (trials) trials[s * D + mu] = tr;
        if (margin) margin[s * D + mu] = (double)m;
        if (knorm) knorm[s * D + mu] = kn;
        if (delta) delta[s * D + mu] = dl;
    }
    return ORC_OK;
}

/* One sweep [R4]: for mu = 0..D-1: for parity = 0, 1: sub-step(mu, parity). */
int FN(orc_heatbath_sweep)(int D, const int *dims, REAL *links, double beta, uint64_t seed,
                           uint32_t sweep, int32_t *trials, double *margin, double *knorm, double *delta)
{
    for (int mu = 0; mu < D; ++mu)
        for (int parity = 0; parity < 2; ++parity) {
            int rc = FN(orc_heatbath_substep)(D, dims, links, beta, seed, sweep, mu, parity, NULL, trials, margin,
                                              knorm, delta);
            if (rc) return rc;
        }
    return ORC_OK;
}

/* ====================================================================== */
/* Mean plaquette [R10]:                                       */
/*   P = 1/(V D(D-1)/2) sum_x sum_{mu<nu} 1/2 Tr[U_mu(x) U_nu(x+mu)          */
/*                                         U_mu^dag(x+nu) U_nu^dag(x)]       */
/* summed in double with Neumaier compensation.                              */
/* ====================================================================== */
static void neumaier_add(double *sum, double *comp, double term)
{
    double t = *sum + term;
    if (fabs(*sum) >= fabs(term)) *comp += (*sum - t) + term;
    else *comp += (term - t) + *sum;
    *sum = t;
}

int FN(orc_mean_plaquette)(int D, const int *dims, const REAL *links, double *out)
{
    geom_t g;
    if (geom_init(&g, D, dims) || !links || !out) return ORC_EARG;
    double sum = 0.0, comp = 0.0;
    for (int64_t s = 0; s < g.V; ++s) {
        int x[ORC_MAXD];
        site_coords(&g, s, x);
        for (int mu = 0; mu < D; ++mu)
            for (int nu = mu + 1; nu < D; ++nu) {
                int xpmu[ORC_MAXD], xpnu[ORC_MAXD];
                shifted(&g, x, mu, +1, xpmu);
                shifted(&g, x, nu, +1, xpnu);
                AREAL a[4], b[4], c[4], d[4], cd[4], dd[4], t1[4], t2[4], pl[4];
                load_link(&g, links, x, mu, a);
                load_link(&g, links, xpmu, nu, b);
                load_link(&g, links, xpnu, mu, c);
                load_link(&g, links, x, nu, d);
                qdag(c, cd);
                qdag(d, dd);
                qmul(a, b, t1);
                qmul(t1, cd, t2);
                qmul(t2, dd, pl);
                neumaier_add(&sum, &comp, (double)pl[0]);
            }
    }
    *out = (sum + comp) / ((double)g.V * (double)(D * (D - 1) / 2));
    return ORC_OK;
}

/* 1/2 Tr of the single plaquette (s; mu,nu) — used by the staple pin. */
int FN(orc_plaquette_at)(int D, const int *dims, const REAL *links, int64_t s, int mu, int nu, double *out)
{
    geom_t g;
    if (geom_init(&g, D, dims) || s < 0 || s >= g.V || mu == nu || mu < 0 || mu >= D || nu < 0 || nu >= D)
        return ORC_EARG;
    int x[ORC_MAXD] = {0, 0, 0, 0}, xpmu[ORC_MAXD], xpnu[ORC_MAXD];
    site_coords(&g, s, x);
    shifted(&g, x, mu, +1, xpmu);
    shifted(&g, x, nu, +1, xpnu);
    AREAL a[4], b[4], c[4], d[4], cd[4], dd[4], t1[4], t2[4], pl[4];
    load_link(&g, links, x, mu, a);
    load_link(&g, links, xpmu, nu, b);
    load_link(&g, links, xpnu, mu, c);
    load_link(&g, links, x, nu, d);
    qdag(c, cd);
    qdag(d, dd);
    qmul(a, b, t1);
    qmul(t1, cd, t2);
    qmul(t2, dd, pl);
    *out = (double)pl[0];
    return ORC_OK;
}

/* ====================================================================== */
/* Polyakov loop [R11] (eq. 1): time direction = D-1,        */
/*   l(xs) = 1/2 Tr[ U_t(xs,0) U_t(xs,1) ... U_t(xs,N_t-1) ],                */
/*   returns the SIGNED spatial mean; field (nullable) gets l(xs), indexed by */
/*   the spatial lexicographic index.                                        */
/* ====================================================================== */
int FN(orc_polyakov_loop)(int D, const int *dims, const REAL *links, double *out, double *field)
{
    geom_t g;
    if (geom_init(&g, D, dims) || !links || !out) return ORC_EARG;
    int td = D - 1;
    int64_t Vs = g.V / g.n[td];
    double sum = 0.0, comp = 0.0;
    for (int64_t xs = 0; xs < Vs; ++xs) {
        int x[ORC_MAXD];
        site_coords(&g, xs, x); /* t = 0 because xs < Vs */
        AREAL prod[4] = {1, 0, 0, 0};
        for (int t = 0; t < g.n[td]; ++t) {
            x[td] = t;
            AREAL u[4], nxt[4];
            load_link(&g, links, x, td, u);
            qmul(prod, u, nxt);
            for (int c = 0; c < 4; ++c) prod[c] = nxt[c];
        }
        if (field) field[xs] = (double)prod[0];
        neumaier_add(&sum, &comp, (double)prod[0]);
    }
    *out = (sum + comp) / (double)Vs;
    return ORC_OK;
}

/* ====================================================================== */
/* Polyakov-loop correlator (eq. 3): the colour-averaged free */
/* energy is defined through 1/4 <Tr L(y) Tr L^dag(x)>. In SU(2) Tr L is real, */
/* so 1/4 Tr L(y) Tr L^dag(x) = l(y) l(x) with l = 1/2 Tr L as in [R11].      */
/* On-axis separations only (SURVEY.md 8(f) item 1 - the paper does not say   */
/* which separations it used): for r = 1..rmax                                */
/*   C(r) = 1/((D-1) Vs) sum_xs sum_{i spatial} l(xs) l(xs + r e_i), periodic. */
/* Written as the direct double loop over sites and axes, on the field l that */
/* orc_polyakov_loop defines (recomputed here the same way, product over t in */
/* order); sums in double with Neumaier compensation. out[r-1] = C(r).        */
/* ====================================================================== */
int FN(orc_polyakov_correlator)(int D, const int *dims, const REAL *links, int rmax, double *out)
{
    geom_t g;
    if (geom_init(&g, D, dims) || !links || !out || rmax < 1) return ORC_EARG;
    int td = D - 1;
    for (int i = 0; i < td; ++i)
        if (rmax > g.n[i] / 2) return ORC_EARG;
    int64_t Vs = g.V / g.n[td];
    double *l = (double *)malloc(sizeof(double) * (size_t)Vs);
    if (!l) return ORC_EARG;
    for (int64_t xs = 0; xs < Vs; ++xs) { /* l(xs) = 1/2 Tr prod_t U_t(xs, t) [R11] */
        int x[ORC_MAXD];
        site_coords(&g, xs, x);
        AREAL prod[4] = {1, 0, 0, 0};
        for (int t = 0; t < g.n[td]; ++t) {
            x[td] = t;
            AREAL u[4], nxt[4];
            load_link(&g, links, x, td, u);
            qmul(prod, u, nxt);
            for (int c = 0; c < 4; ++c) prod[c] = nxt[c];
        }
        l[xs] = (double)prod[0];
    }
    for (int r = 1; r <= rmax; ++r) {
        double sum = 0.0, comp = 0.0;
        for (int64_t xs = 0; xs < Vs; ++xs) {
            int x[ORC_MAXD];
            site_coords(&g, xs, x);
            for (int i = 0; i < td; ++i) {
                int y[ORC_MAXD];
                for (int e = 0; e < D; ++e) y[e] = x[e];
                y[i] = (x[i] + r) % g.n[i];
                neumaier_add(&sum, &comp, l[xs] * l[site_index(&g, y)]);
            }
        }
        out[r - 1] = (sum + comp) / ((double)td * (double)Vs);
    }
    free(l);
    return ORC_OK;
}

/* ====================================================================== */
/* Test gauge transformation (purpose tag 2):                                */
/*   U_mu(x) -> g(x) U_mu(x) g^dag(x+mu), g(x) Haar from counter             */
/*   (s, 0, (2<<8)|(p<<2), 0) with the hot-start formula.                    */
/* ====================================================================== */
int FN(orc_gauge_transform)(int D, const int *dims, REAL *links, uint64_t seed)
{
    geom_t g;
    if (geom_init(&g, D, dims) || !links) return ORC_EARG;
    AREAL *gx = (AREAL *)malloc(sizeof(AREAL) * 4 * (size_t)g.V);
    if (!gx) return ORC_EARG;
    for (int64_t s = 0; s < g.V; ++s) {
        int x[ORC_MAXD];
        uint32_t w[4];
        site_coords(&g, s, x);
        draw_words(seed, (uint32_t)s, 0u, 2u, (uint32_t)site_parity(&g, x), 0u, 0u, w);
        haar_from_words(w, gx + 4 * s);
    }
    for (int64_t s = 0; s < g.V; ++s) {
        int x[ORC_MAXD];
        site_coords(&g, s, x);
        for (int mu = 0; mu < D; ++mu) {
            int xp[ORC_MAXD];
            shifted(&g, x, mu, +1, xp);
            AREAL u[4], gd[4], t[4], r[4];
            load_link(&g, links, x, mu, u);
            qdag(gx + 4 * site_index(&g, xp), gd);
            qmul(gx + 4 * s, u, t);
            qmul(t, gd, r);
            REAL *dst = links + (s * D + mu) * 4;
            for (int c = 0; c < 4; ++c) dst[c] = (REAL)r[c];
        }
    }
    free(gx);
    return ORC_OK;
}
