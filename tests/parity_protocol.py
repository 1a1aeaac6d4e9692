"""The GPU-vs-oracle comparison protocol of DESIGN.md §3 [R13] / [R13b] (test infrastructure).

Tolerances are BASELINE.json north_star's: every link after one sweep |d| <= 1e-12 (fp64) /
1e-5 (fp32); per-sweep mean plaquette 1e-12 / 1e-6. A link outside tolerance must be one of:

  flip        [R13]  a rounding-flipped accept decision: the oracle's smallest accept margin
                     |R3^2 - (1 - delta/2)| (R3 = the trial's fourth uniform) over the link's trials is
                     < FLIP_MARGIN. The new link then differs by O(1). Counted against flip_budget().
  conditioned [R13b] (fp32 only) the draw divides the staple sum v by its norm k (Vbar = v/k, [R7]), so a
                     perturbation dv of the staple reaches the new link as |dv|/k. dv has two sources,
                     both known to the harness: the rounding of the 12 fp32 products of the staple,
                     |dv| <= E_V = 2e-6 (measured: max |d| k = 2.1e-6 over the links with k < 0.5 of 1.26e7, which
                     includes the (1 + delta A) factor below; profiles/r02a.md),
                     and the deviations the 18 input links already carry when earlier sub-steps of the
                     same sweep wrote them, |dv| <= 2 S_in, S_in = the sum of their measured |d| (the 2
                     turns the max-norm of d into a bound on the quaternion norm). The link's tolerance is
                         max(TOL, (E_V + 2 S_in) / k),   k = the oracle's staple norm for that link.
                     A second amplifier sits in the draw itself: the vector part of X lives on a sphere of
                     radius rad = sqrt(delta (2 - delta)) [R7], so a change of delta = 1 - x0 moves it by that
                     times A = max(1, |1 - delta| / rad) - unbounded as x0 -> +-1 (probability ~1e-6 per link).
                     delta = -(ln R + cos^2 ln R'')/alpha changes for two reasons: alpha = beta k carries the
                     relative error dv/k of the staple norm (|d delta| = delta dv/k), and two fp32 evaluations
                     of the logs and the cosine differ by <= E_D (delta + 1/alpha), E_D = 4e-7 (a few ulp of the
                     sum, or the MUFU budget of DESIGN.md 6.2). With the oracle's delta for the link and
                     dv = E_V + 2 S_in:
                         tol = max(TOL, dv/k (1 + delta A) + E_D (delta + 1/alpha) A),
                     north_star's 1e-5 wherever the update is well conditioned (k >= 0.2, clean inputs,
                     rad >~ 0.05), wider only by what the two amplifiers explain. Links that need the wider
                     bound are counted against conditioned_budget().
  downstream         a link whose staple contains a flipped link (or a link downstream of one) that was
                     updated earlier in the same sweep: not comparable and not counted; every OTHER link
                     is checked. (Its inputs deviate by O(1), so it also satisfies the bound above.)

Budgets are max(1, ceil(5 x expectation)) in fp32 and 0 in fp64, expectations from the rates measured on
the GPU (profiles/r02a.md).

Observables are never skipped: the GPU's plaquette and Polyakov loop are compared with the oracle's
evaluated on the configuration the GPU returned (exact to rounding whatever happened to single
links), and with the oracle's own configuration whenever no link was excused.
"""
import math

import numpy as np

import oracle

TOL = {64: 1e-12, 32: 1e-5}
PTOL = {64: 1e-12, 32: 1e-6}
FLIP_MARGIN = {64: 1e-11, 32: 1e-5}
MODE = {64: "f64", 32: "f32"}
E_V = {64: 0.0, 32: 2e-6}  # rounding bound of the fp32 staple sum; fp64 has no conditioning excuse
E_D = {64: 0.0, 32: 4e-7}  # rounding bound of the fp32 delta, in units of (delta + 1/alpha)
# measured on B200 (profiles/r02a.md): 0 flips in 1.26e7 teacher-forced fp32 link updates at 32^4 (beta 2.3
# and 6.0), 20 of which had an accept margin < 1e-6, i.e. ~1.6e-7 flips per link expected at the ~1e-7
# rounding of the accept test. FLIP_RATE is the 95 % upper limit 3 / 1.26e7.
FLIP_RATE = {64: 0.0, 32: 2.4e-7}
# links of a Haar-random lattice that need the widened tolerance: 1 in 1.26e7 in single sub-steps (clean
# inputs); in whole sweeps, where the inputs carry deviations, ~1 per 1e5 (profiles/r02a.md)
COND_RATE = {64: 0.0, 32: 2e-5}

SWEEP = [(mu, p) for mu in range(4) for p in range(2)]  # [R4]


def flip_budget(n_updated, prec):
    lam = FLIP_RATE[prec] * n_updated
    return 0 if lam == 0 else max(1, math.ceil(5 * lam))


def conditioned_budget(n_updated, prec, haar=True):
    """haar: the input has the value structure of a hot start (small staple norms occur); a thermalised or
    near-ordered lattice has k >> 0.2 everywhere and gets the minimum budget"""
    lam = COND_RATE[prec] * n_updated if haar else 0.0
    return 0 if prec == 64 else max(1, math.ceil(5 * lam))


def parity_grid(dims):
    """int8 array [t][z][y][x] of the site parity (x+y+z+t) & 1"""
    nx, ny, nz, nt = dims
    ax = [np.arange(n, dtype=np.int8) & 1 for n in (nt, nz, ny, nx)]
    return ax[0][:, None, None, None] ^ ax[1][None, :, None, None] ^ ax[2][None, None, :, None] ^ ax[3][None, None, None, :]


def _axis(nu):
    return 3 - nu  # direction nu = 0..3 = x,y,z,t lives on axis 3,2,1,0 of [t][z][y][x]


def _staple_inputs(T, mu, combine):
    """T: array [t][z][y][x][4]. For every site, `combine` over the 18 links of the staple of U_mu(x) [R3]:
    U_nu(x+mu), U_mu(x+nu), U_nu(x), U_nu(x+mu-nu), U_mu(x-nu), U_nu(x-nu) for the three nu != mu (geometry only)."""
    out = None
    for nu in range(4):
        if nu == mu:
            continue
        am, an = _axis(mu), _axis(nu)
        Tn, Tm = T[..., nu], T[..., mu]
        up_mu = np.roll(Tn, -1, am)
        for term in (up_mu, np.roll(Tm, -1, an), Tn, np.roll(up_mu, 1, an), np.roll(Tm, 1, an), np.roll(Tn, 1, an)):
            out = term.copy() if out is None else combine(out, term)
    return out


def staple_inputs_any(T, mu):
    """bool flags: is any of the 18 staple inputs flagged?"""
    return _staple_inputs(T, mu, np.logical_or)


def staple_inputs_sum(T, mu):
    """float: sum over the 18 staple inputs"""
    return _staple_inputs(T, mu, np.add)


class Records:
    """What the oracle records per updated link for the protocol: smallest accept margin, staple norm k,
    accepted delta = 1 - x0. Pass **rec.kw to oracle.heatbath_substep / heatbath_sweep."""

    def __init__(self, V):
        self.margin, self.knorm, self.delta = np.ones((V, 4)), np.ones((V, 4)), np.ones((V, 4))

    @property
    def kw(self):
        return dict(margin=self.margin, knorm=self.knorm, delta=self.delta)


def allowed_deviation(delta, k, beta, s_in, prec):
    """The per-link bound of [R13b]: dv/k, where dv = E_V + 2 S_in, reaches the link directly (Vbar = v/k) and
    through alpha = beta k (delta ~ 1/alpha: |d delta| = delta dv/k); the rounding of delta itself is
    E_D (delta + 1/alpha); and every change of delta is amplified by A = max(1, |1 - delta| / rad)."""
    k = np.maximum(k, 1e-30)
    alpha = beta * k
    rad = np.sqrt(np.maximum(delta * (2.0 - delta), 1e-30))
    amp = np.maximum(1.0, np.abs(1.0 - delta) / rad)
    dvk = (E_V[prec] + 2.0 * s_in) / k
    return dvk * (1.0 + delta * amp) + E_D[prec] * (delta + 1.0 / alpha) * amp


class Report:
    def __init__(self, flips, conditioned, downstream, worst):
        self.flips, self.conditioned, self.downstream, self.worst = flips, conditioned, downstream, worst

    @property
    def clean(self):
        return self.flips == 0 and self.conditioned == 0 and self.downstream == 0

    def __repr__(self):
        return f"Report(flips={self.flips}, conditioned={self.conditioned}, downstream={self.downstream}, worst={self.worst:.3e})"


def compare_links(gpu, ora, dims, prec, substeps, rec=None, beta=None, max_flips=None, max_conditioned=None,
                  haar=True, what=""):
    """gpu, ora: [V][4][4] after the sub-steps `substeps` (list of (mu, parity) in execution order, every link
    updated at most once) run on both sides at coupling `beta` from a common configuration; rec: the oracle's
    Records of those sub-steps. Asserts the protocol above; returns a Report."""
    nx, ny, nz, nt = dims
    shape = (nt, nz, ny, nx, 4)
    d = np.abs(gpu.astype(np.float64) - ora.astype(np.float64)).max(-1).reshape(shape)
    bad = d > TOL[prec]
    if not bad.any():
        return Report(0, 0, 0, float(d.max()))
    assert rec is not None and beta is not None, f"{what}: {int(bad.sum())} links differ, max {d.max():.3e}"
    assert len(set(substeps)) == len(substeps)
    mg = np.asarray(rec.margin).reshape(shape)
    kn = np.asarray(rec.knorm).reshape(shape)
    dl = np.asarray(rec.delta).reshape(shape)
    par = parity_grid(dims)
    taint = np.zeros(shape, bool)  # flipped links and what is downstream of them
    dev = np.zeros(shape)          # measured deviation of the links updated so far
    n_flip = n_cond = n_down = n_upd = 0
    for mu, p in substeps:
        sel = par == p
        n_upd += int(sel.sum())
        b, m, k, dd = bad[..., mu] & sel, mg[..., mu], kn[..., mu], d[..., mu]
        down = staple_inputs_any(taint, mu) & sel
        flip = b & ~down & (m < FLIP_MARGIN[prec])
        s_in = staple_inputs_sum(dev, mu)
        allowed = allowed_deviation(dl[..., mu], k, beta, s_in, prec)
        cond = b & ~down & ~flip & (k > 0) & (dd <= allowed) & (E_V[prec] > 0)
        unexplained = b & ~down & ~flip & ~cond
        if unexplained.any():
            i = np.unravel_index(np.argmax(np.where(unexplained, dd, 0)), dd.shape)
            raise AssertionError(f"{what} sub-step mu={mu} p={p}: {int(unexplained.sum())} links differ beyond "
                                 f"tolerance with no excuse; worst |d|={dd[i]:.3e} at (t,z,y,x)={i}, accept margin "
                                 f"{m[i]:.3e}, staple norm k={k[i]:.3e}, deviation of its inputs {s_in[i]:.3e}, "
                                 f"delta={dl[..., mu][i]:.6e}, allowed {allowed[i]:.3e}")
        n_flip += int(flip.sum())
        n_cond += int(cond.sum())
        n_down += int((b & down).sum())
        taint[..., mu] = np.where(sel, down | flip, taint[..., mu])
        dev[..., mu] = np.where(sel, dd, dev[..., mu])
    if max_flips is None:
        max_flips = flip_budget(n_upd, prec)
    if max_conditioned is None:
        max_conditioned = conditioned_budget(n_upd, prec, haar)
    assert n_flip <= max_flips, f"{what}: {n_flip} flipped accept decisions over {n_upd} updates, budget {max_flips}"
    assert n_cond <= max_conditioned, \
        f"{what}: {n_cond} links needed the conditioning bound over {n_upd} updates, budget {max_conditioned}"
    return Report(n_flip, n_cond, n_down, float(d.max()))


def sampled_link_excused(d, margin, k, delta, beta, prec):
    """One sampled link outside tolerance (full-size tests recompute single links with
    oracle.heatbath_link from the pre-update configuration, so the inputs are clean and nothing is
    downstream): 'flip' [R13], 'conditioned' [R13b] or None."""
    if margin < FLIP_MARGIN[prec]:
        return "flip"
    if k > 0 and E_V[prec] > 0 and d <= float(allowed_deviation(np.float64(delta), np.float64(k), beta, 0.0, prec)):
        return "conditioned"
    return None


def check_observables(P_gpu, L_gpu, gpu_links, dims, prec, rep=None, ora_links=None, lscale=10.0, what=""):
    """GPU observables against the oracle evaluated on the configuration the GPU returned - always,
    both within PTOL; and against the oracle's own configuration when the link comparison was clean
    (the Polyakov loop then within lscale x PTOL: every line is a product of N_t links that each
    differ by up to TOL)."""
    mode = MODE[prec]
    if P_gpu is not None:
        assert abs(P_gpu - oracle.mean_plaquette(dims, gpu_links, mode)) < PTOL[prec], f"{what}: plaquette"
    if L_gpu is not None:
        assert abs(L_gpu - oracle.polyakov_loop(dims, gpu_links, mode)) < PTOL[prec], f"{what}: Polyakov"
    if ora_links is not None and (rep is None or rep.clean):
        if P_gpu is not None:
            assert abs(P_gpu - oracle.mean_plaquette(dims, ora_links, mode)) < PTOL[prec], f"{what}: plaquette (oracle chain)"
        if L_gpu is not None:
            assert abs(L_gpu - oracle.polyakov_loop(dims, ora_links, mode)) < lscale * PTOL[prec], f"{what}: Polyakov (oracle chain)"
