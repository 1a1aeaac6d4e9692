"""The GPU-vs-oracle comparison protocol of DESIGN.md §3 [R13] / [R13b] (test infrastructure).

Tolerances are BASELINE.json north_star's: every link after one sweep |d| <= 1e-12 (fp64) /
1e-5 (fp32); per-sweep mean plaquette 1e-12 / 1e-6. A link outside tolerance must have one of two
PRIMARY excuses, both read off values the ORACLE computed for that link, or lie DOWNSTREAM of a link
that has one:

  flip     [R13]  a rounding-flipped accept decision: the oracle's smallest accept margin
                  |R'''^2 - (1 - delta/2)| over the link's trials is < FLIP_MARGIN. The new link then
                  differs by O(1).
  small k  [R13b] an ill-conditioned update (fp32 only): the draw divides the staple sum v by its norm k,
                  so the rounding of v (6 terms x 2 products in fp32, |dv| <~ E_V = 1e-6) reaches the
                  new link as |dv|/k. For k >= K_SMALL = E_V / 1e-5 = 0.1 that stays inside 1e-5; below
                  it the link is excused iff |d| <= E_V / k, i.e. iff the deviation is what 1/k explains.
  downstream      within one sweep a later sub-step reads the links earlier sub-steps wrote: a link
                  whose staple contains an excused (or downstream) link that was updated since the
                  common input is itself not comparable. The set is the closure over the sub-steps
                  in execution order; its members are not counted but every OTHER link is checked.

Primary excuses are COUNTED against budgets derived from the measured rates (profiles/r02a.md):
flips at FLIP_RATE per updated link, small-k links at P(k < K_SMALL) = K_SMALL^4 / 18 per link of a
Haar-random lattice (v is a 6-step random walk in R^4, variance 3/2 per component); the budget is
max(1, ceil(5 x expectation)) in fp32 and 0 in fp64.

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
E_V = {64: 0.0, 32: 1e-6}                 # rounding bound of the fp32 staple sum; fp64 has no small-k excuse
K_SMALL = {64: 0.0, 32: 0.1}              # = E_V / TOL
# measured on B200, teacher-forced sub-steps over 1.7e7 (beta 2.3) and 1.7e7 (beta 6.0) links of 32^4:
# see profiles/r02a.md; the larger of the two rates
FLIP_RATE = {64: 0.0, 32: 4e-7}
P_SMALL_K_HAAR = {64: 0.0, 32: 0.1 ** 4 / 18.0}

SWEEP = [(mu, p) for mu in range(4) for p in range(2)]  # [R4]


def flip_budget(n_updated, prec):
    lam = FLIP_RATE[prec] * n_updated
    return 0 if lam == 0 else max(1, math.ceil(5 * lam))


def small_k_budget(n_updated, prec, haar=True):
    lam = P_SMALL_K_HAAR[prec] * n_updated if haar else 0.0
    return 0 if prec == 64 else max(1, math.ceil(5 * lam))


def parity_grid(dims):
    """int8 array [t][z][y][x] of the site parity (x+y+z+t) & 1"""
    nx, ny, nz, nt = dims
    ax = [np.arange(n, dtype=np.int8) & 1 for n in (nt, nz, ny, nx)]
    return ax[0][:, None, None, None] ^ ax[1][None, :, None, None] ^ ax[2][None, None, :, None] ^ ax[3][None, None, None, :]


def _axis(nu):
    return 3 - nu  # direction nu = 0..3 = x,y,z,t lives on axis 3,2,1,0 of [t][z][y][x]


def staple_inputs_any(T, mu):
    """T: bool [t][z][y][x][4]. For every site: does any of the 18 links of the staple of U_mu(x) have
    its flag set? Geometry of [R3] only: U_nu(x+mu), U_mu(x+nu), U_nu(x), U_nu(x+mu-nu), U_mu(x-nu), U_nu(x-nu)."""
    out = np.zeros(T.shape[:4], bool)
    for nu in range(4):
        if nu == mu:
            continue
        am, an = _axis(mu), _axis(nu)
        Tn, Tm = T[..., nu], T[..., mu]
        up_mu = np.roll(Tn, -1, am)
        out |= up_mu | np.roll(Tm, -1, an) | Tn | np.roll(up_mu, 1, an) | np.roll(Tm, 1, an) | np.roll(Tn, 1, an)
    return out


class Report:
    def __init__(self, flips, small_k, downstream, worst):
        self.flips, self.small_k, self.downstream, self.worst = flips, small_k, downstream, worst

    @property
    def clean(self):
        return self.flips == 0 and self.small_k == 0 and self.downstream == 0


def compare_links(gpu, ora, dims, prec, substeps, margin=None, knorm=None, max_flips=None, max_small_k=None,
                  haar=True, what=""):
    """gpu, ora: [V][4][4] after the sub-steps `substeps` (list of (mu, parity) in execution order) run
    on both sides from a common configuration; margin, knorm: the oracle's [V][4] records of those
    sub-steps. Asserts the protocol above; returns a Report."""
    nx, ny, nz, nt = dims
    shape = (nt, nz, ny, nx, 4)
    d = np.abs(gpu.astype(np.float64) - ora.astype(np.float64)).max(-1).reshape(shape)
    bad = d > TOL[prec]
    if not bad.any():
        return Report(0, 0, 0, float(d.max()))
    assert margin is not None and knorm is not None, f"{what}: {int(bad.sum())} links differ, max {d.max():.3e}"
    mg = np.asarray(margin).reshape(shape)
    kn = np.asarray(knorm).reshape(shape)
    par = parity_grid(dims)
    taint = np.zeros(shape, bool)
    n_flip = n_small = n_down = n_upd = 0
    for mu, p in substeps:
        sel = par == p
        n_upd += int(sel.sum())
        b, m, k, dd = bad[..., mu] & sel, mg[..., mu], kn[..., mu], d[..., mu]
        down = staple_inputs_any(taint, mu) & sel
        flip = b & ~down & (m < FLIP_MARGIN[prec])
        small = b & ~down & ~flip & (k < K_SMALL[prec]) & (k > 0) & (dd * k <= E_V[prec])
        unexplained = b & ~down & ~flip & ~small
        if unexplained.any():
            i = np.unravel_index(np.argmax(np.where(unexplained, dd, 0)), dd.shape)
            raise AssertionError(f"{what} sub-step mu={mu} p={p}: {int(unexplained.sum())} links differ beyond "
                                 f"tolerance with no excuse; worst |d|={dd[i]:.3e} at (t,z,y,x)={i}, "
                                 f"accept margin {m[i]:.3e}, staple norm k={k[i]:.3e}")
        n_flip += int(flip.sum())
        n_small += int(small.sum())
        n_down += int((b & down).sum())
        taint[..., mu] = np.where(sel, down | flip | small, taint[..., mu])
    if max_flips is None:
        max_flips = flip_budget(n_upd, prec)
    if max_small_k is None:
        max_small_k = small_k_budget(n_upd, prec, haar)
    assert n_flip <= max_flips, f"{what}: {n_flip} flipped accept decisions over {n_upd} updates, budget {max_flips}"
    assert n_small <= max_small_k, f"{what}: {n_small} small-k excuses over {n_upd} updates, budget {max_small_k}"
    return Report(n_flip, n_small, n_down, float(d.max()))


def sampled_link_excused(d, margin, k, prec):
    """One sampled link outside tolerance (full-size tests recompute single links with
    oracle.heatbath_link from the pre-update configuration, so nothing is downstream):
    'flip' [R13], 'small_k' [R13b] or None."""
    if margin < FLIP_MARGIN[prec]:
        return "flip"
    if 0 < k < K_SMALL[prec] and d * k <= E_V[prec]:
        return "small_k"
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
