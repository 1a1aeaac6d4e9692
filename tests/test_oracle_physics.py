"""Pins of the oracle's update and measurements against closed forms,
invariants and brute force (SURVEY.md §8(c) pin table).
None of the expected values comes from the oracle or from the CUDA path."""
import numpy as np
import pytest
from scipy import integrate, special, stats

import oracle
from paper_1104_5432_b200 import workloads

RATIO = lambda a: special.ive(2, a) / special.ive(1, a)  # I2/I1, overflow-safe


# ---------------------------------------------------------------- staple
@pytest.mark.parametrize("dims", [[4, 4], [4, 6, 4], [4, 4, 6, 4], [2, 2, 2, 2]])
def test_staple_equals_sum_of_plaquettes_through_link(dims):
    """sum over the 2(D-1) plaquettes containing U_mu(x) of 1/2 Tr U_P == 1/2 Tr(U_mu(x) v)."""
    D = len(dims)
    L = workloads.random_links(dims, 5)
    V = oracle.volume(dims)
    strides = np.cumprod([1] + list(dims[:-1]))
    rng = np.random.default_rng(1)
    for s in rng.integers(0, V, size=12):
        s = int(s)
        x = [(s // int(strides[d])) % dims[d] for d in range(D)]
        for mu in range(D):
            v = oracle.staple(dims, L, s, mu)
            lhs = oracle.qmul(L[s, mu], v)[0]
            rhs = 0.0
            for nu in range(D):
                if nu == mu:
                    continue
                rhs += oracle.plaquette_at(dims, L, s, mu, nu)  # forward plaquette at x
                xm = list(x)
                xm[nu] = (xm[nu] - 1) % dims[nu]
                sm = int(sum(xm[d] * int(strides[d]) for d in range(D)))
                rhs += oracle.plaquette_at(dims, L, sm, mu, nu)  # the plaquette at x - nu
            assert abs(lhs - rhs) < 1e-13


def test_staple_cold_lattice():
    for dims in ([4, 4], [4, 4, 4], [4, 4, 4, 4]):
        D = len(dims)
        L = oracle.init(dims, "cold", 0)
        for mu in range(D):
            assert np.allclose(oracle.staple(dims, L, 3, mu), [2 * (D - 1), 0, 0, 0], atol=0)


# ---------------------------------------------------------------- KP law
@pytest.mark.parametrize("alpha,mean_x0,acc", [(2.0, 0.433127, 0.763110), (10.0, 0.854185, 0.961207),
                                               (32.0, 0.953503, 0.988164)])
def test_kp_draw_matches_closed_forms(alpha, mean_x0, acc):
    """<x0> = I2(a)/I1(a); acceptance = sqrt(2 pi a) e^-a I1(a); full CDF of
    sqrt(1-x^2) e^{a x} by quadrature (KS). Printed values: SURVEY.md §8(c) pin table."""
    assert abs(RATIO(alpha) - mean_x0) < 2e-6
    assert abs(np.sqrt(2 * np.pi * alpha) * special.ive(1, alpha) - acc) < 2e-6
    n = 40000
    x0 = np.empty(n)
    trials = np.empty(n, dtype=np.int64)
    for i in range(n):
        x0[i], trials[i] = oracle.kp_x0(alpha, 1234, i, 0)
    dens = lambda x: np.sqrt(max(0.0, 1 - x * x)) * np.exp(alpha * (x - 1))
    Z = integrate.quad(dens, -1, 1, epsabs=1e-13, points=[0.5, 0.9, 0.99])[0]
    var = integrate.quad(lambda x: x * x * dens(x), -1, 1, epsabs=1e-13)[0] / Z - RATIO(alpha) ** 2
    assert abs(x0.mean() - RATIO(alpha)) < 4.5 * np.sqrt(var / n)
    p_acc = 1.0 / trials.mean()
    assert abs(p_acc - acc) < 4.5 * np.sqrt(acc * (1 - acc) / n) / acc
    grid = np.linspace(-1, 1, 4001)
    pdf = np.sqrt(np.clip(1 - grid**2, 0, None)) * np.exp(alpha * (grid - 1))
    cdfg = integrate.cumulative_trapezoid(pdf, grid, initial=0)
    cdfg /= cdfg[-1]
    assert stats.kstest(x0, lambda x: np.interp(x, grid, cdfg)).pvalue > 1e-4
    assert (x0 >= -1).all() and (x0 < 1).all()


def test_kp_fp32_mode_same_law():
    alpha, n = 10.0, 20000
    x = np.array([oracle.kp_x0(alpha, 99, i, 3, "f32")[0] for i in range(n)])
    assert abs(x.mean() - RATIO(alpha)) < 4.5 * 0.12 / np.sqrt(n)


# ------------------------------------------- single-link heat bath on 2^4
def test_single_link_heatbath_matches_brute_force_boltzmann():
    """Freeze all other links of a 2^4 hot lattice, update one link N times with
    sweep_idx = 0..N-1 (north_star pin). E[U'] = (I2(bk)/I1(bk)) Vbar^dagger, and
    each component's histogram equals brute-force integration of
    exp(beta 1/2 Tr(U v)) over S^3 on a hyperspherical grid."""
    dims = [2, 2, 2, 2]
    beta = 2.3
    L = oracle.init(dims, "hot", 17)
    s, mu = 5, 2
    v = oracle.staple(dims, L, s, mu)
    k = np.linalg.norm(v)
    n = 30000
    U = np.array([oracle.heatbath_link(dims, L, beta, 17, i, s, mu)[0] for i in range(n)])
    assert np.abs((U**2).sum(1) - 1).max() < 9e-16
    want = RATIO(beta * k) * v * [1, -1, -1, -1] / k
    # per-component sd <= 1/2
    assert np.abs(U.mean(0) - want).max() < 4.5 * 0.5 / np.sqrt(n)

    # Brute force, per component c: hyperspherical coordinates with the polar axis
    # along c, u_c = t, the other three components = sqrt(1-t^2) * n, n on S^2;
    # dHaar ~ sqrt(1-t^2) dt dOmega(n). Gauss-Legendre in t inside every histogram
    # bin (nodes never straddle a bin edge), midpoint rule on the sphere.
    nth, nph, ngl = 96, 192, 16
    th = (np.arange(nth) + 0.5) * np.pi / nth
    ph = (np.arange(nph) + 0.5) * 2 * np.pi / nph
    T, F = np.meshgrid(th, ph, indexing="ij")
    nvec = np.stack([np.sin(T) * np.cos(F), np.sin(T) * np.sin(F), np.cos(T)])  # [3][nth][nph]
    dom = np.sin(T)
    sgn = np.array([1.0, -1.0, -1.0, -1.0])  # 1/2 Tr(U v) = u0 v0 - u.v  (scalar part of the product)
    glx, glw = np.polynomial.legendre.leggauss(ngl)
    edges = np.linspace(-1, 1, 17)
    for c in range(4):
        others = [i for i in range(4) if i != c]
        lin = sum(sgn[o] * v[o] * nvec[j] for j, o in enumerate(others))  # coefficient of sqrt(1-t^2)
        prob = np.zeros(len(edges) - 1)
        for j in range(len(edges) - 1):
            lo, hi = edges[j], edges[j + 1]
            t = 0.5 * (hi + lo) + 0.5 * (hi - lo) * glx
            for tt, ww in zip(t, glw * 0.5 * (hi - lo)):
                r = np.sqrt(1 - tt * tt)
                prob[j] += ww * r * (dom * np.exp(beta * (sgn[c] * v[c] * tt + r * lin - k))).sum()
        prob /= prob.sum()
        expect = prob * n
        got = np.histogram(U[:, c], bins=edges)[0]
        m = expect > 8
        chi2 = ((got[m] - expect[m]) ** 2 / expect[m]).sum()
        assert chi2 < stats.chi2.ppf(1 - 1e-4, m.sum()), (c, chi2)
    # the update must not depend on the old value of the link
    L2 = L.copy()
    L2[s, mu] = [0, 1, 0, 0]
    assert (oracle.heatbath_link(dims, L2, beta, 17, 0, s, mu)[0] == U[0]).all()


# ---------------------------------------------------------------- invariants
@pytest.mark.parametrize("mode,tol", [("f64", 9e-16), ("f32", 2.4e-7), ("f32x", 1.2e-7)])
def test_unit_norm_after_every_update(mode, tol):
    dims = [4, 4, 4, 6]
    L = oracle.init(dims, "hot", 3, mode)
    for i in range(3):
        oracle.heatbath_sweep(dims, L, 2.3, 3, i, mode)
        n2 = (L.astype(np.float64) ** 2).sum(-1)
        assert np.abs(n2 - 1).max() < tol


def test_visiting_order_inside_substep_is_irrelevant():
    dims = [4, 4, 4, 4]
    V = oracle.volume(dims)
    A = oracle.init(dims, "hot", 8)
    B = A.copy()
    rng = np.random.default_rng(0)
    for mu in range(4):
        for p in range(2):
            oracle.heatbath_substep(dims, A, 2.3, 8, 0, mu, p)
            oracle.heatbath_substep(dims, B, 2.3, 8, 0, mu, p, order=rng.permutation(V))
    assert (A == B).all()
    # and the sweep wrapper is exactly the 8 sub-steps in the order mu-major, parity-minor
    Cc = oracle.init(dims, "hot", 8)
    oracle.heatbath_sweep(dims, Cc, 2.3, 8, 0)
    assert (Cc == A).all()


def test_substep_touches_only_its_links():
    dims = [4, 4, 4, 4]
    A = oracle.init(dims, "hot", 8)
    B = A.copy()
    oracle.heatbath_substep(dims, B, 2.3, 8, 0, 1, 1)
    s = np.arange(oracle.volume(dims))
    par = (s % 4 + s // 4 % 4 + s // 16 % 4 + s // 64) % 2
    changed = (A != B).any(-1)
    assert changed[par == 1, 1].all()
    changed[par == 1, 1] = False
    assert not changed.any()


def test_cold_plaquette_and_polyakov_are_one():
    for dims in ([4, 4], [4, 4, 4], [4, 6, 4, 8]):
        L = oracle.init(dims, "cold", 0)
        assert oracle.mean_plaquette(dims, L) == 1.0
        assert oracle.polyakov_loop(dims, L) == 1.0


@pytest.mark.parametrize("dims", [[6, 4], [4, 4, 6], [4, 6, 4, 4]])
def test_gauge_invariance_of_plaquette_and_polyakov(dims):
    L = oracle.init(dims, "hot", 21)
    for i in range(2):
        oracle.heatbath_sweep(dims, L, 2.0, 21, i)
    P, (Lp, field) = oracle.mean_plaquette(dims, L), oracle.polyakov_loop(dims, L, return_field=True)
    G = L.copy()
    oracle.gauge_transform(dims, G, 77)
    assert np.abs(G - L).max() > 0.1  # it did something
    assert abs(oracle.mean_plaquette(dims, G) - P) < 1e-14
    Lp2, field2 = oracle.polyakov_loop(dims, G, return_field=True)
    assert abs(Lp2 - Lp) < 1e-14 and np.abs(field2 - field).max() < 1e-14


def test_polyakov_centre_flip_and_definition():
    """Multiplying every U_t on ONE time slice by -1 flips every Polyakov line and
    leaves every plaquette unchanged: pins that the product runs over all N_t
    slices of the time direction (D-1) exactly once."""
    dims = [4, 4, 4, 6]
    L = oracle.init(dims, "hot", 4)
    P, (Lp, field) = oracle.mean_plaquette(dims, L), oracle.polyakov_loop(dims, L, return_field=True)
    Vs = 4 * 4 * 4
    F = L.copy().reshape(6, Vs, 4, 4)
    F[2, :, 3, :] *= -1
    F = F.reshape(L.shape)
    Lp2, field2 = oracle.polyakov_loop(dims, F, return_field=True)
    assert np.abs(field2 + field).max() < 1e-15 and abs(Lp2 + Lp) < 1e-15
    assert abs(oracle.mean_plaquette(dims, F) - P) < 1e-15
    # direct definition with 2x2 matrices at a few spatial sites
    sig = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]]),
           np.array([[1, 0], [0, -1]], dtype=complex)]
    mat = lambda a: a[0] * np.eye(2) + 1j * sum(a[i + 1] * sig[i] for i in range(3))
    Lr = L.reshape(6, Vs, 4, 4)
    for xs in (0, 7, 63):
        M = np.eye(2, dtype=complex)
        for t in range(6):
            M = M @ mat(Lr[t, xs, 3])
        assert abs(0.5 * np.trace(M).real - field[xs]) < 1e-14
    assert abs(field.mean() - Lp) < 1e-15


def test_plaquette_direct_definition_with_matrices():
    dims = [4, 4, 4, 4]
    L = workloads.random_links(dims, 2)
    sig = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]]),
           np.array([[1, 0], [0, -1]], dtype=complex)]
    M = L[..., 0, None, None] * np.eye(2) + 1j * sum(L[..., i + 1, None, None] * sig[i] for i in range(3))
    M = M.reshape(4, 4, 4, 4, 4, 2, 2)  # [t][z][y][x][mu]
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            Umu, Unu = M[..., mu, :, :], M[..., nu, :, :]
            Unu_xpmu = np.roll(Unu, -1, axis=3 - mu)
            Umu_xpnu = np.roll(Umu, -1, axis=3 - nu)
            pl = Umu @ Unu_xpmu @ np.conj(np.swapaxes(Umu_xpnu, -1, -2)) @ np.conj(np.swapaxes(Unu, -1, -2))
            tot += 0.5 * np.trace(pl, axis1=-2, axis2=-1).real.sum()
    assert abs(tot / (6 * 256) - oracle.mean_plaquette(dims, L)) < 1e-14


# ---------------------------------------------------------------- whole chain
@pytest.mark.parametrize("beta,exact", [(1.0, 0.240194), (2.0, 0.433127), (6.0, 0.762726)])
def test_d2_equilibrium_plaquette_is_I2_over_I1(beta, exact):
    """North_star pin: in D=2 the equilibrium <1/2 Tr P> is exactly I2(beta)/I1(beta)
    (torus correction < 1e-20 at 16^2). Printed values: SURVEY.md §8(c)."""
    assert abs(RATIO(beta) - exact) < 2e-6
    dims = [16, 16]
    L = oracle.init(dims, "hot", 31)
    nth, nms = 50, 1500
    vals = []
    for i in range(nth + nms):
        oracle.heatbath_sweep(dims, L, beta, 31, i)
        if i >= nth:
            vals.append(oracle.mean_plaquette(dims, L))
    vals = np.array(vals)
    nb = 30  # binned error (autocorrelation)
    bins = vals[: len(vals) // nb * nb].reshape(nb, -1).mean(1)
    err = bins.std(ddof=1) / np.sqrt(nb)
    assert abs(vals.mean() - RATIO(beta)) < 4.5 * err + 1e-9
    assert err < 2e-3


def test_d4_schwinger_dyson_identity():
    """In equilibrium 6<P> = <k I2(beta k)/I1(beta k)> (link-integration identity):
    two estimators on the same ensemble that must agree within errors."""
    dims = [4, 4, 4, 4]
    beta = 2.3
    L = oracle.init(dims, "hot", 41)
    a, b = [], []
    for i in range(260):
        oracle.heatbath_sweep(dims, L, beta, 41, i)
        if i >= 40:
            k = oracle.staple_norms(dims, L)
            a.append(oracle.mean_plaquette(dims, L))
            b.append((k * RATIO(beta * k)).mean() / 6.0)
    d = np.array(a) - np.array(b)
    nb = 20
    bins = d[: len(d) // nb * nb].reshape(nb, -1).mean(1)
    err = bins.std(ddof=1) / np.sqrt(nb)
    assert abs(d.mean()) < 4.5 * err
    assert 0.55 < np.mean(a) < 0.66  # sanity band at beta=2.3 on a small volume


def test_d4_strong_coupling_limit():
    """beta = 0.5: <P> = u + O(u^5), u = I2/I1 = 0.123718 (correction ~1e-4)."""
    beta = 0.5
    assert abs(RATIO(beta) - 0.123718) < 2e-6
    dims = [4, 4, 4, 4]
    L = oracle.init(dims, "hot", 51)
    vals = []
    for i in range(330):
        oracle.heatbath_sweep(dims, L, beta, 51, i)
        if i >= 30:
            vals.append(oracle.mean_plaquette(dims, L))
    vals = np.array(vals)
    bins = vals.reshape(20, -1).mean(1)
    err = bins.std(ddof=1) / np.sqrt(20)
    assert abs(vals.mean() - RATIO(beta)) < 4.5 * err + 3e-4


# ---------------------------------------------------------------- fp32 modes
def test_fp32_modes_track_fp64_on_one_teacher_forced_sweep():
    """fp32 arithmetic differs from fp64 only by rounding: after one sweep from the
    same (fp32-representable) start, every link whose accept decisions did not sit
    on the threshold agrees to ~1e-5 (north_star tolerance) between f32 and f32x."""
    dims = [4, 4, 4, 4]
    A = oracle.init(dims, "hot", 61, "f32")
    B = A.copy()
    V = oracle.volume(dims)
    mg = np.ones((V, 4))
    oracle.heatbath_sweep(dims, A, 2.3, 61, 0, "f32")
    oracle.heatbath_sweep(dims, B, 2.3, 61, 0, "f32x", margin=mg)
    diff = np.abs(A.astype(np.float64) - B.astype(np.float64)).max(-1)
    bad = diff > 1e-5
    # within one sweep later sub-steps read earlier results, so a flipped link could
    # spread; with 1024 links the expected number of flips is ~1e-4: demand none.
    assert not bad.any()
    assert abs(oracle.mean_plaquette(dims, A, "f32") - oracle.mean_plaquette(dims, B, "f32x")) < 1e-6


def test_degenerate_staple_gives_haar_element_independent_of_beta():
    """[R8]: k = 0 exactly on a hand-built lattice -> the new link is the Haar element of the
    n = 0 words: unit norm, no KP trial, the same for every beta, different per sweep_idx."""
    from paper_1104_5432_b200 import workloads
    dims, s, mu = [4, 4, 4, 4], 37, 1
    L = workloads.degenerate_staple_links(dims, s, mu)
    assert np.abs(oracle.staple(dims, L, s, mu)).max() == 0.0
    u1, tr1, _ = oracle.heatbath_link(dims, L, 2.3, 5, 0, s, mu)
    u2, tr2, _ = oracle.heatbath_link(dims, L, 6.0, 5, 0, s, mu)
    u3, _, _ = oracle.heatbath_link(dims, L, 6.0, 5, 1, s, mu)
    assert tr1 == 0 and tr2 == 0
    assert (u1 == u2).all() and not (u1 == u3).all()
    assert abs(np.linalg.norm(u1) - 1) < 1e-15
    # a neighbouring link with a non-zero staple is updated normally
    u4, tr4, _ = oracle.heatbath_link(dims, L, 2.3, 5, 0, s + 1, mu)
    assert tr4 >= 1


# ---------------------------------------------------------------- Creutz draw [R15]
@pytest.fixture
def draw_mode():
    """Switches the oracle's draw for one test and restores the default (KP) afterwards."""
    def use(method, mode="f64"):
        oracle.set_draw(method, mode)
    yield use
    for m in ("f64", "f32", "f32x"):
        oracle.set_draw("kp", m)


@pytest.mark.parametrize("alpha,mean_x0,acc", [(0.5, 0.123718, 0.777400), (1.0, 0.240194, 0.755402),
                                               (2.0, 0.433127, 0.688906)])
def test_creutz_draw_matches_closed_forms(alpha, mean_x0, acc):
    """Same target law as KP: <x0> = I2/I1 (0.123718 and 0.240194 are SURVEY.md §8(c)'s strong-coupling
    and D=2 values of that ratio); acceptance = (pi/2) I1(a)/sinh(a) (0.755 at
    a = 1); CDF of sqrt(1-x^2) e^{a x} by quadrature (KS)."""
    assert abs(RATIO(alpha) - mean_x0) < 2e-6
    assert abs(np.pi / 2 * special.iv(1, alpha) / np.sinh(alpha) - acc) < 2e-6
    n = 40000
    x0 = np.empty(n)
    trials = np.empty(n, dtype=np.int64)
    for i in range(n):
        x0[i], trials[i] = oracle.creutz_x0(alpha, 4321, i, 0)
    dens = lambda x: np.sqrt(max(0.0, 1 - x * x)) * np.exp(alpha * (x - 1))
    Z = integrate.quad(dens, -1, 1, epsabs=1e-13)[0]
    var = integrate.quad(lambda x: x * x * dens(x), -1, 1, epsabs=1e-13)[0] / Z - RATIO(alpha) ** 2
    assert abs(x0.mean() - RATIO(alpha)) < 4.5 * np.sqrt(var / n)
    p_acc = 1.0 / trials.mean()
    assert abs(p_acc - acc) < 4.5 * np.sqrt(acc * (1 - acc) / n) / acc
    grid = np.linspace(-1, 1, 4001)
    pdf = np.sqrt(np.clip(1 - grid**2, 0, None)) * np.exp(alpha * (grid - 1))
    cdfg = integrate.cumulative_trapezoid(pdf, grid, initial=0)
    cdfg /= cdfg[-1]
    assert stats.kstest(x0, lambda x: np.interp(x, grid, cdfg)).pvalue > 1e-4
    assert (x0 >= -1).all() and (x0 < 1).all()


def test_acceptance_crossover_is_alpha_c():
    """[R15]: ALPHA_C is where KP's acceptance sqrt(2 pi a) e^-a I1(a) equals Creutz's (pi/2) I1(a)/sinh(a)."""
    a = oracle.ALPHA_C
    kp = np.sqrt(2 * np.pi * a) * special.ive(1, a)
    cr = np.pi / 2 * special.iv(1, a) / np.sinh(a)
    assert abs(kp - cr) < 2e-5
    assert np.sqrt(2 * np.pi * 1.0) * special.ive(1, 1.0) < np.pi / 2 * special.iv(1, 1.0) / np.sinh(1.0)
    assert np.sqrt(2 * np.pi * 3.0) * special.ive(1, 3.0) > np.pi / 2 * special.iv(1, 3.0) / np.sinh(3.0)


def test_auto_draw_selects_per_link_and_samples_the_boltzmann_weight(draw_mode):
    """'auto' = Creutz iff alpha < ALPHA_C, per link. On a 2^4 hot lattice at beta = 0.5 some links
    have alpha below and some above: the new link equals the always-Creutz result on the former
    and the KP result on the latter; and the single-link mean is (I2/I1)(beta k) Vbar^dagger."""
    dims, beta, seed = [2, 2, 2, 2], 0.5, 23
    L = oracle.init(dims, "hot", seed)
    alpha = beta * oracle.staple_norms(dims, L)
    assert (alpha < oracle.ALPHA_C).any() and (alpha > oracle.ALPHA_C).any()
    res = {}
    for method in ("kp", "creutz", "auto"):
        draw_mode(method)
        res[method] = np.array([[oracle.heatbath_link(dims, L, beta, seed, 0, s, mu)[0] for mu in range(4)]
                                for s in range(16)])
    low = alpha < oracle.ALPHA_C
    assert (res["auto"][low] == res["creutz"][low]).all()
    assert (res["auto"][~low] == res["kp"][~low]).all()
    assert not (res["kp"][low] == res["creutz"][low]).all()
    # law of the updated link under 'auto' at a link with small alpha
    s, mu = np.argwhere(low)[0]
    v = oracle.staple(dims, L, int(s), int(mu))
    k = np.linalg.norm(v)
    n = 30000
    U = np.array([oracle.heatbath_link(dims, L, beta, seed, i, int(s), int(mu))[0] for i in range(n)])
    assert np.abs((U**2).sum(1) - 1).max() < 9e-16
    want = RATIO(beta * k) * v * [1, -1, -1, -1] / k
    assert np.abs(U.mean(0) - want).max() < 4.5 * 0.5 / np.sqrt(n)


def test_d2_equilibrium_plaquette_with_creutz_draw(draw_mode):
    """Whole chain with the always-Creutz draw, D = 2: <1/2 Tr P> = I2(beta)/I1(beta) = 0.240194 at beta = 1."""
    draw_mode("creutz")
    dims, beta = [8, 8], 1.0
    L = oracle.init(dims, "hot", 3)
    vals = []
    for sw in range(1200):
        oracle.heatbath_sweep(dims, L, beta, 3, sw)
        if sw >= 100:
            vals.append(oracle.mean_plaquette(dims, L))
    vals = np.array(vals)
    b = vals[: len(vals) // 20 * 20].reshape(20, -1).mean(1)
    assert abs(vals.mean() - 0.240194) < 4.5 * b.std(ddof=1) / np.sqrt(20)


# ---------------------------------------------------------------- staple norm k returned beside the margin ([R13b])
@pytest.mark.parametrize("mode", ["f64", "f32"])
def test_returned_staple_norm_is_the_norm_of_the_pinned_staple(mode):
    """heatbath_substep(knorm=...) hands out the k of every link it updates. It must be the
    quaternion norm of the staple sum of the PRE-update lattice - orc_staple, which the
    plaquette-sum identity above pins - and only the updated entries may be written.
    orc_staple_norms (all links at once) must agree with the same values."""
    dims = [4, 6, 4, 2]
    L = workloads.random_links(dims, 17, oracle.dtype(mode))
    V = oracle.volume(dims)
    for mu, p in ((0, 1), (3, 0)):
        before = L.copy()
        all_k = oracle.staple_norms(dims, before, mode)
        kn = np.full((V, 4), -7.0)
        oracle.heatbath_substep(dims, L, 2.3, 5, 0, mu, p, mode, knorm=kn)
        s = np.arange(V)
        par = (s % 4 + s // 4 % 6 + s // 24 % 4 + s // 96) % 2
        written = kn != -7.0
        assert written[par == p, mu].all() and written.sum() == (par == p).sum()
        tol = 1e-14 if mode == "f64" else 1e-6
        for site in np.flatnonzero(par == p)[::5]:
            v = oracle.staple(dims, before, int(site), mu, mode).astype(np.float64)
            assert abs(kn[site, mu] - np.linalg.norm(v)) < tol
            assert abs(all_k[site, mu] - np.linalg.norm(v)) < tol
        u, tr, mg, k1 = oracle.heatbath_link(dims, before, 2.3, 5, 0, int(site), mu, mode, return_k=True)
        assert k1 == kn[site, mu]
    # the hand-built k = 0 link [R8] reports k = 0
    Z = workloads.degenerate_staple_links((4, 4, 4, 4), 37, 1, oracle.dtype(mode))
    assert oracle.heatbath_link((4, 4, 4, 4), Z, 2.3, 5, 0, 37, 1, mode, return_k=True)[3] == 0.0


# ---------------------------------------------------------------- Polyakov-loop correlator (eq. 3)
def _with_time_link(dims, sites_and_quats):
    """cold lattice whose time link at (xs, t = 1) is the given unit quaternion: l(xs) = its a0"""
    V = oracle.volume(dims)
    L = np.zeros((V, 4, 4))
    L[..., 0] = 1.0
    Vs = V // dims[3]
    for xs, q in sites_and_quats:
        L[Vs * 1 + xs, 3] = np.asarray(q) / np.linalg.norm(q)
    return L


def test_correlator_cold_and_constant_field():
    dims = [6, 4, 8, 4]
    L = oracle.init(dims, "cold", 0)
    assert (oracle.polyakov_correlator(dims, L, 2) == 1.0).all()
    # every time link on slice 2 equal to one quaternion q: l(x) = q0 everywhere, C(r) = q0^2
    q = np.array([0.3, -0.5, 0.1, 0.8])
    q /= np.linalg.norm(q)
    Lr = L.reshape(4, -1, 4, 4)
    Lr[2, :, 3] = q
    assert np.abs(oracle.polyakov_correlator(dims, L, 2) - q[0] ** 2).max() < 1e-15


def test_correlator_counts_the_pairs_of_two_nontrivial_lines():
    """Cold lattice with two Polyakov lines of value a and b a distance d = 2 apart along y. Of the
    3 Vs ordered pairs (x, x + r e_i), 6 contain the first line and 6 the second; for r = d one pair
    contains both. So C(r) = (3Vs - 12 + 6a + 6b)/(3Vs) for r != d and (3Vs - 11 + 5a + 5b + ab)/(3Vs)
    for r = d: pins the normalisation, the axis loop, the direction of the shift and the r index."""
    dims = [8, 8, 6, 4]
    nx, ny, nz, _ = dims
    Vs = nx * ny * nz
    x0 = 3 + nx * (1 + ny * 2)
    x1 = 3 + nx * (3 + ny * 2)
    qa, qb = [0.6, 0.8, 0.0, 0.0], [-0.28, 0.0, 0.96, 0.0]
    L = _with_time_link(dims, [(x0, qa), (x1, qb)])
    a, b = 0.6, -0.28
    C = oracle.polyakov_correlator(dims, L, 3)
    plain = (3 * Vs - 12 + 6 * a + 6 * b) / (3 * Vs)
    both = (3 * Vs - 11 + 5 * a + 5 * b + a * b) / (3 * Vs)
    assert np.abs(C - [plain, both, plain]).max() < 1e-15
    # the same two lines 2 apart along z, on a lattice with Nz = 6: r = 2 only (r = 3 = Nz/2 does not see it)
    x1z = 3 + nx * (1 + ny * 4)
    C = oracle.polyakov_correlator(dims, _with_time_link(dims, [(x0, qa), (x1z, qb)]), 3)
    assert np.abs(C - [plain, both, plain]).max() < 1e-15
    # wrapped the other way: lines 6 apart along x on Nx = 8 are 2 apart
    x1x = (3 + 6) % nx + nx * (1 + ny * 2)
    C = oracle.polyakov_correlator(dims, _with_time_link(dims, [(x0, qa), (x1x, qb)]), 3)
    assert np.abs(C - [plain, both, plain]).max() < 1e-15


def test_correlator_is_gauge_invariant_and_equals_the_fft_autocorrelation():
    """Eq. 3 'is gauge invariant'; and by Wiener-Khinchin the periodic autocorrelation of
    the field l along one axis is the inverse FFT of |FFT l|^2 - a library route that shares nothing
    with the double loop (the field itself is pinned by the centre-flip and 2x2-matrix tests)."""
    dims = [8, 6, 10, 4]
    L = oracle.init(dims, "hot", 12)
    for i in range(2):
        oracle.heatbath_sweep(dims, L, 2.6, 12, i)
    C = oracle.polyakov_correlator(dims, L, 3)
    G = L.copy()
    oracle.gauge_transform(dims, G, 9)
    assert np.abs(oracle.polyakov_correlator(dims, G, 3) - C).max() < 1e-14
    _, field = oracle.polyakov_loop(dims, L, return_field=True)
    f = field.reshape(dims[2], dims[1], dims[0])  # [z][y][x]
    want = np.zeros(3)
    for ax in range(3):
        F = np.fft.fft(f, axis=ax)
        ac = np.fft.ifft(F * np.conj(F), axis=ax).real  # sum_x l(x) l(x + r) along ax, at index r
        want += np.array([np.take(ac, r, axis=ax).sum() for r in (1, 2, 3)])
    want /= 3 * f.size
    assert np.abs(C - want).max() < 1e-14
    # C(r) = C(N - r): on the mirrored lattice (x -> -x, which maps U_t(x) to U_t(-x)) the values are the same
    Lm = L.reshape(dims[3], dims[2], dims[1], dims[0], 4, 4)[:, :, :, ::-1]
    M = np.zeros_like(L).reshape(Lm.shape)
    M[..., 3, :] = Lm[..., 3, :]     # only the time links enter; the others stay zero (never read)
    M[..., :3, 0] = 1.0
    assert np.abs(oracle.polyakov_correlator(dims, np.ascontiguousarray(M).reshape(L.shape), 3) - C).max() < 1e-14


def test_correlator_rejects_bad_rmax_and_fp32_mode_tracks_fp64():
    dims = [4, 6, 4, 2]
    L = workloads.random_links(dims, 3, np.float64)
    with pytest.raises(RuntimeError):
        oracle.polyakov_correlator(dims, L, 3)      # > min extent / 2
    with pytest.raises(RuntimeError):
        oracle.polyakov_correlator(dims, L, 0)
    a = oracle.polyakov_correlator(dims, L, 2)
    b = oracle.polyakov_correlator(dims, L.astype(np.float32), 2, "f32")
    assert np.abs(a - b).max() < 2e-7


def test_returned_delta_is_one_minus_the_scalar_part_of_the_new_link_times_vbar():
    """heatbath_*(delta=...) hands out the accepted delta = 1 - x0 of each link ([R13b]'s second amplifier). By
    [R7] U' = X Vbar^dagger, so the scalar part of U' Vbar is x0: recomputed here from the returned link, the pinned
    staple and the pinned quaternion product. The degenerate [R8] branch reports delta = 1."""
    dims = [4, 4, 6, 2]
    L = workloads.random_links(dims, 23, np.float64)
    V = oracle.volume(dims)
    for mu, p in ((1, 0), (2, 1)):
        before = L.copy()
        dl = np.full((V, 4), -7.0)
        oracle.heatbath_substep(dims, L, 1.7, 3, 2, mu, p, delta=dl)
        sites = np.flatnonzero(dl[:, mu] != -7.0)
        assert len(sites) == V // 2 and (dl[:, [n for n in range(4) if n != mu]] == -7.0).all()
        assert (dl[sites, mu] > 0).all() and (dl[sites, mu] < 2).all()
        for s in sites[::7]:
            v = oracle.staple(dims, before, int(s), mu)
            x = oracle.qmul(L[s, mu], v / np.linalg.norm(v))
            assert abs((1.0 - x[0]) - dl[s, mu]) < 1e-14
            assert oracle.heatbath_link(dims, before, 1.7, 3, 2, int(s), mu, return_delta=True)[3] == dl[s, mu]
    Z = workloads.degenerate_staple_links((4, 4, 4, 4), 37, 1)
    assert oracle.heatbath_link((4, 4, 4, 4), Z, 2.3, 5, 0, 37, 1, return_delta=True)[3] == 1.0
