"""GPU parity tests proper (-m gpu): the CUDA path, called through the C-ABI
binding, against the CPU oracle on the same seeded inputs, element by element.

Tolerances (BASELINE.json north_star): links after one sweep |d| <= 1e-12 (fp64),
1e-5 (fp32); per-sweep mean plaquette 1e-12 (fp64), 1e-6 (fp32). The comparison
protocol - which deviations are excused (rounding-flipped accept decisions [R13],
ill-conditioned updates [R13b], links downstream of either), how they are counted,
and that observables are never skipped - is tests/parity_protocol.py."""
import numpy as np
import pytest

import oracle
import parity_protocol as pp
from paper_1104_5432_b200 import workloads
from parity_protocol import MODE, PTOL, SWEEP, TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    import paper_1104_5432_b200 as p
    from paper_1104_5432_b200 import build
    build.build()  # no-op unless a source is newer than the library
    p.lib()
    return p


def assert_links_equal_within_tol(gpu, ora, prec, what=""):
    """no excuse of any kind (fp64 chains, untouched links)"""
    d = np.abs(gpu.astype(np.float64) - ora.astype(np.float64))
    assert d.max() <= TOL[prec], f"{what}: max |d| = {d.max():.3e}"


# dims: tiled path with the 8x4x2x2-thread tile (16,8,8,4) and the 16x4x2x1 tile (32,4,4,2),
# linear path (8^4), ragged, minimal
SHAPES = [(16, 8, 8, 4), (32, 4, 4, 2), (8, 8, 8, 8), (6, 4, 10, 2), (2, 2, 2, 2), (4, 2, 6, 2)]


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", SHAPES)
def test_init_matches_oracle(pkg, dims, prec):
    lat = pkg.Lattice(dims, prec)
    lat.init("cold", 5)
    g = lat.get_links()
    assert (g[..., 0] == 1).all() and (g[..., 1:] == 0).all()
    assert lat.mean_plaquette() == 1.0 and lat.polyakov_loop() == 1.0
    lat.init("hot", 5)
    g = lat.get_links()
    o = oracle.init(dims, "hot", 5, MODE[prec])
    # uniforms are bit-identical; only sqrt/sincos rounding differs
    assert np.abs(g.astype(np.float64) - o.astype(np.float64)).max() < (2e-15 if prec == 64 else 1e-6)  # oracle rounds 2*pi*u before sin/cos
    lat.close()


@pytest.mark.parametrize("prec", [64, 32])
def test_set_get_roundtrip_is_bit_exact(pkg, prec):
    dims = (6, 4, 10, 2)
    L = workloads.random_links(dims, 3, np.float64 if prec == 64 else np.float32)
    lat = pkg.Lattice(dims, prec)
    lat.set_links(L)
    assert (lat.get_links() == L).all()
    lat.close()


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", SHAPES)
def test_every_substep_matches_oracle_teacher_forced(pkg, dims, prec):
    mode = MODE[prec]
    beta, seed, sweep = 2.3, 11, 4
    L = workloads.random_links(dims, 21, oracle.dtype(mode))
    lat = pkg.Lattice(dims, prec)
    lat.set_seed(seed)
    V = oracle.volume(dims)
    for mu in range(4):
        for p in range(2):
            lat.set_links(L)  # teacher forcing: same input on both sides
            lat.substep(beta, sweep, mu, p)
            g = lat.get_links()
            o = L.copy()
            rec = pp.Records(V)
            oracle.heatbath_substep(dims, o, beta, seed, sweep, mu, p, mode, **rec.kw)
            pp.compare_links(g, o, dims, prec, [(mu, p)], rec, beta, what=f"mu={mu} p={p}")
            # only the links of this sub-step changed
            untouched = np.ones((V, 4), bool)
            s = np.arange(V)
            par = (s % dims[0] + s // dims[0] % dims[1] + s // (dims[0] * dims[1]) % dims[2]
                   + s // (dims[0] * dims[1] * dims[2])) % 2
            untouched[par == p, mu] = False
            assert (g[untouched] == L[untouched]).all()
            L = o  # continue from the oracle's state
    lat.close()


@pytest.mark.parametrize("eps,beta", [(0.05, 6.0), (0.3, 2.3), (0.01, 100.0), (0.001, 5000.0)])
@pytest.mark.parametrize("prec", [64, 32])
def test_sweep_on_smooth_lattice_matches_oracle(pkg, prec, eps, beta):
    """Thermalised-like inputs (large staple norm, alpha ~ 30 at beta = 6); the last two are the
    weak-coupling extreme (alpha ~ 600 and ~ 3e4: delta ~ 1/alpha, x0 = 1 - delta within a few ulp of 1
    in fp32, the direction on a sphere of radius sqrt(2 delta))."""
    dims = (16, 8, 8, 4)
    mode = MODE[prec]
    L = workloads.smooth_links(dims, 9, eps, oracle.dtype(mode))
    lat = pkg.Lattice(dims, prec)
    lat.set_links(L)
    lat.set_seed(77)
    lat.sweep(beta, 3)
    g = lat.get_links()
    rec = pp.Records(oracle.volume(dims))
    oracle.heatbath_sweep(dims, L, beta, 77, 3, mode, **rec.kw)
    rep = pp.compare_links(g, L, dims, prec, SWEEP, rec, beta, haar=False)
    P, Lp = lat.measure()
    pp.check_observables(P, Lp, g, dims, prec, rep, L)
    lat.close()


def test_config1_ten_sweeps_links_and_plaquette(pkg):
    """BASELINE.json configs[0]: 8^4 fp64, hot start seed 1, beta 2.3, 10 sweeps,
    plaquette after each; teacher-forced link parity AND free-running plaquette."""
    w = workloads.C1
    dims = w.dims
    L = oracle.init(dims, "hot", w.seed)
    lat = pkg.Lattice(dims, 64)
    free = pkg.Lattice(dims, 64)
    free.init("hot", w.seed)
    lat.set_seed(w.seed)
    for i in range(w.sweeps):
        lat.set_links(L)
        lat.sweep(w.betas[0], i)
        free.sweep(w.betas[0], i)
        oracle.heatbath_sweep(dims, L, w.betas[0], w.seed, i)
        assert_links_equal_within_tol(lat.get_links(), L, 64, what=f"sweep {i}")
        P = oracle.mean_plaquette(dims, L)
        assert abs(lat.mean_plaquette() - P) < 1e-12
        # in fp64 no accept decision flips (probability ~1e-16 per link), so the
        # free-running trajectory stays on the oracle's
        assert abs(free.mean_plaquette() - P) < 1e-12
        assert abs(free.polyakov_loop() - oracle.polyakov_loop(dims, L)) < 1e-12
    # free-running links: rounding differences (1e-16 per update) grow chaotically from
    # sweep to sweep (measured ~1e-11 after 10 sweeps); the 1e-12 gate is the teacher-forced one
    assert np.abs(free.get_links() - L).max() < 1e-9
    lat.close()
    free.close()


@pytest.mark.parametrize("prec", [64, 32])
def test_fp32_and_fp64_ten_sweeps_16c4_teacher_forced(pkg, prec):
    """configs[1] shape (16^3 x 4), several teacher-forced sweeps with P and L each."""
    dims = (16, 16, 16, 4)
    mode = MODE[prec]
    L = oracle.init(dims, "hot", 100, mode)
    lat = pkg.Lattice(dims, prec)
    lat.set_seed(100)
    V = oracle.volume(dims)
    flips = 0
    for i in range(4):
        lat.set_links(L)
        lat.sweep(2.4, i)
        rec = pp.Records(V)
        oracle.heatbath_sweep(dims, L, 2.4, 100, i, mode, **rec.kw)
        g = lat.get_links()
        # sweep 0 starts from the Haar-random hot start (small staple norms occur), later ones from beta = 2.4
        rep = pp.compare_links(g, L, dims, prec, SWEEP, rec, 2.4, haar=(i == 0), what=f"sweep {i}")
        flips += rep.flips
        P, Lp = lat.measure()
        pp.check_observables(P, Lp, g, dims, prec, rep, L, what=f"sweep {i}")
    assert flips <= pp.flip_budget(4 * 4 * V, prec)
    lat.close()


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", SHAPES + [(12, 6, 4, 6)])
def test_plaquette_and_polyakov_match_oracle(pkg, dims, prec):
    mode = MODE[prec]
    L = workloads.random_links(dims, 31, oracle.dtype(mode))
    lat = pkg.Lattice(dims, prec)
    lat.set_links(L)
    tol = 1e-14 if prec == 64 else 2e-7
    assert abs(lat.mean_plaquette() - oracle.mean_plaquette(dims, L, mode)) < tol
    assert abs(lat.polyakov_loop() - oracle.polyakov_loop(dims, L, mode)) < tol
    P, Lp = lat.measure()
    assert P == lat.mean_plaquette() and Lp == lat.polyakov_loop()  # fixed-order reduction: same bits
    # smooth lattice: values near 1 test the relative accuracy
    S = workloads.smooth_links(dims, 32, 0.1, oracle.dtype(mode))
    lat.set_links(S)
    assert abs(lat.mean_plaquette() - oracle.mean_plaquette(dims, S, mode)) < tol
    assert abs(lat.polyakov_loop() - oracle.polyakov_loop(dims, S, mode)) < tol
    lat.close()


def test_gauge_invariance_on_gpu(pkg):
    dims = (8, 8, 8, 4)
    L = oracle.init(dims, "hot", 2)
    G = L.copy()
    oracle.gauge_transform(dims, G, 5)
    lat = pkg.Lattice(dims, 64)
    lat.set_links(L)
    a = lat.measure()
    lat.set_links(G)
    b = lat.measure()
    assert abs(a[0] - b[0]) < 1e-14 and abs(a[1] - b[1]) < 1e-14
    lat.close()


@pytest.mark.parametrize("prec", [64, 32])
def test_polyakov_correlator_matches_oracle(pkg, prec):
    """NEXT-1 (eq. 3) against the oracle's direct double loop, unequal spatial extents."""
    dims, mode = (12, 8, 10, 4), MODE[prec]
    L = oracle.init(dims, "hot", 8, mode)
    for i in range(2):
        oracle.heatbath_sweep(dims, L, 2.6, 8, i, mode)
    lat = pkg.Lattice(dims, prec)
    lat.set_links(L)
    got = lat.polyakov_correlator(4)
    want = oracle.polyakov_correlator(dims, L, 4, mode)
    assert np.abs(got - want).max() < (1e-14 if prec == 64 else 2e-7)
    with pytest.raises(pkg.SU2Error):
        lat.polyakov_correlator(5)  # > min extent / 2
    lat.close()


@pytest.mark.parametrize("nt", [4, 8])
def test_polyakov_correlator_config4_full_size(pkg, nt):
    """BASELINE.json configs[3]: 48^3 x N_t in fp64 at beta = 2.5, correlator for r = 1..24, after a few
    sweeps from the hot start (seed 200 + N_t); every r against the oracle on the GPU's configuration."""
    dims = (48, 48, 48, nt)
    lat = pkg.Lattice(dims, 64)
    lat.init("hot", 200 + nt)
    for i in range(5):
        lat.sweep(2.5, i)
    got = lat.polyakov_correlator(24)
    L = lat.get_links()
    want = oracle.polyakov_correlator(dims, L, 24, "f64")
    assert np.abs(got - want).max() < 1e-13, np.abs(got - want).max()
    assert abs(lat.polyakov_loop() - oracle.polyakov_loop(dims, L, "f64")) < 1e-12
    # C(r) of a finite-temperature configuration is not trivial: it decays from C(1)
    assert want[0] > want[5] and np.abs(want).max() < 1.0
    lat.close()


def test_reproducible_and_sweep_idx_matters(pkg):
    dims = (16, 8, 8, 4)
    a = pkg.Lattice(dims, 32)
    b = pkg.Lattice(dims, 32)
    for lat in (a, b):
        lat.init("hot", 9)
    a.sweep(2.3, 0)
    b.sweep(2.3, 0)
    ga, gb = a.get_links(), b.get_links()
    assert (ga == gb).all()
    b.init("hot", 9)
    b.sweep(2.3, 1)
    assert np.abs(b.get_links() - ga).max() > 0.1
    a.close()
    b.close()


def test_error_paths_on_gpu(pkg):
    lat = pkg.Lattice((4, 4, 4, 4), 64)
    with pytest.raises(pkg.SU2Error) as e:
        lat.sweep(2.3, 0)  # before init
    assert e.value.code == pkg.SU2_ESTATE
    lat.init("cold", 1)
    for bad in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(pkg.SU2Error) as e:
            lat.sweep(bad, 0)
        assert e.value.code == pkg.SU2_EARG
    with pytest.raises(pkg.SU2Error):
        lat.substep(2.3, 0, 4, 0)
    with pytest.raises(AssertionError):
        pkg.su2_set_links(lat.h, np.zeros((3, 4, 4))[:, ::2])  # non-contiguous rejected by the binding
    import ctypes as C
    buf = np.zeros(10)
    assert pkg.lib().su2_set_links(lat.h, C.c_void_p(buf.ctypes.data), buf.nbytes) == pkg.SU2_EARG
    lat.sweep(2.3, 0)  # still usable after argument errors
    assert 0.0 < lat.mean_plaquette() <= 1.0
    lat.close()
    # library-owned memory variant
    h = pkg.su2_lattice_create(4, 4, 4, 4, 32)
    pkg.su2_init(h, pkg.SU2_START_COLD, 0)
    assert pkg.su2_mean_plaquette(h) == 1.0
    pkg.su2_lattice_destroy(h)


@pytest.mark.parametrize("prec", [64, 32])
def test_unit_norm_invariant_after_sweeps(pkg, prec):
    dims = (16, 8, 8, 8)
    lat = pkg.Lattice(dims, prec)
    lat.init("hot", 3)
    for i in range(5):
        lat.sweep(6.0, i)
    g = lat.get_links().astype(np.float64)
    assert np.abs((g**2).sum(-1) - 1).max() < (9e-16 if prec == 64 else 5e-7)  # 4 ulp on |a|^2
    lat.close()


@pytest.mark.parametrize("beta", [0.05, 0.3, 1.0])
def test_fp32_small_alpha_exercises_the_accurate_refinement(pkg, beta):
    """At small alpha = beta*k most accepted trials fall under the kernel's refinement
    threshold (radius^2 < 0.12/alpha^2) and many trials are rejected:
    covers the accurate logf/cospif branch and the multi-trial loop."""
    dims, prec, mode = (16, 8, 8, 4), 32, "f32"
    L = workloads.random_links(dims, 5, np.float32)
    lat = pkg.Lattice(dims, prec)
    lat.set_seed(9)
    V = oracle.volume(dims)
    most = 0
    for mu, p in ((0, 0), (1, 1), (3, 0)):
        lat.set_links(L)  # teacher-forced: a flipped accept must not feed the next sub-step
        lat.substep(beta, 0, mu, p)
        g = lat.get_links()
        rec, tr = pp.Records(V), np.zeros((V, 4), np.int32)
        oracle.heatbath_substep(dims, L, beta, 9, 0, mu, p, mode, trials=tr, **rec.kw)
        most = max(most, int(tr.max()))
        # many trials per link at small alpha: each is a chance of a marginal decision
        pp.compare_links(g, L, dims, prec, [(mu, p)], rec, beta, max_flips=pp.flip_budget(int(tr.sum()), prec),
                         what=f"mu={mu} p={p}")
    assert most >= 5  # the retry loop really ran
    lat.close()


def test_substeps_in_any_order_match_oracle(pkg):
    """Sub-steps called out of the canonical order must not overlap their predecessor
    (the handle only allows programmatic dependent launch after the canonical one)."""
    dims, prec, mode = (32, 8, 8, 4), 64, "f64"
    L = workloads.random_links(dims, 8, np.float64)
    lat = pkg.Lattice(dims, prec)
    lat.set_links(L)
    lat.set_seed(3)
    order = [(2, 1), (0, 0), (0, 1), (3, 0), (1, 1), (1, 0), (2, 0), (3, 1), (0, 0), (0, 1), (1, 0)]
    for mu, p in order:
        lat.substep(2.3, 1, mu, p)
    g = lat.get_links()
    for mu, p in order:
        oracle.heatbath_substep(dims, L, 2.3, 3, 1, mu, p, mode)
    assert_links_equal_within_tol(g, L, prec)
    lat.close()


@pytest.mark.parametrize("prec", [64, 32])
def test_overlapped_launches_equal_serialised_launches_bitwise(pkg, prec):
    """32^4 (many CTA waves): sweeps whose sub-steps are chained by programmatic dependent
    launch give bit-identical links to the same sweeps with the overlap disabled."""
    dims = (32, 32, 32, 32)
    res = []
    for overlap in (1, 0):
        lat = pkg.Lattice(dims, prec)
        lat.set_option("overlap", overlap)
        lat.init("hot", 2)
        for i in range(3):
            lat.sweep(6.0, i)
        res.append(lat.get_links())
        lat.close()
    assert (res[0] == res[1]).all()


@pytest.mark.parametrize("prec", [64, 32])
def test_degenerate_staple_matches_oracle(pkg, prec):
    """[R8] on the hand-built k = 0 lattice: the kernel takes the same Haar branch."""
    dims, mu = (4, 4, 4, 4), 1
    mode = MODE[prec]
    for s in (37, 38):  # one site of each parity
        L = workloads.degenerate_staple_links(dims, s, mu, oracle.dtype(mode))
        par = sum((s // int(np.prod(dims[:d]))) % dims[d] for d in range(4)) % 2
        lat = pkg.Lattice(dims, prec)
        lat.set_links(L)
        lat.set_seed(5)
        lat.substep(2.3, 0, mu, par)
        g = lat.get_links()
        tr = np.full((oracle.volume(dims), 4), -1, np.int32)
        oracle.heatbath_substep(dims, L, 2.3, 5, 0, mu, par, mode, trials=tr)
        assert tr[s, mu] == 0  # the oracle took the degenerate branch there
        assert np.abs(g[s, mu].astype(np.float64) - L[s, mu].astype(np.float64)).max() < (2e-15 if prec == 64 else 1e-6)
        assert_links_equal_within_tol(g, L, prec)
        lat.close()


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", SHAPES + [(12, 6, 4, 6)])
def test_sweep_measure_fused_plaquette_matches_oracle_and_standalone_kernel(pkg, dims, prec):
    """su2_heatbath_sweep_measure: same links as su2_heatbath_sweep (bitwise); its fused
    plaquette and its Polyakov loop equal the oracle's on the new configuration."""
    import torch
    mode = MODE[prec]
    L = workloads.random_links(dims, 13, oracle.dtype(mode))
    obs = torch.zeros(6, dtype=torch.float64, device="cuda")
    a, b = pkg.Lattice(dims, prec), pkg.Lattice(dims, prec)
    for lat in (a, b):
        lat.set_links(L)
        lat.set_seed(4)
    for i in range(3):
        a.sweep(2.3, i)
        b.sweep_measure(2.3, i, obs, i)
        ga, gb = a.get_links(), b.get_links()
        assert (ga == gb).all()
        P, Lp = obs.cpu().numpy()[2 * i: 2 * i + 2]
        pp.check_observables(P, Lp, gb, dims, prec)
        assert abs(P - a.mean_plaquette()) < (1e-13 if prec == 64 else 2e-7)
    a.close()
    b.close()


@pytest.mark.parametrize("graphs", ["1", "0"])
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", [(16, 8, 8, 4), (32, 4, 4, 2), (8, 8, 8, 8), (6, 4, 10, 2)])
def test_run_equals_step_by_step_calls_bitwise(pkg, dims, prec, graphs):
    """su2_run (captured CUDA graph replayed n times, loop state in device memory) against n
    su2_heatbath_sweep_measure calls: identical links and observables; also with the graph
    disabled (direct launches reading the same device state)."""
    import torch
    n = 7
    a, b = pkg.Lattice(dims, prec), pkg.Lattice(dims, prec)
    b.set_option("run_graph", int(graphs))
    oa = torch.zeros(2 * n, dtype=torch.float64, device="cuda")
    ob = torch.zeros(2 * n, dtype=torch.float64, device="cuda")
    for lat in (a, b):
        lat.init("hot", 21)
    for i in range(n):
        a.sweep_measure(2.4, 10 + i, oa, i)
    b.run(2.4, 10, 3, ob)          # two calls: the second replays the cached graph
    b.run(2.4, 13, n - 3, ob[6:])
    assert (a.get_links() == b.get_links()).all()
    assert (oa.cpu() == ob.cpu()).all()
    # and the oracle agrees with the whole chain in fp64 (no flips expected)
    if prec == 64:
        L = oracle.init(dims, "hot", 21, "f64")
        for i in range(n):
            oracle.heatbath_sweep(dims, L, 2.4, 21, 10 + i, "f64")
            assert abs(float(ob[2 * i]) - oracle.mean_plaquette(dims, L, "f64")) < 1e-12
        assert_links_equal_within_tol(b.get_links(), L, 64)
    a.close()
    b.close()


# ---------------------------------------------------------------- Creutz draw [R15] (S8(f) NEXT-3(i))
@pytest.fixture
def oracle_draw():
    def use(method):
        for m in ("f64", "f32", "f32x"):
            oracle.set_draw(method, m)
    yield use
    for m in ("f64", "f32", "f32x"):
        oracle.set_draw("kp", m)


@pytest.mark.parametrize("method,beta", [("creutz", 0.3), ("creutz", 2.3), ("auto", 0.3), ("auto", 0.7), ("auto", 2.3)])
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", [(16, 8, 8, 4), (32, 4, 4, 2), (8, 8, 8, 8), (6, 4, 10, 2)])
def test_creutz_and_auto_draw_match_oracle_teacher_forced(pkg, oracle_draw, dims, prec, method, beta):
    """Sub-steps with su2_set_draw(CREUTZ | AUTO) against the oracle in the same mode. At beta = 0.7
    on a hot lattice alpha = beta k straddles ALPHA_C, so 'auto' takes both branches in one launch
    (a choice decided by rounding, |alpha - ALPHA_C| tiny, is excused like a flipped accept)."""
    mode = MODE[prec]
    oracle_draw(method)
    L = workloads.random_links(dims, 21, oracle.dtype(mode))
    if method == "auto" and beta == 0.7:
        a = beta * oracle.staple_norms(dims, L, mode)
        assert (a < oracle.ALPHA_C).mean() > 0.2 and (a > oracle.ALPHA_C).mean() > 0.2
    lat = pkg.Lattice(dims, prec)
    lat.set_seed(33)
    lat.set_draw(method)
    V = oracle.volume(dims)
    for mu, p in ((0, 0), (1, 1), (2, 0), (3, 1)):
        lat.set_links(L)
        lat.substep(beta, 4, mu, p)
        g = lat.get_links()
        rec, tr = pp.Records(V), np.zeros((V, 4), np.int32)
        oracle.heatbath_substep(dims, L, beta, 33, 4, mu, p, mode, trials=tr, **rec.kw)
        pp.compare_links(g, L, dims, prec, [(mu, p)], rec, beta, max_flips=pp.flip_budget(int(tr.sum()), prec),
                         what=f"{method} mu={mu} p={p}")
    lat.close()


@pytest.mark.parametrize("prec", [64, 32])
def test_auto_draw_equals_kp_bitwise_at_large_alpha(pkg, prec):
    """beta = 6 on a smooth lattice: alpha ~ 30 everywhere, so AUTO must reproduce the KP sweep bit for bit
    (the ALT kernels differ from the hot-path kernels only by the branch)."""
    dims = (16, 8, 8, 4)
    L = workloads.smooth_links(dims, 3, 0.05, np.float64 if prec == 64 else np.float32)
    out = []
    for method in ("kp", "auto"):
        lat = pkg.Lattice(dims, prec)
        lat.set_links(L)
        lat.set_seed(8)
        lat.set_draw(method)
        for sw in range(3):
            lat.sweep(6.0, sw)
        out.append(lat.get_links())
        lat.close()
    assert (out[0] == out[1]).all()


def test_run_follows_set_draw_and_bad_method_is_rejected(pkg):
    """su2_run's captured step is rebuilt when the draw changes; results equal the step-by-step calls."""
    import torch
    dims, prec, beta, n = (16, 8, 8, 4), 64, 0.5, 4
    a, b = pkg.Lattice(dims, prec), pkg.Lattice(dims, prec)
    for lat in (a, b):
        lat.init("hot", 6)
    oa = torch.zeros(2 * n, dtype=torch.float64, device="cuda")
    ob = torch.zeros(2 * n, dtype=torch.float64, device="cuda")
    a.run(beta, 0, 2, oa)                      # captures the KP step
    a.set_draw("auto")
    a.run(beta, 2, 2, oa[4:])
    for i in range(n):
        if i == 2:
            b.set_draw("auto")
        b.sweep_measure(beta, i, ob, i)
    torch.cuda.synchronize()
    assert (a.get_links() == b.get_links()).all()
    assert torch.equal(oa, ob)
    with pytest.raises(pkg.SU2Error):
        pkg.su2_set_draw(a.h, 7)
    a.close(); b.close()


@pytest.mark.parametrize("overlap", [0, None])
@pytest.mark.parametrize("how", ["set_seed", "init"])
def test_run_after_reseed_uses_the_new_seed(pkg, how, overlap):
    """The captured step of su2_run carries the seed's expanded Philox keys as kernel parameters:
    a reseed (su2_set_seed, or su2_init with another seed) must drop it. run(seed A); reseed B;
    run must equal the step-by-step calls with seed B, bit for bit."""
    import torch
    dims, prec, beta, n = (16, 8, 8, 4), 64, 2.3, 20   # 20 steps: a captured block of 16 (or 20 one-step graphs) + 4
    a, b = pkg.Lattice(dims, prec), pkg.Lattice(dims, prec)
    if overlap is not None:
        a.set_option("tail_overlap", overlap)   # None: the automatic default (on at this size)
    oa = torch.zeros(4 * n, dtype=torch.float64, device="cuda")
    ob = torch.zeros(4 * n, dtype=torch.float64, device="cuda")
    a.init("hot", 1)
    b.init("hot", 1)
    a.run(beta, 0, n, oa)                       # captures the step with seed 1
    for i in range(n):
        b.sweep_measure(beta, i, ob, i)
    if how == "set_seed":
        a.set_seed(2)
        b.set_seed(2)
    else:
        a.init("hot", 2)
        b.init("hot", 2)
    a.run(beta, n, n, oa[2 * n:])
    for i in range(n):
        b.sweep_measure(beta, n + i, ob, n + i)
    torch.cuda.synchronize()
    assert (a.get_links() == b.get_links()).all()
    assert torch.equal(oa, ob)
    # ... and the oracle agrees on which stream that is: the first steps after the reseed (later ones drift apart
    # chaotically from rounding, see test_config1_ten_sweeps_links_and_plaquette)
    if how == "init":
        L = oracle.init(dims, "hot", 2, "f64")
        for i in range(3):
            oracle.heatbath_sweep(dims, L, beta, 2, n + i, "f64")
            assert abs(float(oa[2 * (n + i)]) - oracle.mean_plaquette(dims, L, "f64")) < 1e-12
    a.close(); b.close()


@pytest.mark.parametrize("graphs", [1, 0])
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", [(16, 8, 8, 4), (32, 32, 32, 32), (6, 4, 10, 2)])
def test_run_with_tail_overlap_equals_plain_run_bitwise(pkg, dims, prec, graphs):
    """SU2_OPT_TAIL_OVERLAP: the Polyakov kernel of step i on a second stream beside step i+1, two alternating sets
    of fused-plaquette partials and loop states, blocks of 16 steps per graph plus a directly enqueued remainder. Links and every observable equal the plain su2_run's bit for bit."""
    import torch
    n1, n2 = 37, 5   # 37 = 2 blocks of 16 + 5 directly enqueued steps; 5 = remainder only
    a, b = pkg.Lattice(dims, prec), pkg.Lattice(dims, prec)
    a.set_option("tail_overlap", 0)   # the plain run (the default is automatic: on for lattices of this size)
    b.set_option("tail_overlap", 1)
    b.set_option("run_graph", graphs)
    oa = torch.zeros(2 * (n1 + n2), dtype=torch.float64, device="cuda")
    ob = torch.zeros(2 * (n1 + n2), dtype=torch.float64, device="cuda")
    for lat, o in ((a, oa), (b, ob)):
        lat.init("hot", 4)
        lat.run(2.4, 0, n1, o)
        lat.run(2.4, n1, n2, o[2 * n1:])
    torch.cuda.synchronize()
    assert torch.equal(oa, ob)
    assert (a.get_links() == b.get_links()).all()
    # switching the option off again drops the captured block
    b.set_option("tail_overlap", 0)
    a.set_option("tail_overlap", 1)
    a.run(2.4, 100, 3, oa)
    b.run(2.4, 100, 3, ob)
    torch.cuda.synchronize()
    assert torch.equal(oa[:6], ob[:6]) and (a.get_links() == b.get_links()).all()
    a.close(); b.close()


def test_set_option_rejects_bad_arguments(pkg):
    lat = pkg.Lattice((4, 4, 4, 4), 32)
    for opt, val in ((7, 1), (pkg.SU2_OPT_OVERLAP, 2), (pkg.SU2_OPT_RUN_GRAPH, -1)):
        with pytest.raises(pkg.SU2Error) as e:
            pkg.su2_set_option(lat.h, opt, val)
        assert e.value.code == pkg.SU2_EARG
    lat.set_option("overlap", 0)
    lat.set_option("run_graph", 0)
    lat.init("cold", 1)
    lat.sweep(2.3, 0)
    assert 0.0 < lat.mean_plaquette() <= 1.0
    lat.close()


# ---------------------------------------------------------------- replica batches (S8(f) NEXT-2)
@pytest.mark.parametrize("method", ["kp", "auto"])
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", [(16, 16, 16, 4), (32, 4, 4, 2), (8, 8, 8, 8), (6, 4, 10, 2)])
def test_batch_equals_single_lattices_bitwise_and_matches_oracle(pkg, oracle_draw, dims, prec, method):
    """A batch of 5 replicas (config 2's beta scan: own beta, own seed each) stepped by
    su2_batch_sweep_measure equals, bit for bit, 5 single-lattice handles stepped by
    su2_heatbath_sweep_measure (same Philox streams, same arithmetic, same reduction order);
    and replica 3 after one teacher-forced batch step matches the oracle."""
    import torch
    betas = [2.2, 2.3, 2.4, 2.5, 0.6 if method == "auto" else 2.6]
    seeds = [100 + i for i in range(5)]
    R, n = 5, 3
    bat = pkg.Lattice(dims, prec, replicas=R)
    bat.set_draw(method)
    bat.batch_init("hot", seeds)
    ob = torch.zeros(2 * R * n, dtype=torch.float64, device="cuda")
    for i in range(n):
        bat.batch_sweep_measure(betas, i, ob, i)
    torch.cuda.synchronize()
    ob = ob.cpu().numpy().reshape(n, R, 2)
    for r in range(R):
        one = pkg.Lattice(dims, prec)
        one.set_draw(method)
        one.init("hot", seeds[r])
        o1 = torch.zeros(2 * n, dtype=torch.float64, device="cuda")
        for i in range(n):
            one.sweep_measure(betas[r], i, o1, i)
        torch.cuda.synchronize()
        bat.select(r)
        assert (bat.get_links() == one.get_links()).all(), r
        assert (ob[:, r, :] == o1.cpu().numpy().reshape(n, 2)).all(), r
        # single-lattice calls act on the selected replica
        assert bat.mean_plaquette() == one.mean_plaquette()
        one.close()
    # teacher-forced against the oracle: load a known configuration into replica 3 only
    mode = MODE[prec]
    oracle_draw(method)
    L = workloads.random_links(dims, 77, oracle.dtype(mode))  # Haar-random: small staple norms occur [R13b]
    bat.select(3)
    bat.set_links(L)
    out = torch.zeros(2 * R, dtype=torch.float64, device="cuda")
    bat.batch_sweep_measure(betas, 9, out, 0)
    g = bat.get_links()
    V = oracle.volume(dims)
    rec = pp.Records(V)
    oracle.heatbath_sweep(dims, L, betas[3], seeds[3], 9, mode, **rec.kw)
    rep = pp.compare_links(g, L, dims, prec, SWEEP, rec, betas[3], what="batch replica 3")
    P, Lp = out.cpu().numpy()[6:8]
    pp.check_observables(P, Lp, g, dims, prec, rep, L, what="batch replica 3")
    bat.close()


@pytest.mark.parametrize("graphs", [1, 0])
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", [(16, 16, 16, 4), (32, 4, 4, 2), (6, 4, 10, 2)])
def test_batch_run_equals_round_by_round_calls_bitwise(pkg, dims, prec, graphs):
    """su2_batch_run (one round captured as a CUDA graph, replayed; sweep index and output slot in device memory, the
    loop state advanced once per round by the last CTA of the last replica) against su2_batch_sweep_measure called
    round by round: identical links of every replica and identical observables; two calls in a row, a change of
    couplings in between, and - on the same handle - su2_run on one selected replica afterwards."""
    import torch
    R, n1, n2 = 5, 6, 5
    seeds = [300 + r for r in range(R)]
    b1 = [2.2 + 0.1 * r for r in range(R)]
    b2 = [2.6 - 0.1 * r for r in range(R)]
    a, b = pkg.Lattice(dims, prec, replicas=R), pkg.Lattice(dims, prec, replicas=R)
    b.set_option("run_graph", graphs)
    oa = torch.zeros(2 * R * (n1 + n2), dtype=torch.float64, device="cuda")
    ob = torch.zeros(2 * R * (n1 + n2), dtype=torch.float64, device="cuda")
    for lat in (a, b):
        lat.batch_init("hot", seeds)
    for i in range(n1):
        a.batch_sweep_measure(b1, i, oa, i)
    for i in range(n2):
        a.batch_sweep_measure(b2, n1 + i, oa, n1 + i)
    b.batch_run(b1, 0, n1, ob)
    b.batch_run(b2, n1, n2, ob[2 * R * n1:])
    torch.cuda.synchronize()
    assert torch.equal(oa, ob)
    assert float(oa.abs().min()) > 0.0          # every slot was written
    for r in range(R):
        a.select(r)
        b.select(r)
        assert (a.get_links() == b.get_links()).all(), r
    # the single-lattice loop on a replica of the same handle still works (it shares the loop state with the batch loop)
    o1, o2 = torch.zeros(6, dtype=torch.float64, device="cuda"), torch.zeros(6, dtype=torch.float64, device="cuda")
    a.select(2)
    b.select(2)
    for i in range(3):
        a.sweep_measure(2.4, 50 + i, o1, i)
    b.run(2.4, 50, 3, o2)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2) and (a.get_links() == b.get_links()).all()
    b.batch_run(b1, 60, 2, ob)                 # ... and the batch loop after it
    for i in range(2):
        a.batch_sweep_measure(b1, 60 + i, oa, i)
    torch.cuda.synchronize()
    assert torch.equal(oa[:4 * R], ob[:4 * R])
    with pytest.raises(pkg.SU2Error):
        b.batch_run([2.3] * (R - 1) + [-1.0], 70, 1, ob)
    a.close(); b.close()


@pytest.mark.parametrize("dims,R,why", [
    ((32, 4, 64, 64), 40, "2048 z-t tiles of the first shape x 40 replicas exceed grid z: second tile shape"),
    ((16, 4, 64, 128), 33, "first shape does not divide Nx/2 = 8, second gives 2048 x 33 > 65535: linear launch"),
])
def test_batch_falls_back_to_another_launch_shape_instead_of_failing(pkg, dims, R, why):
    """A batch carries the replica in grid z next to the z-t tiles; where that exceeds the grid limit, create picks
    the next tile shape or the linear launch (round 1 returned SU2_EARG). Draws are keyed by the site, so the links
    equal those of single-lattice handles (which use another launch shape) bit for bit."""
    import torch
    bat = pkg.Lattice(dims, 32, replicas=R)
    seeds = [500 + r for r in range(R)]
    betas = [2.2 + 0.01 * r for r in range(R)]
    bat.batch_init("hot", seeds)
    out = torch.zeros(2 * R * 2, dtype=torch.float64, device="cuda")
    for i in range(2):
        bat.batch_sweep_measure(betas, i, out, i)
    torch.cuda.synchronize()
    o = out.cpu().numpy().reshape(2, R, 2)
    for r in (0, R // 2, R - 1):
        one = pkg.Lattice(dims, 32)
        one.init("hot", seeds[r])
        o1 = torch.zeros(4, dtype=torch.float64, device="cuda")
        for i in range(2):
            one.sweep_measure(betas[r], i, o1, i)
        torch.cuda.synchronize()
        bat.select(r)
        assert (bat.get_links() == one.get_links()).all(), (r, why)
        # the fused-plaquette partials follow the launch shape: same value to rounding, not the same bits
        assert np.abs(o[:, r, :] - o1.cpu().numpy().reshape(2, 2)).max() < 2e-7
        one.close()
    bat.close()


def test_batch_argument_checks(pkg):
    import torch
    with pytest.raises(pkg.SU2Error):
        pkg.su2_lattice_create_batch(8, 8, 8, 8, 32, 0)
    bat = pkg.Lattice((8, 8, 8, 4), 32, replicas=2)
    assert pkg.su2_replicas(bat.h) == 2
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    with pytest.raises(pkg.SU2Error):     # not initialised
        bat.batch_sweep_measure([2.3, 2.3], 0, out, 0)
    bat.init("hot", 1)                    # replica 0 only
    with pytest.raises(pkg.SU2Error):
        bat.batch_sweep_measure([2.3, 2.3], 0, out, 0)
    bat.select(1)
    bat.init("cold", 2)
    bat.batch_sweep_measure([2.3, 2.3], 0, out, 0)
    with pytest.raises(pkg.SU2Error):
        bat.batch_sweep_measure([2.3, -1.0], 1, out, 0)
    with pytest.raises(pkg.SU2Error):
        bat.select(2)
    bat.close()
