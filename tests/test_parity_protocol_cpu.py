"""The comparison protocol itself (tests/parity_protocol.py) on the CPU: its dependency geometry is
pinned against the oracle (which links change when one link is perturbed), and its verdicts on
hand-made deviations are the ones DESIGN.md §3 [R13]/[R13b] states."""
import numpy as np
import pytest

import oracle
import parity_protocol as pp
from paper_1104_5432_b200 import workloads


@pytest.mark.parametrize("dims", [(4, 6, 4, 2), (2, 2, 2, 2), (4, 4, 4, 4)])
def test_staple_dependency_geometry_matches_the_oracle(dims):
    """Perturb one link; the links of sub-step (mu, p) that the oracle then computes differently are
    exactly those whose staple [R3] contains it - what staple_inputs_any() predicts."""
    nx, ny, nz, nt = dims
    V = oracle.volume(dims)
    L = workloads.random_links(dims, 4, np.float64)
    rng = np.random.default_rng(1)
    par = pp.parity_grid(dims)
    for trial in range(6):
        s0, nu0 = int(rng.integers(V)), int(rng.integers(4))
        Lp = L.copy()
        Lp[s0, nu0] = workloads.random_links((2, 2, 2, 2), 100 + trial)[0, 0]
        flag = np.zeros((V, 4), bool)
        flag[s0, nu0] = True
        flag = flag.reshape(nt, nz, ny, nx, 4)
        for mu in range(4):
            for p in range(2):
                a, b = L.copy(), Lp.copy()
                oracle.heatbath_substep(dims, a, 2.3, 9, 0, mu, p)
                oracle.heatbath_substep(dims, b, 2.3, 9, 0, mu, p)
                changed = (np.abs(a - b).max(-1) > 0).reshape(nt, nz, ny, nx, 4)
                changed[flag] = False   # the perturbed link itself (overwritten if it is in the sub-step)
                want = pp.staple_inputs_any(flag, mu) & (par == p)
                assert np.array_equal(changed[..., mu], want), (trial, mu, p)
                others = np.delete(changed, mu, axis=-1)
                assert not others.any()


BETA = 2.3


def _sweep_records(dims, mode, seed=3):
    L = workloads.random_links(dims, 8, oracle.dtype(mode))
    rec = pp.Records(oracle.volume(dims))
    oracle.heatbath_sweep(dims, L, BETA, seed, 0, mode, **rec.kw)
    return L, rec.margin, rec.knorm


def R(mg, kn):
    """Records with hand-set margins / staple norms and a well-conditioned draw (delta = 1)"""
    rec = pp.Records(len(mg))
    rec.margin, rec.knorm = mg, kn
    return rec


def test_protocol_verdicts_on_hand_made_deviations():
    dims, prec = (8, 4, 4, 4), 32
    ora, mg, kn = _sweep_records(dims, "f32")
    V = oracle.volume(dims)
    # identical and within-tolerance results are clean
    assert pp.compare_links(ora, ora, dims, prec, pp.SWEEP, R(mg, kn), BETA).clean
    near = ora + np.float32(3e-6)
    assert pp.compare_links(near, ora, dims, prec, pp.SWEEP, R(mg, kn), BETA).clean
    # an O(1) deviation with a healthy margin and a healthy k has no excuse
    s, mu = 77, 3   # direction 3 is updated last: nothing is downstream of it
    assert mg[s, mu] > 1e-3 and kn[s, mu] > 0.5
    gpu = ora.copy()
    gpu[s, mu] = -gpu[s, mu]
    with pytest.raises(AssertionError, match="no excuse"):
        pp.compare_links(gpu, ora, dims, prec, pp.SWEEP, R(mg, kn), BETA)
    # the same deviation with a marginal accept decision is one flip ...
    m2 = mg.copy()
    m2[s, mu] = 3e-7
    r = pp.compare_links(gpu, ora, dims, prec, pp.SWEEP, R(m2, kn), BETA)
    assert (r.flips, r.conditioned, r.downstream) == (1, 0, 0)
    # ... two such links exceed the budget of a 2048-link sweep
    gpu2 = gpu.copy()
    gpu2[s + 2, mu] = -gpu2[s + 2, mu]
    m2[s + 2, mu] = 1e-7
    with pytest.raises(AssertionError, match="budget"):
        pp.compare_links(gpu2, ora, dims, prec, pp.SWEEP, R(m2, kn), BETA)
    # a flip in an early sub-step excuses what is downstream of it, and only that
    s1, mu1 = 40, 0
    gpu = ora.copy()
    gpu[s1, mu1] = -gpu[s1, mu1]
    m3 = mg.copy()
    m3[s1, mu1] = 1e-8
    nx, ny, nz, nt = dims
    flag = np.zeros((nt, nz, ny, nx, 4), bool)
    flag.reshape(V, 4)[s1, mu1] = True
    par = pp.parity_grid(dims)
    p1 = int(par.reshape(-1)[s1])
    hit = pp.staple_inputs_any(flag, 1) & (par == 1 - p1)       # links of sub-step (1, 1 - p1) that read it
    idx = np.flatnonzero(hit.reshape(-1))
    assert len(idx) > 0
    gpu[idx[0], 1] = -gpu[idx[0], 1]
    r = pp.compare_links(gpu, ora, dims, prec, pp.SWEEP, R(m3, kn), BETA)
    assert (r.flips, r.downstream) == (1, 1)
    far = int(np.flatnonzero(~hit.reshape(-1) & (par.reshape(-1) == 1 - p1))[-1])
    gpu[far, 1] = -gpu[far, 1]
    with pytest.raises(AssertionError, match="no excuse"):
        pp.compare_links(gpu, ora, dims, prec, pp.SWEEP, R(m3, kn), BETA)


def test_conditioning_bound_scales_with_one_over_k_and_with_the_inputs_and_is_fp32_only():
    dims = (8, 4, 4, 4)
    ora, mg, kn = _sweep_records(dims, "f32")
    V = oracle.volume(dims)
    s, mu = 90, 3
    k2 = kn.copy()
    k2[s, mu] = 0.04                      # E_V / k = 5e-5, twice that with the delta = 1 of R(): directly and through alpha
    gpu = ora.copy()
    gpu[s, mu, 1] += np.float32(4e-5)
    r = pp.compare_links(gpu, ora, dims, 32, pp.SWEEP, R(mg, k2), BETA)
    assert (r.flips, r.conditioned) == (0, 1)
    gpu[s, mu, 1] += np.float32(9e-5)     # 1.3e-4 > 1.05e-4: more than 1/k explains
    with pytest.raises(AssertionError, match="no excuse"):
        pp.compare_links(gpu, ora, dims, 32, pp.SWEEP, R(mg, k2), BETA)
    # a well-conditioned link (k = 0.5) may exceed 1e-5 only by what the measured deviation of its inputs explains
    k3 = kn.copy()
    k3[s, mu] = 0.5
    gpu = ora.copy()
    gpu[s, mu, 2] += np.float32(2.5e-5)
    with pytest.raises(AssertionError, match="no excuse"):
        pp.compare_links(gpu, ora, dims, 32, pp.SWEEP, R(mg, k3), BETA)
    # ... one of its inputs, updated earlier in the sweep (direction 0), deviates by 8e-6 (inside tolerance):
    # (E_V + 2 x 8e-6) / 0.5 = 3.6e-5 >= 2.5e-5 (and as much again through alpha)
    s_in = s                                             # U_0(x): the staple input 'U_nu(x)' with nu = 0
    gpu[s_in, 0, 0] += np.float32(8e-6)
    r = pp.compare_links(gpu, ora, dims, 32, pp.SWEEP, R(mg, k3), BETA)
    assert (r.flips, r.conditioned, r.downstream) == (0, 1, 0)
    # the same deviation on a link of direction 3's own sub-step partner (updated later or never read) does not help
    gpu2 = ora.copy()
    gpu2[s, mu, 2] += np.float32(2.5e-5)
    gpu2[(s + 5) % V, 1, 0] += np.float32(8e-6)
    with pytest.raises(AssertionError, match="no excuse"):
        pp.compare_links(gpu2, ora, dims, 32, pp.SWEEP, R(mg, k3), BETA)
    # fp64 has no conditioning excuse and a zero flip budget
    o64, m64, k64 = _sweep_records(dims, "f64")
    g64 = o64.copy()
    g64[s, mu, 1] += 1e-11
    k64[s, mu] = 1e-4
    with pytest.raises(AssertionError, match="no excuse"):
        pp.compare_links(g64, o64, dims, 64, pp.SWEEP, R(m64, k64), BETA)
    m64[s, mu] = 1e-13
    with pytest.raises(AssertionError, match="budget"):
        pp.compare_links(g64, o64, dims, 64, pp.SWEEP, R(m64, k64), BETA)


def test_draw_radius_term():
    """A rounding of delta = 1 - x0 reaches the link amplified by |1 - delta| / sqrt(delta (2 - delta)): a link whose
    oracle delta is 1e-4 (radius 0.014) may deviate by E_D (delta + 1/alpha) / 0.014 ~ 1.3e-5 at alpha = 2.3, not more;
    the same deviation at delta = 0.5 has no excuse."""
    dims = (8, 4, 4, 4)
    ora, mg, kn = _sweep_records(dims, "f32")
    s, mu = 90, 3
    rec = R(mg, kn.copy())
    rec.knorm[s, mu] = 1.0            # alpha = 2.3, staple term 2e-6
    rec.delta[s, mu] = 1e-4
    allowed = float(pp.allowed_deviation(1e-4, 1.0, BETA, 0.0, 32))
    assert 1.2e-5 < allowed < 1.6e-5
    gpu = ora.copy()
    gpu[s, mu, 2] += np.float32(1.2e-5)
    r = pp.compare_links(gpu, ora, dims, 32, pp.SWEEP, rec, BETA)
    assert (r.flips, r.conditioned) == (0, 1)
    gpu[s, mu, 2] += np.float32(1e-5)
    with pytest.raises(AssertionError, match="no excuse"):
        pp.compare_links(gpu, ora, dims, 32, pp.SWEEP, rec, BETA)
    rec.delta[s, mu] = 0.5
    gpu = ora.copy()
    gpu[s, mu, 2] += np.float32(1.2e-5)
    with pytest.raises(AssertionError, match="no excuse"):
        pp.compare_links(gpu, ora, dims, 32, pp.SWEEP, rec, BETA)
    # x0 -> -1 (delta -> 2) is the same
    rec.delta[s, mu] = 2 - 1e-4
    assert pp.compare_links(gpu, ora, dims, 32, pp.SWEEP, rec, BETA).conditioned == 1


def test_budgets():
    assert pp.flip_budget(65536, 64) == 0 and pp.conditioned_budget(65536, 64) == 0
    assert pp.flip_budget(16, 32) == 1 and pp.flip_budget(65536, 32) == 1
    assert pp.flip_budget(4 * 32**4, 32) == int(np.ceil(5 * pp.FLIP_RATE[32] * 4 * 32**4))
    assert pp.conditioned_budget(65536, 32) == 7 and pp.conditioned_budget(65536, 32, haar=False) == 1


def test_fp32_oracle_modes_agree_under_the_protocol():
    """The oracle's two fp32 modes (float arithmetic vs double arithmetic on float storage, [R12]) play
    'GPU' and 'oracle': a real pair of roundings of the same update must pass the protocol."""
    dims = (8, 8, 4, 4)
    L = workloads.random_links(dims, 2, np.float32)
    V = oracle.volume(dims)
    a, b = L.copy(), L.copy()
    rec = pp.Records(V)
    oracle.heatbath_sweep(dims, a, BETA, 4, 1, "f32x")
    oracle.heatbath_sweep(dims, b, BETA, 4, 1, "f32", **rec.kw)
    r = pp.compare_links(a, b, dims, 32, pp.SWEEP, rec, BETA)
    assert r.flips <= 1
    pp.check_observables(oracle.mean_plaquette(dims, a, "f32x"), oracle.polyakov_loop(dims, a, "f32x"), a, dims, 32,
                         rep=r, ora_links=b)
