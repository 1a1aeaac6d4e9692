"""Measured rates behind the budgets of tests/parity_protocol.py (-m gpu): how often the fp32 kernel's accept
decision differs from the oracle's (a 'flip', [R13]) and how often a link needs the conditioning bound [R13b],
over > 10^7 teacher-forced link updates at 32^4 for beta = 2.3 and 6.0 ('measure the real fp32 flip
rate ... over >= 1e7 links'). Every sub-step is teacher-forced (the oracle's configuration is loaded before it),
so nothing is downstream of anything. Prints the counts; profiles/r02a.md keeps the output of one run."""
import numpy as np
import pytest

import oracle
import parity_protocol as pp

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("prec", [32, 64])
def test_flip_and_conditioning_rates_at_32c4(prec):
    import paper_1104_5432_b200 as pkg
    dims, mode = (32, 32, 32, 32), pp.MODE[prec]
    V = oracle.volume(dims)
    par = pp.parity_grid(dims).reshape(-1)
    tot = dict(links=0, flips=0, conditioned=0, margin_lt_1e6=0, k_lt_02=0, trials=0, worst_ok=0.0, worst_dk=0.0)
    cases = ((2.3, "hot"), (6.0, "hot"), (6.0, "thermalised")) if prec == 32 else ((2.3, "hot"),)
    for beta, start in cases:
        lat = pkg.Lattice(dims, prec)
        lat.init("hot", 1)
        if start == "thermalised":
            for i in range(10):
                lat.sweep(beta, 1000 + i)
        L = lat.get_links()
        lat.set_seed(5)
        for mu, p in pp.SWEEP:
            lat.set_links(L)
            lat.substep(beta, 0, mu, p)
            g = lat.get_links()
            rec, tr = pp.Records(V), np.zeros((V, 4), np.int32)
            oracle.heatbath_substep(dims, L, beta, 5, 0, mu, p, mode, trials=tr, **rec.kw)
            mg, kn = rec.margin, rec.knorm
            rep = pp.compare_links(g, L, dims, prec, [(mu, p)], rec, beta, what=f"beta={beta} {start} mu={mu} p={p}")
            sel = par == p
            d = np.abs(g.astype(np.float64) - L.astype(np.float64)).max(-1)[sel, mu]
            tot["links"] += int(sel.sum())
            tot["flips"] += rep.flips
            tot["conditioned"] += rep.conditioned
            tot["margin_lt_1e6"] += int((mg[sel, mu] < 1e-6).sum())
            tot["k_lt_02"] += int((kn[sel, mu] < 0.2).sum())
            tot["trials"] += int(tr[sel, mu].sum())
            ok = d <= pp.TOL[prec]
            tot["worst_ok"] = max(tot["worst_ok"], float(d[ok].max()))
            small = (kn[sel, mu] < 0.5) & (mg[sel, mu] > pp.FLIP_MARGIN[prec]) & (rec.delta[sel, mu] > 0.01) & (rec.delta[sel, mu] < 1.99)
            if small.any():  # |d| k of ill-conditioned staples (well-conditioned draws): what E_V has to cover
                tot["worst_dk"] = max(tot["worst_dk"], float((d * kn[sel, mu])[small].max()))
        lat.close()
    print(f"\nfp{prec}: {tot}")
    n = tot["links"]
    assert n >= (1.2e7 if prec == 32 else 4e6)
    # the budgets the parity tests use are 5x these expectations
    assert tot["flips"] <= max(3, 3 * pp.FLIP_RATE[prec] * n)
    assert tot["conditioned"] <= max(3, 3 * pp.COND_RATE[prec] * n) if prec == 32 else tot["conditioned"] == 0
    # worst_dk (printed): the largest |d| k over ill-conditioned staples with a well-conditioned draw - what E_V covers


def test_conditioned_rate_of_whole_sweeps_from_haar_random_lattices():
    """Whole fp32 sweeps (8 sub-steps, no teacher forcing in between) of Haar-random 16^3 x 4 lattices - the case in
    which the inputs of a link carry the deviations of earlier sub-steps: how many links need the conditioning
    bound (E_V + 2 S_in)/k of [R13b]. 24 lattices = 1.6e6 link updates."""
    import paper_1104_5432_b200 as pkg
    from paper_1104_5432_b200 import workloads
    dims, prec, mode = (16, 16, 16, 4), 32, "f32"
    V = oracle.volume(dims)
    lat = pkg.Lattice(dims, prec)
    lat.set_seed(9)
    links = cond = flips = down = 0
    worst = 0.0
    for s in range(24):
        L = workloads.random_links(dims, 1000 + s, np.float32)
        lat.set_links(L)
        lat.sweep(2.3, s)
        g = lat.get_links()
        rec = pp.Records(V)
        oracle.heatbath_sweep(dims, L, 2.3, 9, s, mode, **rec.kw)
        rep = pp.compare_links(g, L, dims, prec, pp.SWEEP, rec, 2.3, max_conditioned=10**6, what=f"lattice {s}")
        links += 4 * V
        cond += rep.conditioned
        flips += rep.flips
        down += rep.downstream
        worst = max(worst, rep.worst)
    lat.close()
    print(f"\nwhole sweeps, Haar-random: links={links} conditioned={cond} flips={flips} downstream={down} worst |d|={worst:.3e}")
    assert cond <= 3 * pp.COND_RATE[32] * links
