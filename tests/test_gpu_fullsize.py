"""Full-size parity (-m gpu) in the launch configuration bench.py times: 32^4 and
64^4 are too big for a full oracle sweep inside a test, so outputs are sampled and
recomputed one by one by the oracle from the pre-update configuration, and the
size-independent properties (unit norm, untouched links, plaquette) are checked."""
import numpy as np
import pytest

import oracle
import parity_protocol as pp
from parity_protocol import MODE, PTOL, TOL, sampled_link_excused

pytestmark = pytest.mark.gpu



@pytest.mark.parametrize("dims,prec,start,beta", [
    ((32, 32, 32, 32), 32, "hot", 6.0),
    ((32, 32, 32, 32), 64, "hot", 6.0),
    ((64, 64, 64, 64), 32, "cold", 6.0),
    ((64, 64, 64, 64), 64, "cold", 6.0),
    ((48, 48, 48, 6), 64, "hot", 2.5),
    # grid-limit fall-backs of choose_tiling: 128 x 512 z-t tiles of the first tile shape exceed grid z
    # (second shape used); Nx = 4 fits neither shape (linear launch over 1M sites)
    ((32, 8, 256, 512), 32, "hot", 2.3),
    ((4, 4, 64, 1024), 64, "hot", 2.3),
])
def test_sampled_link_parity_at_bench_sizes(dims, prec, start, beta):
    import paper_1104_5432_b200 as pkg
    mode = MODE[prec]
    seed = 1
    lat = pkg.Lattice(dims, prec)
    lat.init(start, seed)
    import torch
    obs = torch.zeros(4, dtype=torch.float64, device="cuda")
    lat.sweep_measure(beta, 0, obs, 0)  # the call bench.py times
    lat.sweep_measure(beta, 1, obs, 1)  # a cold start needs a sweep to become non-trivial
    before = lat.get_links()
    # fused plaquette / Polyakov loop of the call against the standalone kernels at full size ...
    P_fused, L_fused = obs.cpu().numpy()[2:4]
    P_gpu = lat.mean_plaquette()
    assert abs(P_fused - P_gpu) < (1e-13 if prec == 64 else 2e-7)
    assert abs(L_fused - lat.polyakov_loop()) < 1e-15
    # ... and all of them against the oracle on the same configuration, at full size (64^4 included:
    # 1e8 plaquette terms, where a reduction's rounding is largest)
    P_ora, L_ora = oracle.mean_plaquette(dims, before, mode), oracle.polyakov_loop(dims, before, mode)
    assert abs(P_fused - P_ora) < PTOL[prec] and abs(P_gpu - P_ora) < PTOL[prec], (P_fused, P_gpu, P_ora)
    assert abs(L_fused - L_ora) < PTOL[prec], (L_fused, L_ora)
    V = oracle.volume(dims)
    rng = np.random.default_rng(5)
    n_sample = 600
    s_all = np.arange(V)
    par_of = lambda s: (s % dims[0] + s // dims[0] % dims[1] + s // (dims[0] * dims[1]) % dims[2]
                        + s // (dims[0] * dims[1] * dims[2])) % 2
    flips = small = sampled = 0
    for mu, p in ((0, 0), (1, 1), (2, 0), (3, 1)):
        lat.set_links(before)
        lat.substep(beta, 2, mu, p)
        after = lat.get_links()
        # corners, faces (periodic wrap) and random interior sites of parity p
        cand = np.concatenate([rng.integers(0, V, size=4 * n_sample), [0, V - 1, dims[0] - 1, V - dims[0]],
                               np.arange(0, 2 * dims[0]), V - 1 - np.arange(0, 2 * dims[0])])
        cand = np.unique(cand[par_of(cand) == p])[: n_sample + 2 * dims[0]]
        for s in cand:
            u, tr, mg, k, dl = oracle.heatbath_link(dims, before, beta, seed, 2, int(s), mu, mode, return_k=True, return_delta=True)
            d = np.abs(after[s, mu].astype(np.float64) - u.astype(np.float64)).max()
            sampled += 1
            if d > TOL[prec]:
                why = sampled_link_excused(d, mg, k, dl, beta, prec)
                assert why, (s, mu, d, mg, k)
                flips += why == "flip"
                small += why == "conditioned"
        # properties that hold at any size
        mask = np.ones((V, 4), bool)
        mask[par_of(s_all) == p, mu] = False
        assert (after[mask] == before[mask]).all()
        upd = after[~mask].astype(np.float64)
        assert np.abs((upd**2).sum(-1) - 1).max() < (9e-16 if prec == 64 else 5e-7)  # 4 ulp on |a|^2
        assert np.abs(after[~mask] - before[~mask]).max() > 1e-3
        del after
    assert flips <= pp.flip_budget(sampled, prec) and small <= pp.conditioned_budget(sampled, prec, haar=False)
    lat.close()


@pytest.mark.parametrize("prec", [32, 64])
def test_sampled_link_parity_at_32c4_with_auto_draw(prec):
    """The ALT kernels (draw selection [R15]) at a bench size: 32^4, beta = 0.5 from a hot start, where
    'auto' takes Creutz's draw on most links and KP on the rest; sampled sites recomputed by the oracle."""
    import paper_1104_5432_b200 as pkg
    dims, beta, seed, mode = (32, 32, 32, 32), 0.5, 7, MODE[prec]
    for m in ("f64", "f32"):
        oracle.set_draw("auto", m)
    try:
        lat = pkg.Lattice(dims, prec)
        lat.set_draw("auto")
        lat.init("hot", seed)
        lat.sweep(beta, 0)
        before = lat.get_links()
        V = oracle.volume(dims)
        rng = np.random.default_rng(9)
        par_of = lambda s: (s % 32 + s // 32 % 32 + s // 1024 % 32 + s // 32768) % 2
        flips = small = sampled = n_creutz = n_kp = 0
        for mu, p in ((0, 1), (3, 0)):
            lat.set_links(before)
            lat.substep(beta, 1, mu, p)
            after = lat.get_links()
            cand = np.concatenate([rng.integers(0, V, size=1200), [0, V - 1, 31, V - 32]])
            cand = np.unique(cand[par_of(cand) == p])[:400]
            for s in cand:
                u, tr, mg, k, dl = oracle.heatbath_link(dims, before, beta, seed, 1, int(s), mu, mode, return_k=True, return_delta=True)
                n_creutz += beta * k < oracle.ALPHA_C
                n_kp += beta * k >= oracle.ALPHA_C
                d = np.abs(after[s, mu].astype(np.float64) - u.astype(np.float64)).max()
                sampled += tr
                if d > TOL[prec]:
                    why = sampled_link_excused(d, mg, k, dl, beta, prec)
                    assert why, (s, mu, d, mg, k)
                    flips += why == "flip"
                    small += why == "conditioned"
            del after
        assert n_creutz > 100 and n_kp > 20      # both branches sampled
        assert flips <= pp.flip_budget(sampled, prec) and small <= pp.conditioned_budget(sampled, prec)
        lat.close()
    finally:
        for m in ("f64", "f32", "f32x"):
            oracle.set_draw("kp", m)
