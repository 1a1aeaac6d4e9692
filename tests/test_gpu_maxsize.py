"""Large-lattice parity (-m gpu): 128^3 x 144 in fp32 = 3.0e8 sites, 19.3 GB of links.
Byte offsets pass 2^32 within one of the 8 link arrays, float indices of the canonical
buffer pass 2^32, quaternion indices of the device layout pass 2^30: any 32-bit offset
arithmetic in the kernels, the layout conversion or the binding fails here and nowhere
else in the suite. The oracle cannot sweep such a lattice inside a test, so outputs
are sampled and recomputed one by one from the pre-update configuration (the highest
sites, the corners and the wraps included), the Polyakov loop is compared in full, and
the size-independent properties are checked over the whole lattice.
Closed-form pins of the CUDA path itself: cold start P = L = 1; the mean plaquette of a
Haar-random lattice is 0 with standard deviation 1/(2 sqrt(6V))."""
import numpy as np
import pytest

import oracle
import parity_protocol as pp
from parity_protocol import sampled_link_excused

pytestmark = pytest.mark.gpu

DIMS = (128, 128, 128, 144)


def _parity_mask(dims):
    """bool (Nt, Nz, Ny, Nx): site parity (x+y+z+t) & 1, lexicographic order x fastest"""
    nx, ny, nz, nt = dims
    ax = [np.arange(n, dtype=np.int8) & 1 for n in (nt, nz, ny, nx)]
    return (ax[0][:, None, None, None] ^ ax[1][None, :, None, None] ^ ax[2][None, None, :, None]
            ^ ax[3][None, None, None, :]).astype(bool)


def test_128c3x144_fp32_offsets_beyond_32_bits():
    import torch
    import paper_1104_5432_b200 as pkg
    dims, prec, mode, seed, beta = DIMS, 32, "f32", 3, 6.0
    nx, ny, nz, nt = dims
    V = oracle.volume(dims)
    assert V * 16 > 2**32 and V * 4 * 16 > 2**32
    lat = pkg.Lattice(dims, prec)

    lat.init("cold", seed)
    assert lat.mean_plaquette() == 1.0 and lat.polyakov_loop() == 1.0

    lat.init("hot", seed)
    sigma = 1.0 / (2.0 * np.sqrt(6.0 * V))
    assert abs(lat.mean_plaquette()) < 5 * sigma          # 8.8e-5 at this size
    assert abs(lat.polyakov_loop()) < 5 * 0.5 / np.sqrt(V / nt)

    obs = torch.zeros(2, dtype=torch.float64, device="cuda")
    lat.sweep_measure(beta, 0, obs, 0)                    # the call bench.py times
    P_fused, L_fused = obs.cpu().numpy()
    assert abs(P_fused - lat.mean_plaquette()) < 2e-7
    assert abs(L_fused - lat.polyakov_loop()) < 1e-15
    assert 0.2 < P_fused < 0.95

    before = lat.get_links()
    # the whole Polyakov loop against the oracle: every U_3 link of the lattice enters it once
    assert abs(L_fused - oracle.polyakov_loop(dims, before, mode)) < 1e-6
    # set/get round trip through the canonical staging buffer, bit for bit
    lat.set_links(before)
    after = lat.get_links()
    assert np.array_equal(after.reshape(-1)[-2**20:], before.reshape(-1)[-2**20:])
    assert np.array_equal(after[:: 4099], before[:: 4099])

    odd = _parity_mask(dims)
    rng = np.random.default_rng(11)
    edge = np.array([0, V - 1, nx - 1, V - nx, V - nx * ny, V - nx * ny * nz, nx * ny * nz - 1], dtype=np.int64)
    flips = small = sampled = 0
    for mu, p in ((0, 1), (3, 0)):
        lat.substep(beta, 1, mu, p)
        lat.get_links(after)
        cand = np.concatenate([rng.integers(0, V, size=900), edge, V - 1 - np.arange(2 * nx), np.arange(2 * nx)])
        par = (cand % nx + cand // nx % ny + cand // (nx * ny) % nz + cand // (nx * ny * nz)) % 2
        cand = np.unique(cand[par == p])
        assert len(cand) > 500 and cand.max() * 16 > 2**32
        for s in cand:
            u, tr, mg, k, dl = oracle.heatbath_link(dims, before, beta, seed, 1, int(s), mu, mode, return_k=True, return_delta=True)
            d = np.abs(after[s, mu].astype(np.float64) - u.astype(np.float64)).max()
            sampled += 1
            if d > 1e-5:
                why = sampled_link_excused(d, mg, k, dl, beta, prec)
                assert why, (s, mu, d, mg, k)
                flips += why == "flip"
                small += why == "conditioned"
        a6, b6 = after.reshape(nt, nz, ny, nx, 4, 4), before.reshape(nt, nz, ny, nx, 4, 4)
        for nu in range(4):                               # one time slice at a time: bounded temporaries
            for t in range(nt):
                a, b = a6[t, :, :, :, nu], b6[t, :, :, :, nu]
                if nu != mu:
                    assert np.array_equal(a, b), (nu, t)
                    continue
                upd = odd[t] if p == 1 else ~odd[t]
                assert np.array_equal(a[~upd], b[~upd]), (nu, t)
                new = a[upd].astype(np.float64)
                assert np.abs((new**2).sum(-1) - 1).max() < 5e-7
                assert (np.abs(new - b[upd]).max(-1) > 0).mean() > 0.999
        lat.set_links(before)
    assert flips <= pp.flip_budget(sampled, prec) and small <= pp.conditioned_budget(sampled, prec)
    lat.close()


def test_2pow30_sites_fp32_properties():
    """256 x 256 x 128 x 128 = 2^30 sites (64 GiB of fp32 links): the largest class of lattice the handle
    accepts (V < 2^32; a single lattice indexes each of its 8 arrays with 32 bits). The canonical
    staging buffer of get/set_links would double the footprint, so this case checks what needs no copy:
    closed forms of the CUDA path itself and the agreement of its two plaquette routes."""
    import torch
    import paper_1104_5432_b200 as pkg
    dims = (256, 256, 128, 128)
    V = oracle.volume(dims)
    assert V == 2**30
    lat = pkg.Lattice(dims, 32)
    lat.init("cold", 1)
    assert lat.mean_plaquette() == 1.0 and lat.polyakov_loop() == 1.0
    lat.init("hot", 1)
    sigma = 1.0 / (2.0 * np.sqrt(6.0 * V))
    assert abs(lat.mean_plaquette()) < 5 * sigma
    obs = torch.zeros(4, dtype=torch.float64, device="cuda")
    lat.sweep_measure(6.0, 0, obs, 0)
    lat.sweep_measure(6.0, 1, obs, 1)
    P, L = obs.cpu().numpy()[2:4]
    assert abs(P - lat.mean_plaquette()) < 2e-7 and abs(L - lat.polyakov_loop()) < 1e-15
    assert 0.5 < P < 0.95          # two sweeps at beta = 6 from a hot start
    lat.close()
