"""su2_bandwidth_probe (-m gpu): the library's own L2 / HBM bandwidth measurement, which
bench.py uses as the roofline denominator of the cache-resident point of the metric. Plausibility bounds only - the
numbers of record are in the bench line and profiles/r02a.md - plus the argument checks."""
import ctypes as C

import pytest

pytestmark = pytest.mark.gpu


def test_probe_orders_l2_above_hbm_and_rejects_bad_arguments():
    import torch
    assert torch.cuda.is_available()
    import paper_1104_5432_b200 as pkg
    pkg.lib()
    l2, us = pkg.su2_bandwidth_probe(64 << 20, 200, pkg.SU2_PROBE_READ)
    hbm, _ = pkg.su2_bandwidth_probe(2 << 30, 10, pkg.SU2_PROBE_READ)
    cpy, _ = pkg.su2_bandwidth_probe(2 << 30, 10, pkg.SU2_PROBE_COPY)
    # B200: ~10.9 TB/s L2-resident read, ~7.1 TB/s HBM read, ~6.0 TB/s HBM copy (profiles/r02a.md); wide windows
    assert 8000 < l2 < 16000, l2
    assert 4500 < hbm < 8500, hbm
    assert 4000 < cpy < 8000, cpy
    assert l2 > 1.2 * hbm and abs(us - (64 << 20) / l2 / 1e3) < 0.01 * us
    L = pkg.lib()
    g, u = C.c_double(), C.c_double()
    for args in ((1000, 10, 0), (64 << 20, 0, 0), (64 << 20, 10, 2), ((64 << 20) + 8, 10, 0)):
        assert L.su2_bandwidth_probe(args[0], args[1], args[2], None, C.byref(g), C.byref(u)) == pkg.SU2_EARG
    assert L.su2_bandwidth_probe(64 << 20, 10, 0, None, None, None) == pkg.SU2_EARG
