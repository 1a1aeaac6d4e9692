"""su2_mean_plaquette_noalloc (-m gpu): the entry point that allocates nothing - its per-CTA partial sums live in a
file-scope static __device__ array of the library instead of a handle's cudaMalloc'd scratch - against the existing
path (su2_mean_plaquette on a handle), on two calls in a row. Same kernels and the same fixed reduction order, so the
results agree to the bit; the assertion uses the tolerance the other plaquette tests use (1e-14 fp64 / 2e-7 fp32).
Collected last on purpose (file name): the suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {64: 1e-14, 32: 2e-7}


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    import paper_1104_5432_b200 as p
    from paper_1104_5432_b200 import build
    build.build()  # no-op unless a source is newer than the library
    p.lib()
    return p


# tiled launch with the first tile shape, with the second, the linear launch (ragged), minimal
@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims", [(32, 8, 8, 4), (16, 8, 8, 4), (6, 4, 10, 2), (2, 2, 2, 2)])
def test_noalloc_plaquette_equals_handle_path_on_two_calls_in_a_row(pkg, dims, prec):
    import torch
    lat = pkg.Lattice(dims, prec)
    lat.init("hot", 17)
    out = torch.full((2,), -7.0, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    got, want = [], []
    for call in range(2):  # two calls in a row share the static scratch; the configuration changes in between
        lat.sweep(2.4, call)
        pkg.su2_mean_plaquette_noalloc(pkg.su2_device_links(lat.h), *dims, prec, out.data_ptr() + 8 * call, stream)
        torch.cuda.synchronize()
        got.append(float(out[call].item()))
        want.append(lat.mean_plaquette())  # the existing path: handle-owned scratch
    for g, w in zip(got, want):
        assert abs(g - w) <= TOL[prec], (g, w)
    assert got == want            # same kernels, same reduction order: the same bits
    assert got[0] != got[1]       # the second call did not return the first call's stale partials
    # and once more on the unchanged configuration: the scratch keeps the last call's contents, the result does not care
    pkg.su2_mean_plaquette_noalloc(pkg.su2_device_links(lat.h), *dims, prec, out.data_ptr(), stream)
    torch.cuda.synchronize()
    assert float(out[0].item()) == want[1]
    lat.close()


def test_noalloc_plaquette_at_32c4_after_a_smaller_call(pkg):
    """A large call after a small one: the stale tail of the shared array belongs to nobody's sum."""
    import torch
    small, big = pkg.Lattice((16, 8, 8, 4), 32), pkg.Lattice((32, 32, 32, 32), 32)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    for lat in (big, small, big):
        lat.init("hot", 3)
        lat.sweep(6.0, 0)
        pkg.su2_mean_plaquette_noalloc(pkg.su2_device_links(lat.h), *lat.dims, 32, out.data_ptr())
        torch.cuda.synchronize()
        assert abs(float(out[0].item()) - lat.mean_plaquette()) <= TOL[32]
    small.close()
    big.close()


def test_noalloc_rejects_sizes_beyond_its_static_scratch_and_bad_arguments(pkg):
    import torch
    L = pkg.lib()
    buf = torch.zeros(1024, dtype=torch.float64, device="cuda")
    out = torch.full((1,), 5.0, dtype=torch.float64, device="cuda")
    ptr, optr = C.c_void_p(buf.data_ptr()), C.c_void_p(out.data_ptr())
    # 128 x 64^3 = 2^25 sites is the limit; 128^2 x 64^2 = 2^26 is beyond it: refused before anything is launched
    assert pkg.SU2_NOALLOC_MAX_SITES == 2 ** 25
    rc = L.su2_mean_plaquette_noalloc(ptr, 128, 128, 64, 64, 32, None, optr)
    assert rc == pkg.SU2_ETOOBIG
    assert b"SU2_NOALLOC_MAX_SITES" in L.su2_strerror(rc)
    with pytest.raises(pkg.SU2Error) as e:
        pkg.su2_mean_plaquette_noalloc(buf.data_ptr(), 128, 128, 64, 64, 32, out.data_ptr())
    assert e.value.code == pkg.SU2_ETOOBIG
    for args in ((None, 4, 4, 4, 4, 32, None, optr), (ptr, 4, 4, 4, 4, 32, None, None), (ptr, 4, 3, 4, 4, 32, None, optr),
                 (ptr, 4, 4, 4, 4, 16, None, optr), (C.c_void_p(buf.data_ptr() + 8), 4, 4, 4, 4, 32, None, optr)):
        assert L.su2_mean_plaquette_noalloc(*args) == pkg.SU2_EARG
    torch.cuda.synchronize()
    assert float(out.item()) == 5.0  # no rejected call wrote anything
