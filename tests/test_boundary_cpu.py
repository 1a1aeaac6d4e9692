"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports
every symbol include/su2_heatbath.h declares; argument validation that needs no
GPU; the product path never imports the oracle."""
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    from paper_1104_5432_b200 import build
    return build.build()


def _declared():
    src = open(os.path.join(ROOT, "include", "su2_heatbath.h")).read()
    return sorted(set(re.findall(r"SU2_API[^;(]*?\b(su2_\w+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for required in ("su2_lattice_create", "su2_init", "su2_heatbath_sweep", "su2_mean_plaquette",
                     "su2_polyakov_loop"):
        assert required in names


def test_library_exports_every_declared_symbol(built):
    out = subprocess.run(["nm", "-D", "--defined-only", built], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r" T (su2_\w+)", out))
    assert set(_declared()) <= exported
    import paper_1104_5432_b200 as pkg
    assert set(pkg.EXPORTS) == set(_declared())
    pkg.lib()  # loads and binds every symbol without touching a GPU


def test_sass_is_sm100a(built):
    out = subprocess.run(["cuobjdump", "-lelf", built], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_argument_validation_without_gpu(built):
    import ctypes as C
    import paper_1104_5432_b200 as pkg
    L = pkg.lib()
    assert L.su2_lattice_bytes(8, 8, 8, 8, 64) == 8**4 * 4 * 32
    assert L.su2_lattice_bytes(8, 8, 8, 8, 32) == 8**4 * 4 * 16
    assert L.su2_lattice_bytes(7, 8, 8, 8, 64) == 0  # odd extent
    assert L.su2_lattice_bytes(8, 8, 8, 0, 64) == 0
    assert L.su2_lattice_bytes(8, 8, 8, 8, 16) == 0
    assert L.su2_lattice_bytes(512, 512, 512, 32, 32) == 0  # V = 2^32
    h = C.c_void_p()
    assert L.su2_lattice_create(7, 8, 8, 8, 64, C.byref(h)) == pkg.SU2_EARG and not h.value
    assert L.su2_lattice_create(8, 8, 8, 8, 64, None) == pkg.SU2_EARG
    assert L.su2_lattice_destroy(None) == pkg.SU2_OK
    # batches: replica count, 32-bit link index over the whole batch, replica in the grid
    assert L.su2_lattice_create_batch(8, 8, 8, 8, 64, 0, C.byref(h)) == pkg.SU2_EARG and not h.value
    assert L.su2_lattice_create_batch(8, 8, 8, 8, 64, 70000, C.byref(h)) == pkg.SU2_EARG
    assert L.su2_lattice_create_batch(64, 64, 64, 64, 32, 64, C.byref(h)) == pkg.SU2_EARG  # 64 * 4V = 2^32
    assert L.su2_replicas(None) == 0
    assert L.su2_select_replica(None, 0) == pkg.SU2_EARG
    assert L.su2_batch_init(None, 0, None) == pkg.SU2_EARG
    assert L.su2_batch_sweep_measure(None, None, 0, None, 0) == pkg.SU2_EARG
    assert L.su2_set_draw(None, 0) == pkg.SU2_EARG
    assert L.su2_init(None, 0, 1) == pkg.SU2_EARG
    assert L.su2_heatbath_sweep(None, 2.3, 0) == pkg.SU2_EARG
    assert L.su2_strerror(pkg.SU2_ESTATE).decode().startswith("bad state")


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1104_5432_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, re.M), f
                assert "liborc" not in text and "su2_oracle" not in text, f
    # and the oracle does not import the product
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_1104_5432_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "paper_1104_5432_b200/", "")


def test_no_gpu_means_loud_failure(built):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_1104_5432_b200 as pkg
    with pytest.raises(RuntimeError):
        pkg.Lattice((8, 8, 8, 8), 64)
