"""Pins of the oracle's building blocks against things other than itself:
Philox (published known-answer vectors + ATen's host engine), the uniform
conversion rules, the quaternion algebra (2x2 complex matrices), the hot start
(closed-form moments of the Haar measure). DESIGN.md §3 [R1][R5][R9]."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest
from scipy import stats

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


def _kat():
    rows = []
    with open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(t, 16) for t in line.split()]
            rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answers():
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, want in rows:
        assert list(oracle.philox4x32_10(ctr, key)) == want


@pytest.fixture(scope="session")
def aten_philox(tmp_path_factory):
    torch = pytest.importorskip("torch")
    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    so = str(tmp_path_factory.mktemp("aten") / "aten_philox.so")
    r = subprocess.run(["g++", "-O1", "-std=c++17", "-fPIC", "-shared", f"-I{inc}",
                        os.path.join(HERE, "helpers", "aten_philox.cpp"), "-o", so], capture_output=True, text=True)
    if r.returncode != 0:
        pytest.skip("ATen Philox header did not compile here: " + r.stderr[-300:])
    lib = C.CDLL(so)
    lib.aten_philox4x32_10.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p]
    lib.aten_philox4x32_10.restype = None
    return lib


def test_philox_matches_aten_host_engine(aten_philox):
    """3000 random (counter, key) pairs against at::Philox4_32 (library routine)."""
    rng = np.random.default_rng(7)
    words = rng.integers(0, 2**32, size=(3000, 6), dtype=np.uint64)
    out = np.zeros(4, dtype=np.uint32)
    for c0, c1, c2, c3, k0, k1 in words:
        aten_philox.aten_philox4x32_10(int(k0 | (k1 << np.uint64(32))), int(c2 | (c3 << np.uint64(32))),
                                       int(c0 | (c1 << np.uint64(32))), out.ctypes.data)
        mine = oracle.philox4x32_10([c0, c1, c2, c3], [k0, k1])
        assert (mine == out).all()


def test_uniform_rules_exact_and_open_interval():
    edge = [0, 1, 255, 256, 511, 512, 2**31 - 1, 2**31, 2**32 - 512, 2**32 - 2, 2**32 - 1]
    rng = np.random.default_rng(3)
    words = edge + [int(w) for w in rng.integers(0, 2**32, size=2000, dtype=np.uint64)]
    for w in words:
        u64 = oracle.uniform(w, "f64")
        u32 = oracle.uniform(w, "f32")
        u32x = oracle.uniform(w, "f32x")
        # exact rational values of the written rules (python ints/fractions are exact)
        assert u64 == (2 * w + 1) / 2**33
        assert u32 == (2 * (w >> 9) + 1) / 2**24
        assert u32x == u32
        assert np.float32(u32) == u32  # representable in fp32
        assert 0.0 < u64 < 1.0 and 0.0 < u32 < 1.0
        assert abs(u64 - u32) < 2.0**-23


def test_uniform_equidistribution():
    n = 40000
    u = np.array([oracle.uniform(int(oracle.philox4x32_10([i, 0, 0, 0], [5, 0])[j]), "f64")
                  for i in range(n // 4) for j in range(4)])
    assert stats.kstest(u, "uniform").pvalue > 1e-3
    assert abs(u.mean() - 0.5) < 5 * np.sqrt(1 / 12 / n)


SIGMA = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]]),
         np.array([[1, 0], [0, -1]], dtype=complex)]


def _mat(a):
    return a[0] * np.eye(2) + 1j * sum(a[i + 1] * SIGMA[i] for i in range(3))


def test_quaternion_product_is_su2_matrix_product():
    rng = np.random.default_rng(11)
    for _ in range(200):
        a, b = rng.standard_normal(4), rng.standard_normal(4)
        c = oracle.qmul(a, b)
        assert np.allclose(_mat(c), _mat(a) @ _mat(b), atol=1e-14, rtol=0)
        assert abs(np.linalg.norm(c) - np.linalg.norm(a) * np.linalg.norm(b)) < 1e-13
        # half trace is the scalar part; dagger is (a0, -a)
        assert abs(0.5 * np.trace(_mat(a)).real - a[0]) < 1e-15
        assert np.allclose(_mat(a * [1, -1, -1, -1]), _mat(a).conj().T, atol=1e-15)
    # non-commutativity pins the sign of the cross term: (i s1)(i s2) = -i s3
    assert np.allclose(oracle.qmul([0, 1, 0, 0], [0, 0, 1, 0]), [0, 0, 0, -1])


def test_quaternion_product_fp32_modes():
    rng = np.random.default_rng(12)
    for _ in range(50):
        a, b = rng.standard_normal(4), rng.standard_normal(4)
        ref = oracle.qmul(a, b)
        for m in ("f32", "f32x"):
            assert np.allclose(oracle.qmul(a, b, m), ref, atol=2e-6)


def test_cold_start_is_identity():
    L = oracle.init([4, 4, 4, 4], "cold", 9)
    assert (L[..., 0] == 1).all() and (L[..., 1:] == 0).all()


@pytest.mark.parametrize("mode", ["f64", "f32"])
def test_hot_start_is_haar(mode):
    dims = [8, 8, 8, 8]
    L = oracle.init(dims, "hot", 1, mode).astype(np.float64).reshape(-1, 4)
    n = len(L)
    tol = 1e-6 if mode == "f32" else 9e-16  # 4 ulp
    assert np.abs((L**2).sum(1) - 1).max() < tol
    # <a_i> = 0 (sd 1/2 per component), <a_i a_j> = delta_ij / 4
    assert np.abs(L.mean(0)).max() < 5 * 0.5 / np.sqrt(n)
    cov = L.T @ L / n
    assert np.abs(cov - np.eye(4) / 4).max() < 5 * 0.25 / np.sqrt(n)
    # each component has density (2/pi) sqrt(1-a^2): CDF = 1/2 + (a sqrt(1-a^2) + asin a)/pi
    cdf = lambda a: 0.5 + (a * np.sqrt(1 - a * a) + np.arcsin(a)) / np.pi
    for c in range(4):
        assert stats.kstest(L[:, c], cdf).pvalue > 1e-4
    # different seeds / directions decorrelated; same seed reproducible
    L2 = oracle.init(dims, "hot", 1, mode).astype(np.float64).reshape(-1, 4)
    assert (L2 == L).all()
    L3 = oracle.init(dims, "hot", 2, mode).astype(np.float64).reshape(-1, 4)
    assert abs((L * L3).sum(1).mean()) < 5 * 0.5 / np.sqrt(n)


def test_hot_start_plaquette_is_zero_within_error():
    """Each 1/2 Tr U_P of a Haar lattice is the a0 of a Haar element (variance 1/4),
    pairwise uncorrelated: |P| < 5 / (2 sqrt(6V))."""
    dims = [8, 8, 8, 8]
    for seed in (1, 2, 3):
        L = oracle.init(dims, "hot", seed)
        P = oracle.mean_plaquette(dims, L)
        assert abs(P) < 5 * 0.5 / np.sqrt(6 * 8**4)
