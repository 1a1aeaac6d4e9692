"""Host check of the CUDA path's own fp64 elementary functions (csrc/su2_math64.cuh:
table log of a uniform, cos^2 / sincos of 2 pi u from the Philox word, rsqrt by one cubic
iteration) against the C library in long double. The functions are __host__ __device__;
the harness csrc/su2_math64_check.cu is compiled for the host by nvcc. No oracle code."""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "..", "paper_1104_5432_b200", "csrc")


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if c and os.path.exists(c):
            return c
    return None


@pytest.mark.skipif(_nvcc() is None, reason="nvcc not available")
def test_math64_against_libm(tmp_path):
    exe = str(tmp_path / "m64check")
    subprocess.run([_nvcc(), "-O2", "-std=c++17", "-o", exe, os.path.join(CSRC, "su2_math64_check.cu")],
                   check=True, capture_output=True)
    out = subprocess.run([exe, "3000000"], check=True, capture_output=True, text=True).stdout.split()
    r = dict(zip(out[0::2], map(float, out[1::2])))
    assert r["log_rel"] < 5e-16        # relative, including u -> 1 (ln u ~ -1e-10)
    assert r["cos2_abs"] < 5e-16
    assert r["sincos_abs"] < 3e-16
    assert r["rsqrt_rel"] < 3e-16
    assert r["sqrt0_rel"] < 3e-16      # m64::sqrt0_n itself (the function M<double>::sqrt0 calls)
    assert r["sqrt0_zero"] == 0.0      # exactly 0 at 0, no NaN
    assert 0.0 <= r["sqrt0_denormal"] < 1e-150
    assert abs(r["sqrt_tiny"] - 1e-150) < 1e-165


def test_log_table_is_what_its_generator_writes(tmp_path):
    """su2_log_table.inc is generated; the committed file must equal a fresh run."""
    import importlib.util
    spec = importlib.util.spec_from_file_location("gen_log_table", os.path.join(CSRC, "gen_log_table.py"))
    gen = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(gen)
    committed = open(os.path.join(CSRC, "su2_log_table.inc")).read()
    gen.HERE = str(tmp_path)
    gen.main()
    assert open(tmp_path / "su2_log_table.inc").read() == committed
