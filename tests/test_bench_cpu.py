"""bench.py host logic that needs no GPU: the reference arm (the oracle timed on the host
cores) alone and under a 2-rank launch (rank 0 prints one JSON line, the other rank exits 0),
and a 2-rank gloo check of the max-over-ranks reduction the GPU arm uses for its timing."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _json_lines(out):
    return [json.loads(l) for l in out.splitlines() if l.startswith("{")]


def test_reference_arm_prints_the_contract_line():
    r = subprocess.run([sys.executable, "bench.py", "--impl", "reference", "--steps", "2", "--warmup", "1",
                        "--workload", "C1_8^4", "--precision", "64"], cwd=ROOT, capture_output=True, text=True,
                       timeout=300)
    assert r.returncode == 0, r.stderr
    (line,) = _json_lines(r.stdout)
    assert line["impl"] == "reference" and line["metric"] == "su2_heatbath_link_updates_per_s"
    assert line["unit"] == "link updates/s" and line["higher_is_better"] is True
    assert line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert line["e2e"]["value"] == line["value"] and line["steps"] == 2


def test_reference_arm_under_two_ranks_only_rank0_works():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29533", "bench.py", "--impl", "reference",
                        "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "C1_8^4", "--precision", "32"],
                       cwd=ROOT, capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1 and lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2


_WORKER = r"""
import os, sys, torch, torch.distributed as dist
dist.init_process_group("gloo")
rank = dist.get_rank()
# replicas only: each rank times its own lattice; the job's time is the max over ranks
t = torch.tensor([10.0 + 5.0 * rank], dtype=torch.float64)
dist.all_reduce(t, op=dist.ReduceOp.MAX)
dist.barrier()
if rank == 0:
    print("MAX", float(t.item()), dist.get_world_size())
dist.destroy_process_group()
"""


def test_max_over_ranks_reduction_gloo_world_size_2(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER)
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29534", str(w)], capture_output=True,
                       text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    assert "MAX 15.0 2" in r.stdout


def test_roofline_point_record():
    """bench.py's per-point roofline record (no GPU): algorithmic bytes = (V/2) x 8 quaternions, the L2 denominator
    for the lattice that fits L2 and the HBM copy peak otherwise, burst and sustained fractions side by side."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_1104_5432_b200 import workloads
    r = {"sweep_ms": 8 * 0.190, "ms_total": 20 * 1.57, "ms_per_step": 1.57, "t_wall": (0.0, 0.0),
         "sustained": {"sweep_ms": 8 * 0.220, "ms_total": 1100.0, "steps": 600, "ms_per_step": 1.83, "t_wall": (0.0, 0.0)}}
    traffic = {"C5_64^4_fp32": (1.079e9, "some capture")}
    pt = bench.roofline_point(workloads.BY_NAME["C5_64^4"], 32, r, 6540.0, "measured", 10900.0, traffic, None)
    assert pt["bound"] == "hbm" and pt["peak"] == 6540.0 and pt["unit"] == "GB/s"
    assert pt["algorithmic_bytes_per_launch"] == (64**4 // 2) * 128 == 1073741824
    assert abs(pt["achieved"] - 1073741824 / 190e-6 / 1e9) < 1e-6 and abs(pt["frac"] - pt["achieved"] / 6540.0) < 1e-12
    assert abs(pt["frac_sustained"] - 1073741824 / 220e-6 / 1e9 / 6540.0) < 1e-12 and pt["frac_sustained"] < pt["frac"]
    assert pt["traffic"] == 1.079e9 and "not measured in this run" in pt["traffic_kind"] and pt["steps"] == 20
    # the 64 MiB lattice is quoted against the measured L2 bandwidth, its HBM fraction kept beside it
    r32 = dict(r, sweep_ms=8 * 0.0132)
    r32["sustained"] = dict(r["sustained"], sweep_ms=8 * 0.0131)
    pt = bench.roofline_point(workloads.BY_NAME["C3_32^4"], 32, r32, 6540.0, "measured", 10900.0, {}, None)
    assert pt["bound"] == "l2" and pt["peak"] == 10900.0 and pt["traffic"] is None
    assert abs(pt["frac"] * 10900.0 - pt["frac_of_hbm_peak"] * 6540.0) < 1e-6
    # ... its fp64 twin (128 MiB) and a run without the probe against HBM
    assert bench.roofline_point(workloads.BY_NAME["C3_32^4"], 64, r32, 6540.0, "m", 10900.0, {}, None)["bound"] == "hbm"
    assert bench.roofline_point(workloads.BY_NAME["C3_32^4"], 32, r32, 6540.0, "m", None, {}, None)["bound"] == "hbm"
    # the committed citation file parses
    t = bench.load_traffic()
    assert set(t) >= {"C5_64^4_fp32", "C5_64^4_fp64", "C3_32^4_fp32", "C3_32^4_fp64"}
    assert 0.99 < t["C5_64^4_fp32"][0] / 1073741824 < 1.05
