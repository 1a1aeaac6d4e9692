"""Sweep-only timing of the four points of the metric (fp32/fp64 at 32^4 and 64^4) for the library as built:
the tool behind the tuning tables of profiles/ (tile shape, resident CTAs, walk length are compile-time
knobs of csrc/, set through SU2HB_NVCC_EXTRA, e.g.

    SU2HB_NVCC_EXTRA="-DHB_T0=3 -DHB_T1=2 -DHB_T2=1 -DHB_T3=1" python -m paper_1104_5432_b200.build --force
    python -m paper_1104_5432_b200.tune            # one JSON line: ms per sweep, fraction of the HBM copy peak
    python -m paper_1104_5432_b200.tune --one      # two sweeps + one su2_measure per point, no timing (for ncu)

Burst = 40 (64^4) / 300 (32^4) sweeps after 2 s of idle; sustained = the second half of a further 1.2 s of
continuous sweeps. A `links` signature (sha256 of small lattices after three sweeps) shows at a glance that a
build computes the same links as another. bench.py is the measurement of record; this is the quick A/B."""
import argparse
import hashlib
import json
import os
import time

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--one", action="store_true", help="two sweeps per point, no timing (profiling target)")
    ap.add_argument("--lib", default=None, help="path of another build of libsu2hb.so to time instead")
    ap.add_argument("--beta", type=float, default=6.0)
    args = ap.parse_args()
    import torch

    import paper_1104_5432_b200 as pkg
    if args.lib:
        pkg.LIB_PATH = os.path.abspath(args.lib)
    pkg.lib()
    points = (("64_f32", (64,) * 4, 32), ("64_f64", (64,) * 4, 64), ("32_f32", (32,) * 4, 32), ("32_f64", (32,) * 4, 64))
    if args.one:
        for _, dims, prec in points:
            lat = pkg.Lattice(dims, prec)
            lat.init("hot", 1)
            lat.sweep(args.beta, 0)
            lat.sweep(args.beta, 1)
            lat.measure()  # the standalone plaquette and Polyakov kernels
            lat.close()
        return 0
    peak = 6539.9
    path = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
    if os.path.exists(path):
        peak = float(json.load(open(path))["hbm_gbs"])
    res = {"lib": pkg.LIB_PATH, "hbm_gbs": peak}
    sig = hashlib.sha256()
    for prec in (32, 64):
        for dims in ((32, 16, 8, 8), (16, 8, 8, 4), (64, 8, 4, 4)):
            lat = pkg.Lattice(dims, prec)
            lat.init("hot", 3)
            for i in range(3):
                lat.sweep(2.4, i)
            sig.update(lat.get_links().tobytes())
            lat.close()
    res["links"] = sig.hexdigest()[:16]
    ev = lambda: torch.cuda.Event(enable_timing=True)
    for name, dims, prec in points:
        lat = pkg.Lattice(dims, prec)
        lat.init("hot", 1)
        n = 40 if dims[0] == 64 else 300
        for i in range(5):
            lat.sweep(args.beta, i)
        lat.synchronize()
        time.sleep(2.0)
        for i in range(3):
            lat.sweep(args.beta, 10 + i)
        torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record()
        for i in range(n):
            lat.sweep(args.beta, 20 + i)
        b.record()
        torch.cuda.synchronize()
        ms = a.elapsed_time(b) / n
        m = int(1200 / ms) // 2
        for i in range(m):
            lat.sweep(args.beta, 1000 + i)
        a2, b2 = ev(), ev()
        a2.record()
        for i in range(m):
            lat.sweep(args.beta, 1000 + m + i)
        b2.record()
        torch.cuda.synchronize()
        ms2 = a2.elapsed_time(b2) / m
        bytes_per_sweep = 4 * int(np.prod(dims)) * (128 if prec == 32 else 256)
        res[name] = {"ms_sweep": round(ms, 5), "frac": round(bytes_per_sweep / (ms * 1e-3) / (peak * 1e9), 4),
                     "ms_sweep_sustained": round(ms2, 5),
                     "frac_sustained": round(bytes_per_sweep / (ms2 * 1e-3) / (peak * 1e9), 4)}
        lat.synchronize()
        lat.close()
        torch.cuda.empty_cache()
    print(json.dumps(res), flush=True)
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
