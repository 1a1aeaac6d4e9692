#!/usr/bin/env python
"""bench.py — SU(2) heat-bath throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload C5_64^4|C3_32^4|...] [--precision 32|64] [--headline-only]

A "step" is one pass of the whole hot path over one lattice, one call of
su2_heatbath_sweep_measure: one heat-bath sweep (8 checkerboard sub-steps), the mean
plaquette of the new configuration (accumulated inside three of the sub-steps,
DESIGN.md 6.5) and its Polyakov loop (the paper's loop: "100 iterations of the heat
bath method and the calculation of the mean average plaquette at each iteration",
PAPER.md:46).
The random initialisation (row 1) runs once before the warm-up and is reported
separately as `init_ms`. value = link updates/s = 4V * steps / time.

Headline workload (N=1): BASELINE.json configs[4], 64^4 at beta = 6.0 from a cold
start in fp32 — the HBM-bound point of the metric ("link updates/s (fp32/fp64) at
32^4 and 64^4; % of HBM roofline"); the other three points of the metric (64^4
fp64, 32^4 fp32/fp64) are timed the same way and reported under "workloads".
The path does not shard (north_star: no multi-GPU path): with --gpus N every rank
runs an independent replica (different seed), no collective on the data path.

--impl reference times the CPU oracle as it stands on the host cores.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "su2_heatbath_link_updates_per_s"
UNIT = "link updates/s"
COOL_DOWN_S = 2.0  # idle time before each workload (outside every timed region)
BYTES_PER_UPDATE = {32: 128, 64: 256}  # 8 quaternions per link update


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            with open(path) as f:
                return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region: NVML in a
    background thread every 10 ms (nvidia-smi -lms as fallback if pynvml is unusable)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index = index
        self.rows = []  # (time, sm_mhz, sm_max_mhz, power_w, [reasons])
        self.proc = None
        self.stop_flag = False
        self.thread = None
        self.source = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            # NVML indexes physical devices: honour CUDA_VISIBLE_DEVICES if it is a list of indices
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = self.index
            if vis:
                try:
                    idx = int(vis.split(",")[self.index])
                except Exception:
                    idx = self.index
            h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            smax = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            bits = [(pynvml.nvmlClocksEventReasonHwSlowdown, "hw_slowdown"),
                    (pynvml.nvmlClocksEventReasonHwThermalSlowdown, "hw_thermal_slowdown"),
                    (pynvml.nvmlClocksEventReasonSwThermalSlowdown, "sw_thermal_slowdown"),
                    (pynvml.nvmlClocksEventReasonSwPowerCap, "sw_power_cap")]

            def loop():
                while not self.stop_flag:
                    try:
                        mhz = float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                        mask = pynvml.nvmlDeviceGetCurrentClocksEventReasons(h)
                        pw = pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0
                        self.rows.append((time.time(), mhz, smax, pw, [n for b, n in bits if mask & b]))
                    except Exception:
                        pass
                    time.sleep(0.01)

            self.thread = threading.Thread(target=loop, daemon=True)
            self.thread.start()
            self.source = "nvml"
            return
        except Exception:
            pass
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
            self.source = "nvidia-smi"
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            f = [x.strip() for x in line.split(",")]
            try:
                self.rows.append((time.time(), float(f[0]), float(f[1]), float(f[2]),
                                  [n for n, v in zip(self.NAMES, f[3:7]) if v.lower().startswith("active")]))
            except Exception:
                continue

    def ready(self):
        return bool(self.rows)

    def mark(self):
        return time.time()

    def stop(self):
        self.stop_flag = True
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self, t0, t1):
        rows = [r for r in self.rows if t0 <= r[0] <= t1]
        if not rows:  # region shorter than one sampling period: nearest samples around it
            rows = [r for r in self.rows if t0 - 0.1 <= r[0] <= t1 + 0.1]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "source": self.source}
        reasons = sorted({n for r in rows for n in r[4]})
        return {"sm_mhz": float(np.median([r[1] for r in rows])), "sm_max_mhz": max(r[2] for r in rows),
                "power_w": float(np.median([r[3] for r in rows])), "reasons": reasons, "samples": len(rows),
                "source": self.source}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# ------------------------------------------------------------------------------- ours
def _sweep_leg(lat, torch, beta, obs, idx0, n, every=1, dist=None, sampler=None):
    """`n` consecutive su2_heatbath_sweep_measure calls, timed on the device as a whole, with a CUDA-event
    pair around the 8 sub-step kernels of every `every`-th step (the second event of a pair is recorded by
    the library between the 8th sub-step and the reduction kernel): the heat-bath kernel's average launch
    duration for the roofline comes from the SAME region as the step time."""
    ev = lambda: torch.cuda.Event(enable_timing=True)
    pairs = {k: (ev(), ev()) for k in range(0, n, every)}
    for a, b in pairs.values():  # materialise the CUDA events (torch creates them on first record)
        a.record()
        b.record()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    n0 = lat.launch_count
    t0 = sampler.mark() if sampler else 0.0
    start, stop = ev(), ev()
    start.record()
    for k in range(n):
        if k in pairs:
            pairs[k][0].record()
            lat.sweep_measure(beta, idx0 + k, obs, idx0 + k, pairs[k][1])
        else:
            lat.sweep_measure(beta, idx0 + k, obs, idx0 + k)
    stop.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t1 = sampler.mark() if sampler else 0.0
    lat.synchronize()  # surfaces device-side error flags
    return {"ms_total": start.elapsed_time(stop), "steps": n, "launches": int(lat.launch_count - n0),
            "sweep_ms": float(np.mean([a.elapsed_time(b) for a, b in pairs.values()])), "t_wall": (t0, t1)}


def time_workload(pkg, torch, w, prec, beta, steps, warmup, seed, sampler=None, dist=None, sustained_s=1.0):
    """Device-resident timing. Burst leg: EXACTLY `steps` steps after a cool-down and `warmup` untimed steps
    (the line's `value`). Sustained leg: a continuous run of the same steps, the first third untimed (the GPU
    reaches its power-capped state), then >= `sustained_s` seconds timed. Returns a dict of measurements."""
    time.sleep(COOL_DOWN_S)  # every workload starts from the same power state, whatever ran before it
    lat = pkg.Lattice(w.dims, prec)
    ev = lambda: torch.cuda.Event(enable_timing=True)

    e0, e1 = ev(), ev()
    torch.cuda.synchronize()
    e0.record()
    lat.init(w.start, seed)
    e1.record()
    torch.cuda.synchronize()
    init_ms = e0.elapsed_time(e1)

    obs = torch.zeros(2 * (steps + warmup), dtype=torch.float64, device=lat.device)
    for i in range(warmup):
        lat.sweep_measure(beta, i, obs, i)
    lat.synchronize()
    burst = _sweep_leg(lat, torch, beta, obs, warmup, steps, 1, dist, sampler)
    o = obs.cpu().numpy().reshape(-1, 2).copy()

    res = {"ms_total": burst["ms_total"], "ms_per_step": burst["ms_total"] / steps, "sweep_ms": burst["sweep_ms"],
           "init_ms": init_ms, "launches": burst["launches"], "plaquette_last": float(o[warmup + steps - 1, 0]),
           "polyakov_last": float(o[warmup + steps - 1, 1]), "t_wall": burst["t_wall"], "links": w.links}

    if sustained_s > 0:
        n_sus = max(steps, int(np.ceil(sustained_s * 1e3 / res["ms_per_step"] * 1.1)))
        n_pre = max(warmup, n_sus // 3)
        obs2 = torch.zeros(2 * (n_pre + n_sus), dtype=torch.float64, device=lat.device)
        base = warmup + steps
        for i in range(n_pre):  # untimed: continuous load until the power cap has settled
            lat.sweep_measure(beta, base + i, obs2, i)
        sus = _sweep_leg(lat, torch, beta, _Shifted(obs2, base), base + n_pre, n_sus, max(1, n_sus // 200), dist,
                         sampler)
        res["sustained"] = {"ms_total": sus["ms_total"], "steps": n_sus, "ms_per_step": sus["ms_total"] / n_sus,
                            "sweep_ms": sus["sweep_ms"], "t_wall": sus["t_wall"], "untimed_steps_before": n_pre}
        del obs2

    # extra (not the headline): the same `steps` steps as ONE su2_run call - the step captured as
    # a CUDA graph and replayed, no host work per step (matters on small lattices)
    time.sleep(COOL_DOWN_S)  # same power state as the burst leg started from
    lat.set_option("tail_overlap", 0)  # (the default is automatic; both settings are timed explicitly)
    lat.run(beta, 1 << 20, min(warmup, steps), obs)  # captures the graph
    torch.cuda.synchronize()
    s2, e2 = ev(), ev()
    s2.record()
    lat.run(beta, (1 << 20) + warmup, steps, obs)
    e2.record()
    torch.cuda.synchronize()
    lat.synchronize()
    res["ms_per_step_run"] = s2.elapsed_time(e2) / steps
    # ... and with the opt-in tail overlap (SU2_OPT_TAIL_OVERLAP): the Polyakov kernel of a step
    # beside the next step's first six sub-steps
    lat.set_option("tail_overlap", 1)
    time.sleep(COOL_DOWN_S)
    lat.run(beta, (1 << 21), 16, obs[:32] if obs.numel() >= 32 else torch.zeros(32, dtype=torch.float64, device=lat.device))
    torch.cuda.synchronize()
    s3, e3 = ev(), ev()
    s3.record()
    lat.run(beta, (1 << 21) + 16, steps, obs)
    e3.record()
    torch.cuda.synchronize()
    lat.synchronize()
    res["ms_per_step_run_tail_overlap"] = s3.elapsed_time(e3) / steps
    lat.close()
    del lat, obs
    torch.cuda.empty_cache()
    return res


class _Shifted:
    """A device tensor addressed with the sweep index minus `base` (su2_heatbath_sweep_measure takes the
    output slot and the sweep index separately; the sustained leg continues the chain's sweep indices)."""

    def __init__(self, t, base):
        self.t, self.base = t, base

    def data_ptr(self):
        return self.t.data_ptr() - 16 * self.base


def time_aux(pkg, torch, workloads):
    """Not part of the metric: the finite-temperature configs through su2_run (one call, CUDA graph
    replay) and the Polyakov-loop correlator (S8(f) NEXT-1) on BASELINE config 4, wall clock."""
    out = {}
    for name, prec, beta, n in (("C2_16^3x4", 32, 2.4, 200), ("C4_48^3x8", 64, 2.5, 100)):
        w = workloads.BY_NAME[name]
        lat = pkg.Lattice(w.dims, prec)
        lat.init(w.start, w.seed)
        obs = torch.zeros(2 * n, dtype=torch.float64, device=lat.device)
        lat.run(beta, 0, 10, obs)
        lat.synchronize()
        t0 = time.perf_counter()
        lat.run(beta, 10, n, obs)
        lat.synchronize()
        dt = time.perf_counter() - t0
        rec = {"su2_run_us_per_step": dt / n * 1e6, "value": w.links * n / dt, "unit": UNIT, "beta": beta,
               "precision": prec, "steps": n}
        if name.startswith("C4"):
            lat.polyakov_correlator(24)
            t0 = time.perf_counter()
            for _ in range(10):
                c = lat.polyakov_correlator(24)
            rec["correlator_r1_24_us_per_call"] = (time.perf_counter() - t0) / 10 * 1e6
            rec["correlator_r1"] = float(c[0])
        out[name] = rec
        lat.close()
    # replica batches (S8(f) NEXT-2): config 2's beta scan, R lattices stepped by the launches of one
    w = workloads.BY_NAME["C2_16^3x4"]
    for R in (5, 20):
        bat = pkg.Lattice(w.dims, 32, replicas=R)
        bat.batch_init(w.start, [w.seed + r for r in range(R)])
        betas = [2.2 + 0.1 * (r % 5) for r in range(R)]
        n = 200
        obs = torch.zeros(2 * R * n, dtype=torch.float64, device=bat.device)
        for i in range(10):
            bat.batch_sweep_measure(betas, i, obs, i)
        bat.synchronize()
        t0 = time.perf_counter()
        for i in range(n):
            bat.batch_sweep_measure(betas, 10 + i, obs, i)
        bat.synchronize()
        dt = time.perf_counter() - t0
        out[f"C2_16^3x4_batch{R}"] = {"us_per_round": dt / n * 1e6, "value": R * w.links * n / dt, "unit": UNIT,
                                      "replicas": R, "precision": 32, "rounds": n}
        # the same rounds as ONE su2_batch_run call (one round captured as a CUDA graph, replayed)
        bat.batch_run(betas, 1000, 10, obs)
        bat.synchronize()
        t0 = time.perf_counter()
        bat.batch_run(betas, 1010, n, obs)
        bat.synchronize()
        dt = time.perf_counter() - t0
        out[f"C2_16^3x4_batch{R}"].update({"batch_run_us_per_round": dt / n * 1e6, "batch_run_value": R * w.links * n / dt})
        bat.close()
    # ... and the paper's benchmark shape: four 32^4 lattices stepped by the launches of one (a 32^4 launch is 3.5 CTA
    # waves and latency-bound; four of them are 14 waves)
    w3 = workloads.BY_NAME["C3_32^4"]
    R, n = 4, 100
    bat = pkg.Lattice(w3.dims, 32, replicas=R)
    bat.batch_init(w3.start, [w3.seed + r for r in range(R)])
    obs = torch.zeros(2 * R * n, dtype=torch.float64, device=bat.device)
    for i in range(5):
        bat.batch_sweep_measure([6.0] * R, i, obs, i)
    bat.synchronize()
    time.sleep(2.0)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for i in range(n):
        bat.batch_sweep_measure([6.0] * R, 5 + i, obs, i)
    b.record()
    torch.cuda.synchronize()
    ms = a.elapsed_time(b) / n
    out["C3_32^4_fp32_batch4"] = {"ms_per_round": ms, "value": R * w3.links / ms * 1e3, "unit": UNIT, "replicas": R,
                                  "precision": 32, "rounds": n}
    bat.close()
    torch.cuda.empty_cache()
    # time slabs (S8(f) NEXT-4) with every slab on this ONE GPU: the slabs' kernels of a sub-step run one
    # after the other, so the sweep time is the sum over slabs - what the split costs in kernel time
    # (ALT kernels, peer stores, no launch overlap), not a multi-GPU number
    from paper_1104_5432_b200 import slabs
    w = workloads.BY_NAME["C5_64^4"]
    for prec in (32, 64):
        for n_slabs in (2, 4):
            ring = slabs.SlabRing(w.dims, prec, n_slabs)
            ring.init(w.start, w.seed)
            time.sleep(2.0)
            for k in range(3):
                ring.sweep(6.0, k)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            n = 20
            a.record()
            for k in range(n):
                ring.sweep(6.0, 3 + k)
            b.record()
            torch.cuda.synchronize()
            ms = a.elapsed_time(b) / n
            out[f"C5_64^4_fp{prec}_slabs{n_slabs}_on_one_gpu"] = {"ms_per_sweep": ms, "value": w.links / ms * 1e3,
                                                                 "unit": UNIT, "sweeps": n}
            ring.close()
            torch.cuda.empty_cache()
    # the paper's Fig. 1 benchmark over lattice sizes: random SU(2) initialisation, 100
    # heat-bath iterations at beta = 6.0 with the mean plaquette at each iteration, wall clock of the
    # whole job (su2_init + one su2_run call, which also takes the Polyakov loop at each iteration)
    fig1 = []
    for prec in (32, 64):
        for L in (8, 16, 24, 32, 48, 64, 96):
            lat = pkg.Lattice((L, L, L, L), prec)
            obs = torch.zeros(2 * 100, dtype=torch.float64, device=lat.device)
            lat.init("hot", 1)
            lat.run(6.0, 0, 3, obs)  # untimed: graph capture
            lat.synchronize()
            time.sleep(1.0)
            t0 = time.perf_counter()
            lat.init("hot", 1)
            lat.run(6.0, 0, 100, obs)
            lat.synchronize()
            dt = time.perf_counter() - t0
            fig1.append({"L": L, "precision": prec, "seconds": dt, "value": 4 * L**4 * 100 / dt, "unit": UNIT,
                         "plaquette_last": float(obs[198])})
            lat.close()
            torch.cuda.empty_cache()
    out["fig1_init_100_sweeps_plaquette_beta6"] = fig1
    return out


def time_e2e(pkg, torch, w, prec, beta, steps, warmup, seed):
    """Same step through the C-ABI with HOST buffers: every step copies the input
    configuration host->device (su2_set_links, pinned), runs sweep + plaquette +
    Polyakov, and reads the new configuration and the observables back
    (su2_get_links + su2_measure)."""
    lat = pkg.Lattice(w.dims, prec)
    nbytes = pkg.su2_lattice_bytes(*w.dims, prec)
    dt = np.float32 if prec == 32 else np.float64
    pinned = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    host = pinned.numpy().view(dt).reshape(w.volume, 4, 4)
    lat.init(w.start, seed)
    lat.get_links(host)
    obs = torch.zeros(2, dtype=torch.float64, device=lat.device)
    t = []
    for k in range(warmup + steps):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        lat.set_links(host)
        lat.sweep_measure(beta, k, obs, 0)
        lat.get_links(host)
        P, L = obs.cpu().numpy()
        torch.cuda.synchronize()
        t.append(time.perf_counter() - t0)
    lat.close()
    sec = float(np.mean(t[warmup:]))
    return {"value": w.links / sec, "unit": UNIT, "h2d_bytes_per_step": int(nbytes),
            "d2h_bytes_per_step": int(nbytes + 16), "ms_per_step": sec * 1e3, "steps": steps,
            "what": "su2_set_links(pinned host) + su2_heatbath_sweep_measure + su2_get_links(pinned host) + 16 B of observables"}


def cpu_fig1(fig1):
    """The CPU side of the paper's Fig. 1 job ("the serial code in one CPU core"), part of
    the cpu_baseline leg: the oracle on the same job at 32^4 in fp32 - random start, then heat-bath iterations with the
    plaquette after each - timed over 3 iterations and scaled to the 100 of the figure (the full job is ~2.5
    minutes of one core)."""
    import oracle
    dims, n_cpu = (32, 32, 32, 32), 3
    t0 = time.perf_counter()
    L = oracle.init(dims, "hot", 1, "f32")
    t_init = time.perf_counter() - t0
    t0 = time.perf_counter()
    P = 0.0
    for i in range(n_cpu):
        oracle.heatbath_sweep(dims, L, 6.0, 1, i, "f32")
        P = oracle.mean_plaquette(dims, L, "f32")
    t_iter = (time.perf_counter() - t0) / n_cpu
    gpu = next(f for f in fig1 if f["L"] == 32 and f["precision"] == 32)
    return {"seconds_scaled_to_100_iterations": t_init + 100 * t_iter, "seconds_per_iteration": t_iter,
            "init_seconds": t_init, "iterations_timed": n_cpu, "cores": 1, "kind": "oracle", "plaquette_after_3": P,
            "gpu_seconds_same_job": gpu["seconds"], "ratio": (t_init + 100 * t_iter) / gpu["seconds"],
            "note": "context only (the paper quotes > 200x for 2 GTX 480 over one i7-920 core, PAPER.md:95)"}


# ------------------------------------------------------------------------------- oracle
class OracleSlab:
    """The oracle as it stands (gcc -O2, serial, one host core) on a BOUNDED sample of the
    workload: the same lattice cut down to its first Nt' time slices (periodic), Nt' even,
    chosen so that one step costs about `seconds_per_step`. A step is the whole hot path:
    one heat-bath sweep + mean plaquette + Polyakov loop, continuing one chain."""

    def __init__(self, w, prec, beta, seed, seconds_per_step):
        import oracle
        self.oracle, self.w, self.beta, self.seed = oracle, w, beta, seed
        self.mode = "f32" if prec == 32 else "f64"
        nx, ny, nz, nt = w.dims
        # calibrate on the 2-slice slab
        self.dims = (nx, ny, nz, 2)
        self.links = oracle.init(self.dims, w.start, seed, self.mode)
        rate = self._step(0)[0]  # link updates/s
        want = seconds_per_step * rate / (4.0 * nx * ny * nz)
        nts = int(min(nt, max(2, 2 * round(want / 2.0))))
        if nts != 2:
            self.dims = (nx, ny, nz, nts)
            self.links = oracle.init(self.dims, w.start, seed, self.mode)
        self.k = 1

    def _step(self, k):
        o = self.oracle
        t0 = time.perf_counter()
        o.heatbath_sweep(self.dims, self.links, self.beta, self.seed, k, self.mode)
        P = o.mean_plaquette(self.dims, self.links, self.mode)
        L = o.polyakov_loop(self.dims, self.links, self.mode)
        sec = time.perf_counter() - t0
        n = 4 * int(np.prod(self.dims))
        return n / sec, sec, n, P, L

    def step(self):
        r = self._step(self.k)
        self.k += 1
        return r

    def describe(self, prec):
        return (f"1 oracle step (heat-bath sweep + mean plaquette + Polyakov loop) on the first {self.dims[3]} of "
                f"{self.w.dims[3]} time slices of the {self.w.name} lattice = {4 * int(np.prod(self.dims))} link "
                f"updates per step, fp{prec} oracle mode, gcc -O2, serial")


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    from paper_1104_5432_b200 import workloads
    w = workloads.BY_NAME[args.workload]
    prec = args.precision
    # the whole --steps K --warmup W run is sized to about two minutes of host time
    slab = OracleSlab(w, prec, args.beta, args.seed, args.ref_seconds / max(1, args.warmup + args.steps))
    vals, secs = [], []
    for k in range(args.warmup + args.steps):
        v, sec, n, P, L = slab.step()
        if k >= args.warmup:
            vals.append(v)
            secs.append(sec)
    value = float(np.sum([4 * np.prod(slab.dims)] * len(secs)) / np.sum(secs))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(secs)) * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if prec == 32 else "f64", "data": "synthetic",
        "config": {"workload": f"{w.name} beta={args.beta} start={w.start} (bounded sample)", "precision": prec},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": slab.describe(prec)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "plaquette_last": P, "polyakov_last": L,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------- one lattice over N GPUs
def run_slabs(args, torch, pkg, workloads, dist, rank, world, local):
    """--gpus N --split slabs: ONE lattice as N time slabs, one rank per GPU - the paper's second mode
    ("2 GPUs"). Each sub-step's kernel also stores the slab's edge slices
    into the neighbours' halos over NVLink (CUDA-IPC-mapped peer buffers, no pack/send/unpack), a 1-element
    NCCL all-reduce on the kernels' stream is the barrier between sub-steps. A step = sweep (plaquette
    fused) + plaquette sum over ranks + chained Polyakov loop. Total work is fixed: strong scaling.
    Off by default: north_star's metric is single-GPU and --gpus N runs replicas."""
    from paper_1104_5432_b200 import slabs
    w = workloads.BY_NAME[args.workload]
    prec = args.precision
    ds = slabs.DistributedSlab(w.dims, prec, f"cuda:{local}", barrier="stream")
    ds.init(w.start, args.seed)
    P = L = 0.0
    for i in range(args.warmup):
        ds.sweep(args.beta, i, fuse_plaquette=True)
        P, L = ds.mean_plaquette(fused=True), ds.polyakov_loop()
    dist.barrier()
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for k in range(args.steps):
        ds.sweep(args.beta, args.warmup + k, fuse_plaquette=True)
        P, L = ds.mean_plaquette(fused=True), ds.polyakov_loop()
    b.record()
    torch.cuda.synchronize()
    dist.barrier()
    t = torch.tensor([a.elapsed_time(b)], dtype=torch.float64, device="cuda")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    ds.close()
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": w.links * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32" if prec == 32 else "f64", "data": "synthetic",
            "config": {"workload": f"{w.name} beta={args.beta} start={w.start} seed={args.seed}", "precision": prec,
                       "parallelism": f"time slabs: one lattice split along t over {world} GPUs, halo links stored "
                                      "into peer memory by the sub-step kernel, NCCL stream barrier per sub-step",
                       "l2": "inputs larger than L2, no flush needed"},
            "gpu_launches": 8 * args.steps + 2 * args.steps, "plaquette_last": P, "polyakov_last": L,
            "roofline": None, "e2e": None,
            "note": "opt-in arm (--split slabs); the headline metric and its roofline are the single-GPU run"}))
    return 0


# ------------------------------------------------------------------------------- roofline
def load_traffic():
    """profiles/traffic.csv: key,bytes_per_launch,source - dram__bytes_read.sum + dram__bytes_write.sum per
    heat-bath launch from the committed `ncu --set full` captures (a citation, not a quantity of this run)"""
    out = {}
    prof = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(prof):
        with open(prof) as f:
            for row in f:
                k = row.strip().split(",")
                if len(k) >= 2 and not k[0].startswith("#"):
                    try:
                        out[k[0]] = (float(k[1]), k[2] if len(k) > 2 else "profiles/")
                    except ValueError:
                        pass
    return out


def roofline_point(w, prec, r, hbm_peak, hbm_src, l2_gbs, traffic, sampler):
    """Roofline of the dominant kernel (heat-bath sub-step) at one point of the metric. Algorithmic bytes per
    launch = (V/2 updates) x 8 quaternions; duration = mean time of the 8 sub-steps of a
    sweep / 8, CUDA events on the launching stream inside the timed region; burst (`frac`) and sustained
    (`frac_sustained`, >= 1 s of continuous steps) legs. A lattice that fits the 126 MB L2 is bound by the L2
    bandwidth of the box (measured by su2_bandwidth_probe in this run) and is quoted against it; its
    fraction of the HBM copy peak is kept beside it for comparison with the other points."""
    alg = (w.volume // 2) * BYTES_PER_UPDATE[prec]
    lattice_mib = w.links * 4 * prec // 8 >> 20
    resident = lattice_mib <= 100 and l2_gbs is not None
    peak = l2_gbs if resident else hbm_peak
    sub_us = r["sweep_ms"] * 1e3 / 8.0
    ach = alg / (sub_us * 1e-6) / 1e9
    key = f"{w.name}_fp{prec}"
    pt = {"bound": "l2" if resident else "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
          "traffic": traffic.get(key, (None, None))[0],
          "traffic_kind": "ncu --set full capture committed under profiles/ (not measured in this run): "
                          + str(traffic.get(key, (None, "none for this point"))[1]),
          "peak_source": ("measured in this run: su2_bandwidth_probe, 64 MiB read, L2-resident (lattice %d MiB)" % lattice_mib)
          if resident else hbm_src,
          "algorithmic_bytes_per_launch": alg, "avg_launch_us": sub_us,
          "frac_of_hbm_peak": ach / hbm_peak, "steps": int(round(r["ms_total"] / r["ms_per_step"])),
          "ms_per_step": r["ms_per_step"], "clocks": sampler.summary(*r["t_wall"]) if sampler else None}
    if "sustained" in r:
        su = r["sustained"]
        sus_us = su["sweep_ms"] * 1e3 / 8.0
        a2 = alg / (sus_us * 1e-6) / 1e9
        pt.update({"frac_sustained": a2 / peak, "achieved_sustained": a2, "avg_launch_us_sustained": sus_us,
                   "sustained_region_ms": su["ms_total"], "sustained_steps": su["steps"],
                   "sustained_ms_per_step": su["ms_per_step"], "frac_of_hbm_peak_sustained": a2 / hbm_peak,
                   "clocks_sustained": sampler.summary(*su["t_wall"]) if sampler else None})
    if l2_gbs is not None:
        pt["l2_read_gbs_measured"] = l2_gbs
    return pt


# ------------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5_64^4")
    ap.add_argument("--precision", type=int, default=32, choices=[32, 64])
    ap.add_argument("--beta", type=float, default=6.0)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--headline-only", action="store_true", help="skip the other metric points, e2e and cpu_baseline")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--ref-seconds", type=float, default=120.0, help="host time the whole reference run may take")
    ap.add_argument("--cpu-baseline-seconds", type=float, default=12.0)
    ap.add_argument("--sustained-seconds", type=float, default=1.0,
                    help="length of the sustained (power-capped) timed region per metric point; 0 = skip")
    ap.add_argument("--split", default="replicas", choices=["replicas", "slabs"],
                    help="--gpus N > 1: independent replicas (default, north_star) or ONE lattice as N time slabs")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.warmup < 3:
        args.warmup = 3  # timing rule: W >= 3

    import torch
    from paper_1104_5432_b200 import workloads
    import paper_1104_5432_b200 as pkg

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_1104_5432_b200 import build as lib_build
    lib_build.build()  # no-op unless a source is newer than the in-tree library
    pkg.lib()
    if world > 1 and args.split == "slabs":
        rc = run_slabs(args, torch, pkg, workloads, dist, rank, world, local)
        dist.destroy_process_group()
        return rc
    peak, peak_src = measured_peaks()
    w = workloads.BY_NAME[args.workload]
    prec = args.precision

    sampler = ClockSampler(local)
    sampler.start()
    t_wait = time.time()
    while not sampler.ready() and time.time() - t_wait < 5.0:  # nvidia-smi takes ~1 s to emit its first line
        time.sleep(0.05)
    sus_s = 0.0 if args.headline_only else args.sustained_seconds
    r = time_workload(pkg, torch, w, prec, args.beta, args.steps, args.warmup, args.seed + rank, sampler, dist, sus_s)
    clocks = sampler.summary(*r["t_wall"])

    ms = r["ms_total"]
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
        # every timed region is over: release the other ranks now (rank 0 alone goes on to the other metric points,
        # e2e and the CPU baseline - minutes during which they would sit in a collective)
        dist.barrier()
        dist.destroy_process_group()
        if rank != 0:
            sampler.stop()
            return 0
    value = world * w.links * args.steps / (ms * 1e-3)

    # L2 roofline denominator: read bandwidth of a 64 MiB buffer - the size of the
    # 32^4 fp32 lattice - once it is resident in the 126 MB L2; measured live by the library's probe kernel
    l2_gbs = None
    if rank == 0 and not args.headline_only:
        time.sleep(COOL_DOWN_S)
        l2_gbs, _ = pkg.su2_bandwidth_probe(64 << 20, 400, pkg.SU2_PROBE_READ)

    traffic = load_traffic()
    point = lambda name, p, rr: roofline_point(workloads.BY_NAME[name], p, rr, peak, peak_src, l2_gbs, traffic, sampler)
    head_key = f"{w.name}_fp{prec}"
    roofline = point(w.name, prec, r)
    roofline["kernel"] = "heatbath sub-step (one launch per (mu, parity), 8 per sweep)"
    roofline["points"] = {head_key: {k: v for k, v in roofline.items() if k != "kernel"}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32" if prec == 32 else "f64", "data": "synthetic",
        "config": {"workload": f"{w.name} beta={args.beta} start={w.start} seed={args.seed}",
                   "precision": prec, "step": "su2_heatbath_sweep_measure: 1 heat-bath sweep (8 sub-steps, plaquette fused into 3 of them) + Polyakov loop",
                   "l2": (("inputs larger than L2 (%d MiB lattice vs 126 MiB L2), no flush needed"
                           if (w.links * 4 * prec // 8 >> 20) > 126 else
                           "lattice %d MiB is L2-resident by nature of the workload; no flush between steps")
                          % (w.links * 4 * prec // 8 >> 20)),
                   "cool_down": f"{COOL_DOWN_S} s idle before each workload's warm-up (power state independent of the workload before)",
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": r["launches"], "roofline": roofline,
        "sweep_only": {"value": world * w.links / (r["sweep_ms"] * 1e-3), "unit": UNIT, "ms_per_sweep": r["sweep_ms"]},
        "init_ms": r["init_ms"], "plaquette_last": r["plaquette_last"], "polyakov_last": r["polyakov_last"],
        "su2_run": {"value": world * w.links / (r["ms_per_step_run"] * 1e-3), "unit": UNIT,
                    "ms_per_step": r["ms_per_step_run"],
                    "ms_per_step_tail_overlap": r["ms_per_step_run_tail_overlap"],
                    "what": "the same steps as one su2_run call (captured CUDA graph replayed), timed after the same cool-down; "
                            "tail_overlap = the same with SU2_OPT_TAIL_OVERLAP"},
    }

    if not args.headline_only and rank == 0:
        # the other three points of the metric (fp32/fp64 at 32^4 and 64^4), device-resident, same step, each
        # with its burst and sustained fraction inside `roofline.points`
        others = {}
        for name, p in (("C5_64^4", 32), ("C5_64^4", 64), ("C3_32^4", 32), ("C3_32^4", 64)):
            if name == w.name and p == prec:
                continue
            ww = workloads.BY_NAME[name]
            rr = time_workload(pkg, torch, ww, p, args.beta, args.steps, args.warmup, args.seed, sampler, None, sus_s)
            roofline["points"][f"{name}_fp{p}"] = point(name, p, rr)
            others[f"{name}_fp{p}"] = {
                "value": ww.links * args.steps / (rr["ms_total"] * 1e-3), "unit": UNIT,
                "ms_per_step": rr["ms_per_step"], "ms_per_sweep": rr["sweep_ms"],
                "plaquette_last": rr["plaquette_last"], "su2_run_ms_per_step": rr["ms_per_step_run"],
                "su2_run_tail_overlap_ms_per_step": rr["ms_per_step_run_tail_overlap"],
            }
        line["workloads"] = others
        line["aux"] = time_aux(pkg, torch, workloads)
        line["e2e"] = time_e2e(pkg, torch, w, prec, args.beta, args.e2e_steps, 1, args.seed)
        slab = OracleSlab(w, prec, args.beta, args.seed, args.cpu_baseline_seconds)
        v, sec, n, _, _ = slab.step()
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": slab.describe(prec) + f" ({sec:.1f} s)"}
        line["cpu_baseline"]["fig1_32^4_fp32"] = cpu_fig1(line["aux"]["fig1_init_100_sweeps_plaquette_beta6"])
    sampler.stop()
    if rank == 0:
        print(json.dumps(line))
    return 0


if __name__ == "__main__":
    sys.exit(main())
