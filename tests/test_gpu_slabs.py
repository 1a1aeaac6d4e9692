"""GPU parity tests (-m gpu) of the time-slab mode: the
lattice split into slabs whose sub-step kernels store their edge slices into the neighbours'
halos. All slabs live on the one GPU of the test box (SlabRing: one process, one stream, no
kernel waits for another); a two-process run maps the peer buffers through CUDA IPC.

What is compared: every sub-step against the oracle on the WHOLE lattice (teacher-forced, same
tolerances as test_gpu_parity.py), the slab run against the unsplit library run bit for bit
(draws are keyed by the global site), halos against the slices they copy bit for bit, and the
plaquette / Polyakov loop against the oracle."""
import os
import subprocess
import sys

import numpy as np
import pytest

import oracle
import parity_protocol as pp
from paper_1104_5432_b200 import workloads

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

TOL = {64: 1e-12, 32: 1e-5}
PTOL = {64: 1e-12, 32: 1e-6}
MODE = {64: "f64", 32: "f32"}


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    import paper_1104_5432_b200 as p
    from paper_1104_5432_b200 import build
    build.build()
    p.lib()
    return p


@pytest.fixture(scope="module")
def slabs(pkg):
    from paper_1104_5432_b200 import slabs as s
    return s


def _parity(dims):
    V = oracle.volume(dims)
    s = np.arange(V)
    return (s % dims[0] + s // dims[0] % dims[1] + s // (dims[0] * dims[1]) % dims[2]
            + s // (dims[0] * dims[1] * dims[2])) % 2


# (dims, number of slabs): 8x4x2x2 tile / 16x4x2x1 tile / linear launch / ragged; equal and unequal
# slabs (Nt = 8 in 3 slabs = 4 + 2 + 2), one slab that is its own neighbour, minimal slabs (Lt = 2)
CASES = [((16, 4, 2, 8), 2), ((32, 4, 4, 4), 2), ((8, 8, 8, 8), 3), ((4, 2, 6, 4), 2), ((6, 4, 2, 6), 3),
         ((16, 4, 2, 4), 1), ((8, 4, 4, 8), 4)]


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,n", CASES)
def test_slab_hot_start_equals_whole_lattice(pkg, slabs, dims, n, prec):
    ring = slabs.SlabRing(dims, prec, n)
    ring.init("hot", 5)
    lat = pkg.Lattice(dims, prec)
    lat.init("hot", 5)
    assert np.array_equal(ring.get_links(), lat.get_links())
    assert ring.halos_consistent()
    ring.close()
    lat.close()


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,n", CASES)
def test_slab_substeps_match_oracle_teacher_forced(pkg, slabs, dims, n, prec):
    mode = MODE[prec]
    beta, seed, sweep = 2.3, 11, 4
    L = workloads.random_links(dims, 21, oracle.dtype(mode))
    ring = slabs.SlabRing(dims, prec, n)
    ring.set_seed(seed)
    V = oracle.volume(dims)
    par = _parity(dims)
    for mu in range(4):
        for p in range(2):
            ring.set_links(L)
            ring.substep(beta, sweep, mu, p)
            g = ring.get_links()
            o = L.copy()
            rec = pp.Records(V)
            oracle.heatbath_substep(dims, o, beta, seed, sweep, mu, p, mode, **rec.kw)
            pp.compare_links(g, o, dims, prec, [(mu, p)], rec, beta, what=f"mu={mu} p={p}")  # DESIGN.md 3 [R13], [R13b]
            untouched = np.ones((V, 4), bool)
            untouched[par == p, mu] = False
            assert (g[untouched] == L[untouched]).all()
            assert ring.halos_consistent(), f"halo differs from the slice it copies after ({mu},{p})"
            L = o
    ring.close()


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,n", CASES)
def test_slab_run_is_bitwise_the_unsplit_run(pkg, slabs, dims, n, prec):
    """Three free-running sweeps from a hot start: same links bit for bit as the whole lattice stepped by
    su2_heatbath_sweep, and the fused plaquette / chained Polyakov loop agree with the whole-lattice ones."""
    beta = 2.4
    ring = slabs.SlabRing(dims, prec, n)
    lat = pkg.Lattice(dims, prec)
    ring.init("hot", 9)
    lat.init("hot", 9)
    for k in range(3):
        ring.sweep(beta, k, fuse_plaquette=True)
        lat.sweep(beta, k)
    a, b = ring.get_links(), lat.get_links()
    assert np.array_equal(a, b), f"{int((a != b).any(-1).sum())} links differ"
    assert ring.halos_consistent()
    P, Lp = lat.measure()
    assert abs(ring.mean_plaquette(fused=True) - P) < PTOL[prec]
    assert abs(ring.mean_plaquette(fused=False) - P) < PTOL[prec]
    assert abs(ring.polyakov_loop() - Lp) < PTOL[prec]
    ring.close()
    lat.close()


@pytest.mark.parametrize("prec", [64, 32])
@pytest.mark.parametrize("dims,n", [((8, 8, 8, 8), 3), ((16, 4, 2, 8), 2), ((4, 2, 6, 4), 2)])
def test_slab_observables_match_oracle(pkg, slabs, dims, n, prec):
    mode = MODE[prec]
    L = workloads.smooth_links(dims, 4, 0.4, oracle.dtype(mode))
    ring = slabs.SlabRing(dims, prec, n)
    ring.set_links(L)
    assert abs(ring.mean_plaquette() - oracle.mean_plaquette(dims, L, mode)) < PTOL[prec]
    assert abs(ring.polyakov_loop() - oracle.polyakov_loop(dims, L, mode)) < PTOL[prec]
    # a centre flip of one time slice inside one slab flips the loop and leaves the plaquette alone [R11]
    Lf = L.reshape(dims[3], -1, 4, 4).copy()
    Lf[dims[3] - 1, :, 3, :] *= -1
    ring.set_links(Lf.reshape(L.shape))
    assert abs(ring.polyakov_loop() + oracle.polyakov_loop(dims, L, mode)) < PTOL[prec]
    assert abs(ring.mean_plaquette() - oracle.mean_plaquette(dims, L, mode)) < PTOL[prec]
    ring.close()


def test_slab_handle_refuses_whole_lattice_calls_and_bad_arguments(pkg, slabs):
    import ctypes as C
    L = pkg.lib()
    h = C.c_void_p()
    for bad in [(8, 8, 8, 8, 64, 1, 2), (8, 8, 8, 8, 64, 0, 3), (8, 8, 8, 8, 64, 6, 4), (8, 8, 8, 8, 16, 0, 4),
                (8, 8, 8, 8, 64, 0, 0), (7, 8, 8, 8, 64, 0, 4)]:
        assert L.su2_slab_create(*bad, C.byref(h)) == pkg.SU2_EARG
    assert pkg.su2_slab_bytes(8, 8, 8, 4, 64) == pkg.su2_lattice_bytes(8, 8, 8, 8, 64)
    s = slabs.Slab((8, 8, 8, 8), 64, 4, 4)
    s.init("cold", 1)
    with pytest.raises(pkg.SU2Error) as e:  # peers first
        s.substep(2.3, 0, 0, 0)
    assert e.value.code == pkg.SU2_ESTATE
    for call in (lambda: pkg.su2_heatbath_sweep(s.h, 2.3, 0), lambda: pkg.su2_mean_plaquette(s.h),
                 lambda: pkg.su2_polyakov_correlator(s.h, 2), lambda: pkg.su2_run(s.h, 2.3, 0, 1, s.out.data_ptr())):
        with pytest.raises(pkg.SU2Error) as e:
            call()
        assert e.value.code == pkg.SU2_ESTATE
    with pytest.raises(pkg.SU2Error):  # dev_prev must be given exactly when t0 > 0
        pkg.su2_slab_polyakov(s.h, 0, s.field.data_ptr(), 0)
    lat = pkg.Lattice((8, 8, 8, 8), 64)
    with pytest.raises(pkg.SU2Error):
        pkg.su2_slab_substep(lat.h, 2.3, 0, 0, 0, 0)
    lat.close()
    s.close()


_WORKER = r"""
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, os.environ["SU2_ROOT"])
import paper_1104_5432_b200 as pkg
from paper_1104_5432_b200 import slabs, workloads
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
dims, prec, beta = (16, 4, 2, 8), int(os.environ["SU2_PREC"]), 2.4
ds = slabs.DistributedSlab(dims, prec, "cuda:0", barrier="host")   # both ranks on the one GPU of the box
L = workloads.random_links(dims, 21, np.float64 if prec == 64 else np.float32)
ds.set_links(L)
ds.slab.set_seed(7)
for k in range(2):
    ds.sweep(beta, k, fuse_plaquette=True)
P, Lp = ds.mean_plaquette(fused=True), ds.polyakov_loop()
mine = torch.from_numpy(np.ascontiguousarray(ds.interior()))
parts = [torch.empty_like(mine) for _ in range(world)]
dist.all_gather(parts, mine)
ds.close()
if rank == 0:
    lat = pkg.Lattice(dims, prec)
    lat.set_links(L); lat.set_seed(7)
    for k in range(2):
        lat.sweep(beta, k)
    ref = lat.get_links().reshape(dims[3], -1)
    got = torch.cat(parts).numpy().reshape(dims[3], -1)
    P0, L0 = lat.measure()
    tol = 1e-12 if prec == 64 else 1e-6
    assert np.array_equal(ref, got), "links differ"
    assert abs(P - P0) < tol and abs(Lp - L0) < tol, (P, P0, Lp, L0)
    print("SLAB2 OK", world)
dist.destroy_process_group()
"""


@pytest.mark.parametrize("prec", [64, 32])
def test_two_processes_peer_stores_through_cuda_ipc(pkg, tmp_path, prec):
    """One process per slab, the neighbour's buffer mapped with CUDA IPC and written by this process's
    kernels; host barrier between sub-steps (gloo), so no kernel ever waits for another process."""
    w = tmp_path / "worker.py"
    w.write_text(_WORKER)
    env = dict(os.environ, SU2_ROOT=ROOT, SU2_PREC=str(prec), MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", str(29541 + prec), str(w)],
                       capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-3000:])
    assert "SLAB2 OK 2" in r.stdout
