"""Host logic of the time-slab mode that needs no GPU: the decomposition arithmetic,
and the torch.distributed plumbing (RingComm) on gloo with world_size 2 and 3."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_plan_slabs_covers_the_time_axis_with_even_slabs():
    from paper_1104_5432_b200.slabs import plan_slabs
    for Nt in (2, 4, 6, 8, 32, 48, 64):
        for n in range(1, Nt // 2 + 1):
            plan = plan_slabs(Nt, n)
            assert len(plan) == n and plan[0][0] == 0
            assert all(t0 % 2 == 0 and Lt % 2 == 0 and Lt >= 2 for t0, Lt in plan)
            assert all(plan[i][0] + plan[i][1] == plan[i + 1][0] for i in range(n - 1))
            assert plan[-1][0] + plan[-1][1] == Nt
            assert max(Lt for _, Lt in plan) - min(Lt for _, Lt in plan) <= 2
    assert plan_slabs(8, 3) == [(0, 4), (4, 2), (6, 2)]
    for bad in ((8, 5), (7, 1), (8, 0), (0, 1)):
        with pytest.raises(ValueError):
            plan_slabs(*bad)


def test_global_slices_halo_map():
    from paper_1104_5432_b200.slabs import global_slices, plan_slabs
    assert global_slices(0, 4, 8) == [6, 7, 0, 1, 2, 3, 4, 5]
    assert global_slices(4, 4, 8) == [2, 3, 4, 5, 6, 7, 0, 1]
    assert global_slices(0, 2, 2) == [0, 1, 0, 1, 0, 1]  # one slab of Nt = 2: its own neighbour twice over
    # local and global time parity agree on every slice (what keeps the parity arrays aligned)
    for Nt, n in ((8, 3), (48, 4), (6, 3)):
        for t0, Lt in plan_slabs(Nt, n):
            assert all((g - t) % 2 == 0 for t, g in enumerate(global_slices(t0, Lt, Nt)))
    # slab r's lower halo is the last interior slice of slab r-1, its upper halo the first of slab r+1
    plan = plan_slabs(12, 3)
    for r, (t0, Lt) in enumerate(plan):
        gs = global_slices(t0, Lt, 12)
        lo, hi = plan[(r - 1) % 3], plan[(r + 1) % 3]
        assert gs[1] == lo[0] + lo[1] - 1 and gs[Lt + 2] == hi[0]


def test_slab_bytes_without_gpu():
    import paper_1104_5432_b200 as pkg
    from paper_1104_5432_b200 import build
    build.build()
    assert pkg.su2_slab_bytes(8, 8, 8, 4, 32) == 8 * 8 * 8 * 8 * 4 * 16
    assert pkg.su2_slab_bytes(8, 8, 8, 3, 32) == 0 and pkg.su2_slab_bytes(8, 8, 8, 0, 64) == 0


_WORKER = r"""
import os, sys, torch, torch.distributed as dist
sys.path.insert(0, os.environ["SU2_ROOT"])
from paper_1104_5432_b200.slabs import RingComm
dist.init_process_group("gloo")
c = RingComm()
assert (c.lo, c.hi) == ((c.rank - 1) % c.world, (c.rank + 1) % c.world)
# rank-ordered sum: float addition is not associative; every rank must get the rank-order bits
vals = [1e16, 1.0, -1e16, 3.0][:c.world]
tot = c.ordered_sum(torch.tensor(vals[c.rank], dtype=torch.float64))
ref = 0.0
for v in vals:
    ref += v
assert tot == ref, (tot, ref)
# chain: rank r multiplies the travelling buffer by (r + 2), in rank order
buf = torch.zeros(4, dtype=torch.float64)
def step(prev):
    if prev is None:
        buf.fill_(1.0)
    buf.mul_(c.rank + 2)
c.chain(step, buf)
want = 1.0
for r in range(c.rank + 1):
    want *= r + 2
assert (buf == want).all(), (buf, want)
last = c.broadcast_from_last(buf[0])
full = 1.0
for r in range(c.world):
    full *= r + 2
assert last == full
c.barrier_host(lambda: None)
tok = torch.zeros(1)
c.barrier_stream(tok)   # on gloo an ordinary all-reduce; on NCCL the stream-ordered barrier
if c.rank == 0:
    print("RING OK", c.world)
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world", [2, 3])
def test_ring_comm_gloo(tmp_path, world):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER)
    env = dict(os.environ, SU2_ROOT=ROOT, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
                        "--master-addr", "127.0.0.1", "--master-port", str(29550 + world), str(w)],
                       capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, r.stderr[-3000:]
    assert f"RING OK {world}" in r.stdout
