"""Time-slab drivers for the lattice split over GPUs (the paper's second
mode: PAPER.md:27, :54, :95; design in DESIGN.md §6.9; C calls su2_slab_* of include/su2_heatbath.h).

Argument marshalling and orchestration only: the update, the stores into the neighbours' halos
(peer memory), the plaquette and the Polyakov product all run in the library's kernels.

  plan_slabs / global_slices   host arithmetic of the decomposition (no GPU needed)
  Slab                         one slab handle + its link buffer
  SlabRing                     all slabs of a lattice in ONE process on one device (stream order is
                               the barrier between sub-steps) - what the 1-GPU tests run
  RingComm                     the torch.distributed plumbing of one-process-per-GPU runs: neighbours,
                               barrier, rank-ordered sum, the Polyakov chain (works on gloo/CPU tensors too)
  DistributedSlab              one slab per rank; peers' halos are reached through CUDA IPC
"""
import numpy as np

from . import (SU2_START_COLD, SU2_START_HOT, su2_device_links, su2_get_links, su2_init, su2_ipc_close,
               su2_ipc_export, su2_ipc_open, su2_lattice_destroy, su2_set_links, su2_set_seed, su2_slab_bytes,
               su2_slab_create, su2_slab_create_external, su2_slab_plaquette, su2_slab_polyakov, su2_slab_set_peers,
               su2_slab_substep, su2_synchronize)

_START = {"cold": SU2_START_COLD, "hot": SU2_START_HOT}


def plan_slabs(Nt, n_slabs):
    """Split the Nt time slices into n_slabs contiguous slabs of even extent >= 2 (the checkerboard
    needs t0 and Lt even); sizes differ by at most 2. Returns [(t0, Lt)] in slab order."""
    if Nt < 2 or Nt % 2 or n_slabs < 1 or 2 * n_slabs > Nt:
        raise ValueError(f"cannot split Nt={Nt} into {n_slabs} slabs of even extent >= 2")
    pairs, extra = divmod(Nt // 2, n_slabs)
    plan, t0 = [], 0
    for r in range(n_slabs):
        Lt = 2 * (pairs + (1 if r < extra else 0))
        plan.append((t0, Lt))
        t0 += Lt
    return plan


def global_slices(t0, Lt, Nt):
    """Global time slice held by each of the Lt + 4 local slices of a slab (2 below, interior, 2 above)."""
    return [(t0 - 2 + t) % Nt for t in range(Lt + 4)]


class Slab:
    """One time slab on the current CUDA device. own=True: the library allocates the links
    (cudaMalloc: exportable through CUDA IPC); else a torch uint8 tensor holds them."""

    def __init__(self, dims, precision, t0, Lt, device="cuda:0", own=False):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1104_5432_b200 needs a CUDA device (no CPU fallback)")
        Nx, Ny, Nz, Nt = (int(d) for d in dims)
        self.dims, self.precision, self.t0, self.Lt = (Nx, Ny, Nz, Nt), int(precision), int(t0), int(Lt)
        self.dtype = np.float32 if self.precision == 32 else np.float64
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.current_stream(self.device)
        nbytes = su2_slab_bytes(Nx, Ny, Nz, self.Lt, self.precision)
        if nbytes == 0:
            raise ValueError("bad slab extents")
        if own:
            self.storage = None
            self.h = su2_slab_create(Nx, Ny, Nz, Nt, self.precision, self.t0, self.Lt)
            from . import su2_set_stream
            su2_set_stream(self.h, self.stream.cuda_stream)
        else:
            self.storage = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.h = su2_slab_create_external(Nx, Ny, Nz, Nt, self.precision, self.t0, self.Lt,
                                              self.storage.data_ptr(), nbytes, self.stream.cuda_stream)
        self.v3 = Nx * Ny * Nz
        self.local_shape = (self.Lt + 4, Nz, Ny, Nx, 4, 4)
        tdt = torch.float32 if self.precision == 32 else torch.float64
        self.out = torch.zeros(2, dtype=torch.float64, device=self.device)       # plaquette share, Polyakov mean
        self.field = torch.empty((self.v3, 4), dtype=tdt, device=self.device)    # running Polyakov product

    @property
    def links_ptr(self):
        return su2_device_links(self.h)

    def close(self):
        if getattr(self, "h", None):
            su2_lattice_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_peers(self, lo_ptr, lo_Lt, hi_ptr, hi_Lt):
        su2_slab_set_peers(self.h, lo_ptr, lo_Lt, hi_ptr, hi_Lt)

    def init(self, start, seed):
        su2_init(self.h, _START[start], seed)

    def set_seed(self, seed):
        su2_set_seed(self.h, seed)

    def scatter_from_global(self, links):
        """links: the whole configuration in canonical order [t][z][y][x][mu][4] (any leading shape)."""
        Nx, Ny, Nz, Nt = self.dims
        g = np.asarray(links, dtype=self.dtype).reshape(Nt, Nz, Ny, Nx, 4, 4)
        su2_set_links(self.h, np.ascontiguousarray(g[global_slices(self.t0, self.Lt, Nt)]))

    def get_local(self):
        out = np.empty(self.local_shape, dtype=self.dtype)
        su2_get_links(self.h, out)
        return out

    def substep(self, beta, sweep_idx, mu, parity, fuse_plaquette=False):
        su2_slab_substep(self.h, beta, sweep_idx, mu, parity, fuse_plaquette)

    def plaquette_share(self, fused=False):
        """Enqueue; self.out[0] <- this slab's share of the mean plaquette."""
        su2_slab_plaquette(self.h, fused, self.out.data_ptr())

    def polyakov_step(self, prev, last):
        """Enqueue the slab's part of the ordered product: prev = field tensor of the slabs below (None on
        the slab with t0 = 0); the result goes to self.field, and on the last slab the mean to self.out[1]."""
        su2_slab_polyakov(self.h, prev.data_ptr() if prev is not None else 0, self.field.data_ptr(),
                          self.out.data_ptr() + 8 if last else 0)

    def synchronize(self):
        su2_synchronize(self.h)


class SlabRing:
    """Every slab of one lattice in this process, on one device and one stream: the slabs' kernels of a
    sub-step run one after the other, none waits for another, and stream order is the barrier."""

    def __init__(self, dims, precision, n_slabs, device="cuda:0"):
        self.dims, self.precision = tuple(int(d) for d in dims), int(precision)
        self.plan = plan_slabs(self.dims[3], n_slabs)
        self.slabs = [Slab(self.dims, precision, t0, Lt, device) for t0, Lt in self.plan]
        n = len(self.slabs)
        for r, s in enumerate(self.slabs):
            lo, hi = self.slabs[(r - 1) % n], self.slabs[(r + 1) % n]
            s.set_peers(lo.links_ptr, lo.Lt, hi.links_ptr, hi.Lt)
        self.dtype = self.slabs[0].dtype

    def close(self):
        for s in self.slabs:
            s.close()

    def init(self, start, seed):
        for s in self.slabs:
            s.init(start, seed)

    def set_seed(self, seed):
        for s in self.slabs:
            s.set_seed(seed)

    def set_links(self, links):
        for s in self.slabs:
            s.scatter_from_global(links)

    def get_links(self):
        """The whole configuration, canonical order, assembled from the slabs' interior slices."""
        Nx, Ny, Nz, Nt = self.dims
        out = np.empty((Nt, Nz, Ny, Nx, 4, 4), dtype=self.dtype)
        for s in self.slabs:
            out[s.t0:s.t0 + s.Lt] = s.get_local()[2:s.Lt + 2]
        return out.reshape(Nx * Ny * Nz * Nt, 4, 4)

    def substep(self, beta, sweep_idx, mu, parity, fuse_plaquette=False):
        for s in self.slabs:
            s.substep(beta, sweep_idx, mu, parity, fuse_plaquette)

    def sweep(self, beta, sweep_idx, fuse_plaquette=False):
        for mu in range(4):
            for p in range(2):
                self.substep(beta, sweep_idx, mu, p, fuse_plaquette)

    def mean_plaquette(self, fused=False):
        for s in self.slabs:
            s.plaquette_share(fused)
        tot = 0.0
        for s in self.slabs:  # slab order: a given decomposition always gives the same bits
            s.synchronize()
            tot += float(s.out[0].item())
        return tot

    def polyakov_loop(self):
        prev = None
        for r, s in enumerate(self.slabs):
            s.polyakov_step(prev, r == len(self.slabs) - 1)
            prev = s.field
        self.slabs[-1].synchronize()
        return float(self.slabs[-1].out[1].item())

    def halos_consistent(self):
        """True iff every halo slice equals, bit for bit, the interior slice it copies."""
        Nt = self.dims[3]
        loc = [s.get_local() for s in self.slabs]
        glob = self.get_links().reshape(Nt, -1)
        for s, a in zip(self.slabs, loc):
            gs = global_slices(s.t0, s.Lt, Nt)
            a = a.reshape(s.Lt + 4, -1)
            for t in (1, s.Lt + 2):
                if not np.array_equal(a[t], glob[gs[t]]):
                    return False
        return True


class RingComm:
    """torch.distributed plumbing of a ring of slabs, one rank per slab. Works on any backend and device
    (the CPU tests run it on gloo): the data it moves are one scalar per rank and the Polyakov field."""

    def __init__(self, group=None):
        import torch.distributed as dist

        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.lo, self.hi = (self.rank - 1) % self.world, (self.rank + 1) % self.world

    def barrier_stream(self, token):
        """Stream-ordered barrier (NCCL): a 1-element all-reduce on the stream the kernels run on; the next
        sub-step queues behind it, the host does not wait."""
        self.dist.all_reduce(token, group=self.group)

    def barrier_host(self, synchronize=None):
        """Host barrier for backends that are not stream-ordered (gloo): finish the device work first."""
        if synchronize is not None:
            synchronize()
        self.dist.barrier(group=self.group)

    def ordered_sum(self, value):
        """Sum of one float64 per rank, added in rank order on every rank (same bits everywhere)."""
        import torch

        mine = value.detach().reshape(1).to(torch.float64)
        parts = [torch.empty_like(mine) for _ in range(self.world)]
        self.dist.all_gather(parts, mine, group=self.group)
        tot = 0.0
        for p in parts:
            tot += float(p.item())
        return tot

    def chain(self, step, buf):
        """Polyakov chain: rank 0 starts, every rank continues the product of its lower neighbour.
        step(prev_or_None) fills buf; buf travels up the ring; returns after this rank's part."""
        if self.rank > 0:
            self.dist.recv(buf, src=self.rank - 1, group=self.group)
            step(buf)
        else:
            step(None)
        if self.rank < self.world - 1:
            self.dist.send(buf, dst=self.rank + 1, group=self.group)

    def broadcast_from_last(self, value):
        import torch

        t = value.detach().reshape(1).to(torch.float64).clone()
        self.dist.broadcast(t, src=self.world - 1, group=self.group)
        return float(t.item())


class DistributedSlab:
    """One slab per rank (one process per GPU, launched by torchrun). The neighbours' link buffers are
    mapped with CUDA IPC and written by this rank's sub-step kernel (NVLink peer stores); between
    sub-steps a barrier: stream-ordered on NCCL (barrier="stream"), or host-side (barrier="host", any
    backend; what a 2-process run on ONE GPU uses, where NCCL refuses two ranks per device)."""

    def __init__(self, dims, precision, device, group=None, barrier="stream"):
        import torch

        self.comm = RingComm(group)
        self.dims = tuple(int(d) for d in dims)
        self.plan = plan_slabs(self.dims[3], self.comm.world)
        t0, Lt = self.plan[self.comm.rank]
        self.slab = Slab(self.dims, precision, t0, Lt, device, own=True)
        self.barrier = barrier
        self.token = torch.zeros(1, device=self.slab.device if barrier == "stream" else "cpu")
        handles = [None] * self.comm.world
        self.comm.dist.all_gather_object(handles, su2_ipc_export(self.slab.h), group=group)
        self._opened = {}
        ptrs = []
        for r in (self.comm.lo, self.comm.hi):
            if r == self.comm.rank:
                ptrs.append(self.slab.links_ptr)
            else:
                if r not in self._opened:
                    self._opened[r] = su2_ipc_open(handles[r])
                ptrs.append(self._opened[r])
        self.slab.set_peers(ptrs[0], self.plan[self.comm.lo][1], ptrs[1], self.plan[self.comm.hi][1])
        self._sync()

    def _sync(self):
        if self.barrier == "stream":
            self.comm.barrier_stream(self.token)
        else:
            self.comm.barrier_host(self.slab.synchronize)

    def close(self):
        self._sync()
        self.slab.synchronize()
        for p in self._opened.values():
            su2_ipc_close(p)
        self._opened = {}
        self.comm.dist.barrier(group=self.comm.group)  # nobody frees a buffer a peer still has mapped
        self.slab.close()

    def init(self, start, seed):
        self.slab.init(start, seed)
        self._sync()

    def set_links(self, links):
        self.slab.scatter_from_global(links)
        self._sync()

    def sweep(self, beta, sweep_idx, fuse_plaquette=False):
        for mu in range(4):
            for p in range(2):
                self.slab.substep(beta, sweep_idx, mu, p, fuse_plaquette)
                self._sync()

    def mean_plaquette(self, fused=False):
        self.slab.plaquette_share(fused)
        self.slab.synchronize()
        v = self.slab.out[0]
        return self.comm.ordered_sum(v if self.barrier == "stream" else v.cpu())

    def polyakov_loop(self):
        last = self.comm.rank == self.comm.world - 1
        import torch

        prev_dev = torch.empty_like(self.slab.field)  # the product of the slabs below (received)
        if self.barrier == "stream":
            # NCCL send/recv are stream-ordered with the kernels; the field goes from device to device
            if self.comm.rank > 0:
                self.comm.dist.recv(prev_dev, src=self.comm.rank - 1, group=self.comm.group)
            self.slab.polyakov_step(prev_dev if self.comm.rank > 0 else None, last)
            if not last:
                self.comm.dist.send(self.slab.field, dst=self.comm.rank + 1, group=self.comm.group)
            self.slab.synchronize()
            return self.comm.broadcast_from_last(self.slab.out[1])
        host = self.slab.field.cpu()

        def step(prev):
            if prev is not None:
                prev_dev.copy_(prev)
            self.slab.polyakov_step(prev_dev if prev is not None else None, last)
            self.slab.synchronize()
            host.copy_(self.slab.field)

        self.comm.chain(step, host)
        return self.comm.broadcast_from_last(self.slab.out[1].cpu())

    def interior(self):
        """This rank's interior slices, canonical order [Lt][z][y][x][mu][4] (host)."""
        return self.slab.get_local()[2:self.slab.Lt + 2]
