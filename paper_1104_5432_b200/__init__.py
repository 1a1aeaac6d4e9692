"""paper_1104_5432_b200 — B200-native SU(2) heat-bath lattice generator.

Thin Python binding of the C-ABI library `libsu2hb.so` (include/su2_heatbath.h).
Argument marshalling only: every step of the path (init, heat-bath sweep,
plaquette, Polyakov loop) runs in the hand-written sm_100a kernels under csrc/.
PyTorch is used for device memory and streams, nothing else. There is no CPU
fallback: if the library is missing or no CUDA device is present, calls raise.

The functions carry the names of the C calls; `Lattice` is a small convenience
wrapper that owns a handle and a torch-allocated link buffer.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsu2hb.so")

SU2_OK, SU2_EARG, SU2_EALLOC, SU2_ECUDA, SU2_ESTATE, SU2_ETOOBIG = 0, 1, 2, 3, 4, 5
SU2_NOALLOC_MAX_SITES = 1 << 25
SU2_START_COLD, SU2_START_HOT = 0, 1
SU2_DRAW_KP, SU2_DRAW_AUTO, SU2_DRAW_CREUTZ = 0, 1, 2
SU2_ALPHA_C = 1.6847
SU2_OPT_OVERLAP, SU2_OPT_RUN_GRAPH, SU2_OPT_TAIL_OVERLAP = 0, 1, 2
SU2_PROBE_READ, SU2_PROBE_COPY = 0, 1

_lib = None

_SIGNATURES = {
    "su2_lattice_bytes": (C.c_size_t, [C.c_int] * 5),
    "su2_lattice_create": (C.c_int, [C.c_int] * 5 + [C.POINTER(C.c_void_p)]),
    "su2_lattice_create_external": (C.c_int, [C.c_int] * 5 + [C.c_void_p, C.c_size_t, C.c_void_p,
                                                             C.POINTER(C.c_void_p)]),
    "su2_lattice_create_batch": (C.c_int, [C.c_int] * 6 + [C.POINTER(C.c_void_p)]),
    "su2_lattice_create_batch_external": (C.c_int, [C.c_int] * 6 + [C.c_void_p, C.c_size_t, C.c_void_p,
                                                                    C.POINTER(C.c_void_p)]),
    "su2_replicas": (C.c_int, [C.c_void_p]),
    "su2_select_replica": (C.c_int, [C.c_void_p, C.c_int]),
    "su2_batch_init": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "su2_batch_sweep_measure": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p, C.c_size_t]),
    "su2_batch_run": (C.c_int, [C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p]),
    "su2_lattice_destroy": (C.c_int, [C.c_void_p]),
    "su2_set_stream": (C.c_int, [C.c_void_p, C.c_void_p]),
    "su2_init": (C.c_int, [C.c_void_p, C.c_int, C.c_uint64]),
    "su2_set_seed": (C.c_int, [C.c_void_p, C.c_uint64]),
    "su2_set_draw": (C.c_int, [C.c_void_p, C.c_int]),
    "su2_set_option": (C.c_int, [C.c_void_p, C.c_int, C.c_int]),
    "su2_heatbath_sweep": (C.c_int, [C.c_void_p, C.c_double, C.c_uint32]),
    "su2_heatbath_substep": (C.c_int, [C.c_void_p, C.c_double, C.c_uint32, C.c_int, C.c_int]),
    "su2_heatbath_sweep_measure": (C.c_int, [C.c_void_p, C.c_double, C.c_uint32, C.c_void_p, C.c_size_t,
                                             C.c_void_p]),
    "su2_run": (C.c_int, [C.c_void_p, C.c_double, C.c_uint32, C.c_uint32, C.c_void_p]),
    "su2_mean_plaquette": (C.c_int, [C.c_void_p, C.POINTER(C.c_double)]),
    "su2_polyakov_loop": (C.c_int, [C.c_void_p, C.POINTER(C.c_double)]),
    "su2_measure": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "su2_measure_async": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "su2_polyakov_correlator": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "su2_get_links": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "su2_set_links": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "su2_synchronize": (C.c_int, [C.c_void_p]),
    "su2_slab_bytes": (C.c_size_t, [C.c_int] * 5),
    "su2_slab_create": (C.c_int, [C.c_int] * 7 + [C.POINTER(C.c_void_p)]),
    "su2_slab_create_external": (C.c_int, [C.c_int] * 7 + [C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]),
    "su2_slab_set_peers": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int]),
    "su2_slab_substep": (C.c_int, [C.c_void_p, C.c_double, C.c_uint32, C.c_int, C.c_int, C.c_int]),
    "su2_slab_plaquette": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "su2_slab_polyakov": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "su2_ipc_export": (C.c_int, [C.c_void_p, C.c_void_p]),
    "su2_ipc_open": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p)]),
    "su2_ipc_close": (C.c_int, [C.c_void_p]),
    "su2_mean_plaquette_noalloc": (C.c_int, [C.c_void_p] + [C.c_int] * 5 + [C.c_void_p, C.c_void_p]),
    "su2_bandwidth_probe": (C.c_int, [C.c_size_t, C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_double),
                                      C.POINTER(C.c_double)]),
    "su2_launch_count": (C.c_uint64, [C.c_void_p]),
    "su2_device_links": (C.c_void_p, [C.c_void_p]),
    "su2_last_error": (C.c_char_p, [C.c_void_p]),
    "su2_strerror": (C.c_char_p, [C.c_int]),
}
EXPORTS = tuple(_SIGNATURES)


class SU2Error(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"su2 error {code}: {msg}")
        self.code = code


def lib():
    """Load libsu2hb.so (built in-tree by paper_1104_5432_b200.build). Raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not built: run `python -m paper_1104_5432_b200.build` "
                               "(there is no CPU fallback)")
        handle = C.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(handle, name)
            fn.restype, fn.argtypes = res, args
        _lib = handle
    return _lib


def _check(code, handle=None):
    if code != SU2_OK:
        L = lib()
        msg = L.su2_strerror(code).decode()
        if handle:
            detail = L.su2_last_error(handle).decode()
            if detail:
                msg += ": " + detail
        raise SU2Error(code, msg)


# ---- same-named functional API (handles are ctypes.c_void_p) -------------------------
def su2_lattice_bytes(Nx, Ny, Nz, Nt, precision):
    return lib().su2_lattice_bytes(Nx, Ny, Nz, Nt, precision)


def su2_lattice_create(Nx, Ny, Nz, Nt, precision):
    h = C.c_void_p()
    _check(lib().su2_lattice_create(Nx, Ny, Nz, Nt, precision, C.byref(h)))
    return h


def su2_lattice_create_external(Nx, Ny, Nz, Nt, precision, dev_ptr, nbytes, cuda_stream=0):
    h = C.c_void_p()
    _check(lib().su2_lattice_create_external(Nx, Ny, Nz, Nt, precision, C.c_void_p(dev_ptr), nbytes,
                                             C.c_void_p(cuda_stream), C.byref(h)))
    return h


def su2_lattice_create_batch(Nx, Ny, Nz, Nt, precision, n_replicas):
    h = C.c_void_p()
    _check(lib().su2_lattice_create_batch(Nx, Ny, Nz, Nt, precision, n_replicas, C.byref(h)))
    return h


def su2_lattice_create_batch_external(Nx, Ny, Nz, Nt, precision, n_replicas, dev_ptr, nbytes, cuda_stream=0):
    h = C.c_void_p()
    _check(lib().su2_lattice_create_batch_external(Nx, Ny, Nz, Nt, precision, n_replicas, C.c_void_p(dev_ptr), nbytes,
                                                   C.c_void_p(cuda_stream), C.byref(h)))
    return h


def su2_replicas(h):
    return lib().su2_replicas(h)


def su2_select_replica(h, replica):
    _check(lib().su2_select_replica(h, replica), h)


def su2_batch_init(h, start, seeds):
    a = np.ascontiguousarray(seeds, dtype=np.uint64)
    _check(lib().su2_batch_init(h, start, C.c_void_p(a.ctypes.data)), h)


def su2_batch_sweep_measure(h, betas, sweep_idx, dev_out_ptr, index):
    a = np.ascontiguousarray(betas, dtype=np.float64)
    _check(lib().su2_batch_sweep_measure(h, C.c_void_p(a.ctypes.data), sweep_idx, C.c_void_p(dev_out_ptr), index), h)


def su2_batch_run(h, betas, sweep_idx0, n_steps, dev_out_ptr):
    a = np.ascontiguousarray(betas, dtype=np.float64)
    _check(lib().su2_batch_run(h, C.c_void_p(a.ctypes.data), sweep_idx0, n_steps, C.c_void_p(dev_out_ptr)), h)


def su2_lattice_destroy(h):
    _check(lib().su2_lattice_destroy(h))


def su2_set_stream(h, cuda_stream):
    _check(lib().su2_set_stream(h, C.c_void_p(cuda_stream)), h)


def su2_init(h, start, seed):
    _check(lib().su2_init(h, start, seed), h)


def su2_set_seed(h, seed):
    _check(lib().su2_set_seed(h, seed), h)


def su2_set_draw(h, method):
    _check(lib().su2_set_draw(h, method), h)


def su2_set_option(h, option, value):
    _check(lib().su2_set_option(h, option, int(value)), h)


def su2_heatbath_sweep(h, beta, sweep_idx):
    _check(lib().su2_heatbath_sweep(h, beta, sweep_idx), h)


def su2_heatbath_substep(h, beta, sweep_idx, mu, parity):
    _check(lib().su2_heatbath_substep(h, beta, sweep_idx, mu, parity), h)


def su2_heatbath_sweep_measure(h, beta, sweep_idx, dev_out_ptr, index, event_after_sweep=0):
    _check(lib().su2_heatbath_sweep_measure(h, beta, sweep_idx, C.c_void_p(dev_out_ptr), index,
                                            C.c_void_p(event_after_sweep)), h)


def su2_run(h, beta, sweep_idx0, n_steps, dev_out_ptr):
    _check(lib().su2_run(h, beta, sweep_idx0, n_steps, C.c_void_p(dev_out_ptr)), h)


def su2_mean_plaquette(h):
    out = C.c_double()
    _check(lib().su2_mean_plaquette(h, C.byref(out)), h)
    return out.value


def su2_polyakov_loop(h):
    out = C.c_double()
    _check(lib().su2_polyakov_loop(h, C.byref(out)), h)
    return out.value


def su2_measure(h):
    p, l = C.c_double(), C.c_double()
    _check(lib().su2_measure(h, C.byref(p), C.byref(l)), h)
    return p.value, l.value


def su2_measure_async(h, dev_out_ptr, index):
    _check(lib().su2_measure_async(h, C.c_void_p(dev_out_ptr), index), h)


def su2_polyakov_correlator(h, rmax):
    out = np.zeros(rmax, dtype=np.float64)
    _check(lib().su2_polyakov_correlator(h, rmax, C.c_void_p(out.ctypes.data)), h)
    return out


def su2_get_links(h, host_array):
    assert host_array.flags.c_contiguous
    _check(lib().su2_get_links(h, C.c_void_p(host_array.ctypes.data), host_array.nbytes), h)


def su2_set_links(h, host_array):
    assert host_array.flags.c_contiguous
    _check(lib().su2_set_links(h, C.c_void_p(host_array.ctypes.data), host_array.nbytes), h)


def su2_synchronize(h):
    _check(lib().su2_synchronize(h), h)


def su2_mean_plaquette_noalloc(dev_links_ptr, Nx, Ny, Nz, Nt, precision, dev_out_ptr, cuda_stream=0):
    """Mean plaquette of a device-layout configuration into *dev_out_ptr; allocates nothing (static scratch)."""
    _check(lib().su2_mean_plaquette_noalloc(C.c_void_p(dev_links_ptr), Nx, Ny, Nz, Nt, precision,
                                            C.c_void_p(cuda_stream), C.c_void_p(dev_out_ptr)))


def su2_bandwidth_probe(nbytes, passes, mode=SU2_PROBE_READ, cuda_stream=0):
    """(GB/s, microseconds per pass) of a read or copy pass over a scratch buffer of nbytes."""
    gbs, us = C.c_double(), C.c_double()
    _check(lib().su2_bandwidth_probe(nbytes, passes, mode, C.c_void_p(cuda_stream), C.byref(gbs), C.byref(us)))
    return gbs.value, us.value


def su2_launch_count(h):
    return lib().su2_launch_count(h)


# ---- time slabs (S8(f) NEXT-4; drivers in paper_1104_5432_b200.slabs) --------------------------
def su2_slab_bytes(Nx, Ny, Nz, Lt, precision):
    return lib().su2_slab_bytes(Nx, Ny, Nz, Lt, precision)


def su2_slab_create(Nx, Ny, Nz, Nt, precision, t0, Lt):
    h = C.c_void_p()
    _check(lib().su2_slab_create(Nx, Ny, Nz, Nt, precision, t0, Lt, C.byref(h)))
    return h


def su2_slab_create_external(Nx, Ny, Nz, Nt, precision, t0, Lt, dev_ptr, nbytes, cuda_stream=0):
    h = C.c_void_p()
    _check(lib().su2_slab_create_external(Nx, Ny, Nz, Nt, precision, t0, Lt, C.c_void_p(dev_ptr), nbytes,
                                          C.c_void_p(cuda_stream), C.byref(h)))
    return h


def su2_slab_set_peers(h, lo_ptr, lo_Lt, hi_ptr, hi_Lt):
    _check(lib().su2_slab_set_peers(h, C.c_void_p(lo_ptr), lo_Lt, C.c_void_p(hi_ptr), hi_Lt), h)


def su2_slab_substep(h, beta, sweep_idx, mu, parity, fuse_plaquette=0):
    _check(lib().su2_slab_substep(h, beta, sweep_idx, mu, parity, int(fuse_plaquette)), h)


def su2_slab_plaquette(h, fused, dev_out_ptr):
    _check(lib().su2_slab_plaquette(h, int(fused), C.c_void_p(dev_out_ptr)), h)


def su2_slab_polyakov(h, dev_prev_ptr, dev_next_ptr, dev_out_ptr):
    _check(lib().su2_slab_polyakov(h, C.c_void_p(dev_prev_ptr or None), C.c_void_p(dev_next_ptr or None),
                                   C.c_void_p(dev_out_ptr or None)), h)


def su2_ipc_export(h):
    buf = C.create_string_buffer(64)
    _check(lib().su2_ipc_export(h, buf), h)
    return buf.raw


def su2_ipc_open(handle64):
    assert len(handle64) == 64
    p = C.c_void_p()
    _check(lib().su2_ipc_open(C.c_char_p(handle64), C.byref(p)))
    return p.value


def su2_ipc_close(dev_ptr):
    _check(lib().su2_ipc_close(C.c_void_p(dev_ptr)))


def su2_device_links(h):
    return lib().su2_device_links(h)


# ---- convenience wrapper ---------------------------------------------------------------
class Lattice:
    """One SU(2) lattice on the current CUDA device. Link storage is a torch uint8
    tensor (PyTorch owns the memory; the library borrows it), work runs on torch's
    current stream at construction time."""

    def __init__(self, dims, precision=64, device="cuda:0", replicas=1):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1104_5432_b200 needs a CUDA device (no CPU fallback)")
        Nx, Ny, Nz, Nt = (int(d) for d in dims)
        self.dims = (Nx, Ny, Nz, Nt)
        self.precision = int(precision)
        self.dtype = np.float32 if self.precision == 32 else np.float64
        nbytes = su2_lattice_bytes(Nx, Ny, Nz, Nt, self.precision)
        if nbytes == 0:
            raise SU2Error(SU2_EARG, "extents must be even and >= 2, V < 2^32, precision 32 or 64")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.replicas = int(replicas)
        self.storage = torch.empty(nbytes * self.replicas, dtype=torch.uint8, device=self.device)
        self.stream = torch.cuda.current_stream(self.device)
        if self.replicas == 1:
            self.h = su2_lattice_create_external(Nx, Ny, Nz, Nt, self.precision, self.storage.data_ptr(), nbytes,
                                                 self.stream.cuda_stream)
        else:  # a batch of configurations updated together (su2_batch_*); other calls act on the selected one
            self.h = su2_lattice_create_batch_external(Nx, Ny, Nz, Nt, self.precision, self.replicas,
                                                       self.storage.data_ptr(), nbytes * self.replicas,
                                                       self.stream.cuda_stream)
        self.volume = Nx * Ny * Nz * Nt
        self.nlinks = 4 * self.volume

    def close(self):
        if getattr(self, "h", None):
            su2_lattice_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init(self, start, seed):
        su2_init(self.h, {"cold": SU2_START_COLD, "hot": SU2_START_HOT}[start], seed)

    def set_seed(self, seed):
        su2_set_seed(self.h, seed)

    def select(self, replica):
        su2_select_replica(self.h, replica)

    def batch_init(self, start, seeds):
        su2_batch_init(self.h, {"cold": SU2_START_COLD, "hot": SU2_START_HOT}[start], seeds)

    def batch_sweep_measure(self, betas, sweep_idx, dev_out, index):
        """dev_out: float64 device tensor; step `index` of replica r lands at [2*(index*replicas + r) + {0,1}]."""
        assert len(betas) == self.replicas and dev_out.numel() >= 2 * self.replicas * (index + 1)
        su2_batch_sweep_measure(self.h, betas, sweep_idx, dev_out.data_ptr(), index)

    def batch_run(self, betas, sweep_idx0, n_steps, dev_out):
        """n_steps rounds as one call; step i of replica r lands at dev_out[2*(i*replicas + r) + {0,1}]."""
        assert len(betas) == self.replicas and dev_out.numel() >= 2 * self.replicas * n_steps
        su2_batch_run(self.h, betas, sweep_idx0, n_steps, dev_out.data_ptr())

    def set_draw(self, method):
        su2_set_draw(self.h, {"kp": SU2_DRAW_KP, "auto": SU2_DRAW_AUTO, "creutz": SU2_DRAW_CREUTZ}[method])

    def set_option(self, option, value):
        su2_set_option(self.h, {"overlap": SU2_OPT_OVERLAP, "run_graph": SU2_OPT_RUN_GRAPH, "tail_overlap": SU2_OPT_TAIL_OVERLAP}[option], value)

    def sweep(self, beta, sweep_idx):
        su2_heatbath_sweep(self.h, beta, sweep_idx)

    def sweep_measure(self, beta, sweep_idx, dev_out, index, event_after_sweep=None):
        """dev_out: torch float64 device tensor; event_after_sweep: a recorded-once torch.cuda.Event."""
        ev = event_after_sweep.cuda_event if event_after_sweep is not None else 0
        su2_heatbath_sweep_measure(self.h, beta, sweep_idx, dev_out.data_ptr(), index, ev)

    def run(self, beta, sweep_idx0, n_steps, dev_out):
        """n_steps x (sweep + plaquette + Polyakov loop); dev_out: float64 device tensor, 2*n_steps."""
        assert dev_out.numel() >= 2 * n_steps
        su2_run(self.h, beta, sweep_idx0, n_steps, dev_out.data_ptr())

    def substep(self, beta, sweep_idx, mu, parity):
        su2_heatbath_substep(self.h, beta, sweep_idx, mu, parity)

    def mean_plaquette(self):
        return su2_mean_plaquette(self.h)

    def polyakov_loop(self):
        return su2_polyakov_loop(self.h)

    def measure(self):
        return su2_measure(self.h)

    def measure_async(self, dev_out, index):
        su2_measure_async(self.h, dev_out.data_ptr(), index)

    def polyakov_correlator(self, rmax):
        return su2_polyakov_correlator(self.h, rmax)

    def get_links(self, out=None):
        if out is None:
            out = np.empty((self.volume, 4, 4), dtype=self.dtype)
        su2_get_links(self.h, out)
        return out

    def set_links(self, links):
        su2_set_links(self.h, np.ascontiguousarray(links, dtype=self.dtype))

    def synchronize(self):
        su2_synchronize(self.h)

    @property
    def launch_count(self):
        return su2_launch_count(self.h)
