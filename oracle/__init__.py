"""ctypes wrapper of the CPU oracle (oracle/su2_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: import only from tests/, from
__graft_entry__.smoke() and from bench.py's cpu_baseline / --impl reference
leg. Nothing under paper_1104_5432_b200/ imports this package, and this
package imports nothing from paper_1104_5432_b200/.

Links are numpy arrays in canonical order [site][mu][4] (site index
s = x0 + N0*(x1 + N1*(...)), x0 fastest; SURVEY.md §8(b) "[t][z][y][x][mu][4]").
`mode` is "f64", "f32" or "f32x" (fp32 storage, fp64 arithmetic).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None
_DT = {"f64": np.float64, "f32": np.float32, "f32x": np.float32}


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.orc_philox4x32_10.restype = None
        for m in _DT:
            areal = C.c_float if m == "f32" else C.c_double
            f = getattr(_lib, f"orc_uniform_{m}")
            f.argtypes = [C.c_uint32]
            f.restype = areal
            for name in ("orc_init", "orc_staple", "orc_staple_norms", "orc_kp_x0", "orc_creutz_x0", "orc_set_draw", "orc_heatbath_link",
                         "orc_heatbath_substep", "orc_heatbath_sweep", "orc_mean_plaquette",
                         "orc_plaquette_at", "orc_polyakov_loop", "orc_polyakov_correlator", "orc_gauge_transform"):
                getattr(_lib, f"{name}_{m}").restype = C.c_int
            getattr(_lib, f"orc_qmul_{m}").restype = None
    return _lib


def dtype(mode):
    return _DT[mode]


def _dims(dims):
    d = np.ascontiguousarray(dims, dtype=np.int32)
    return len(d), d


def _p(a):
    return C.c_void_p(a.ctypes.data) if a is not None else C.c_void_p(0)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def volume(dims):
    return int(np.prod(np.asarray(dims, dtype=np.int64)))


def philox4x32_10(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def uniform(w, mode="f64"):
    return getattr(lib(), f"orc_uniform_{mode}")(int(w))


def qmul(a, b, mode="f64"):
    a = np.ascontiguousarray(a, dtype=_DT[mode])
    b = np.ascontiguousarray(b, dtype=_DT[mode])
    c = np.zeros(4, dtype=_DT[mode])
    getattr(lib(), f"orc_qmul_{mode}")(_p(a), _p(b), _p(c))
    return c


def init(dims, start, seed, mode="f64"):
    """start: 'cold' or 'hot'. Returns links [V][D][4]."""
    D, d = _dims(dims)
    links = np.empty((volume(dims), D, 4), dtype=_DT[mode])
    rc = getattr(lib(), f"orc_init_{mode}")(D, _p(d), {"cold": 0, "hot": 1}[start], C.c_uint64(seed), _p(links))
    _check(rc, "init")
    return links


def staple(dims, links, s, mu, mode="f64"):
    D, d = _dims(dims)
    v = np.zeros(4, dtype=_DT[mode])
    _check(getattr(lib(), f"orc_staple_{mode}")(D, _p(d), _p(links), C.c_int64(s), mu, _p(v)), "staple")
    return v


def staple_norms(dims, links, mode="f64"):
    D, d = _dims(dims)
    k = np.zeros((volume(dims), D), dtype=np.float64)
    _check(getattr(lib(), f"orc_staple_norms_{mode}")(D, _p(d), _p(links), _p(k)), "staple_norms")
    return k


def kp_x0(alpha, seed, s, sweep, mode="f64"):
    x0 = C.c_double(0)
    tr = C.c_int(0)
    rc = getattr(lib(), f"orc_kp_x0_{mode}")(C.c_double(alpha), C.c_uint64(seed), C.c_uint32(s), C.c_uint32(sweep),
                                            C.byref(x0), C.byref(tr))
    _check(rc, "kp_x0")
    return x0.value, tr.value


def creutz_x0(alpha, seed, s, sweep, mode="f64"):
    x0 = C.c_double(0)
    tr = C.c_int(0)
    rc = getattr(lib(), f"orc_creutz_x0_{mode}")(C.c_double(alpha), C.c_uint64(seed), C.c_uint32(s),
                                                C.c_uint32(sweep), C.byref(x0), C.byref(tr))
    _check(rc, "creutz_x0")
    return x0.value, tr.value


DRAW = {"kp": 0, "auto": 1, "creutz": 2}
ALPHA_C = 1.6847  # [R15]


def set_draw(method, mode="f64"):
    """Draw of x0 used by the heat-bath calls of `mode` from now on: 'kp' (default, [R6]),
    'creutz' ([R15]) or 'auto' (per link: Creutz iff alpha < ALPHA_C). Process-wide per mode."""
    _check(getattr(lib(), f"orc_set_draw_{mode}")(DRAW[method]), "set_draw")


def heatbath_link(dims, links, beta, seed, sweep, s, mu, mode="f64", return_k=False, return_delta=False):
    """New link of (site s, direction mu), lattice untouched. Returns (u, trials, margin[, k][, delta])."""
    D, d = _dims(dims)
    u = np.zeros(4, dtype=_DT[mode])
    tr = C.c_int(0)
    mg = C.c_double(0)
    kn, dl = C.c_double(0), C.c_double(0)
    rc = getattr(lib(), f"orc_heatbath_link_{mode}")(D, _p(d), _p(links), C.c_double(beta), C.c_uint64(seed),
                                                    C.c_uint32(sweep), C.c_int64(s), mu, _p(u), C.byref(tr),
                                                    C.byref(mg), C.byref(kn), C.byref(dl))
    _check(rc, "heatbath_link")
    out = (u, tr.value, mg.value)
    if return_k:
        out += (kn.value,)
    if return_delta:
        out += (dl.value,)
    return out


def heatbath_substep(dims, links, beta, seed, sweep, mu, parity, mode="f64", order=None, trials=None, margin=None,
                     knorm=None, delta=None):
    """In place on `links`. trials: int32 [V][D]; margin, knorm (staple norm k of each updated link), delta
    (the accepted 1 - x0 of its draw): float64 [V][D]; all optional, only the entries of the updated links
    are written."""
    D, d = _dims(dims)
    assert links.dtype == _DT[mode] and links.flags.c_contiguous
    if order is not None:
        order = np.ascontiguousarray(order, dtype=np.int64)
    rc = getattr(lib(), f"orc_heatbath_substep_{mode}")(D, _p(d), _p(links), C.c_double(beta), C.c_uint64(seed),
                                                       C.c_uint32(sweep), mu, parity, _p(order), _p(trials),
                                                       _p(margin), _p(knorm), _p(delta))
    _check(rc, "heatbath_substep")


def heatbath_sweep(dims, links, beta, seed, sweep, mode="f64", trials=None, margin=None, knorm=None, delta=None):
    """In place on `links`. trials: int32 [V][D]; margin, knorm, delta: float64 [V][D] (all optional)."""
    D, d = _dims(dims)
    assert links.dtype == _DT[mode] and links.flags.c_contiguous
    rc = getattr(lib(), f"orc_heatbath_sweep_{mode}")(D, _p(d), _p(links), C.c_double(beta), C.c_uint64(seed),
                                                     C.c_uint32(sweep), _p(trials), _p(margin), _p(knorm), _p(delta))
    _check(rc, "heatbath_sweep")


def mean_plaquette(dims, links, mode="f64"):
    D, d = _dims(dims)
    out = C.c_double(0)
    _check(getattr(lib(), f"orc_mean_plaquette_{mode}")(D, _p(d), _p(links), C.byref(out)), "mean_plaquette")
    return out.value


def plaquette_at(dims, links, s, mu, nu, mode="f64"):
    D, d = _dims(dims)
    out = C.c_double(0)
    rc = getattr(lib(), f"orc_plaquette_at_{mode}")(D, _p(d), _p(links), C.c_int64(s), mu, nu, C.byref(out))
    _check(rc, "plaquette_at")
    return out.value


def polyakov_loop(dims, links, mode="f64", return_field=False):
    D, d = _dims(dims)
    out = C.c_double(0)
    field = np.zeros(volume(dims) // int(dims[-1]), dtype=np.float64) if return_field else None
    rc = getattr(lib(), f"orc_polyakov_loop_{mode}")(D, _p(d), _p(links), C.byref(out), _p(field))
    _check(rc, "polyakov_loop")
    return (out.value, field) if return_field else out.value


def polyakov_correlator(dims, links, rmax, mode="f64"):
    """C(r) = <l(x) l(x + r e_i)> over all spatial x and the D-1 spatial axes, r = 1..rmax (eq. 3)."""
    D, d = _dims(dims)
    out = np.zeros(rmax, dtype=np.float64)
    rc = getattr(lib(), f"orc_polyakov_correlator_{mode}")(D, _p(d), _p(links), int(rmax), _p(out))
    _check(rc, "polyakov_correlator")
    return out


def gauge_transform(dims, links, seed, mode="f64"):
    """In place."""
    D, d = _dims(dims)
    _check(getattr(lib(), f"orc_gauge_transform_{mode}")(D, _p(d), _p(links), C.c_uint64(seed)), "gauge_transform")
