"""Seeded, synthetic workload descriptions and input generators.

This module serves BOTH the tests/oracle side and the CUDA side, and therefore
holds none of the method's arithmetic: only the configurations of
BASELINE.json (`configs[0..4]`) and a numpy-seeded
generator of arbitrary unit-quaternion lattices used as common inputs of the
teacher-forced parity tests. The paper measures on no dataset: its workload is
a synthetic lattice, so these ARE the paper's workload shapes.
"""
from dataclasses import dataclass, field
from typing import Tuple

import numpy as np


@dataclass(frozen=True)
class Workload:
    name: str
    dims: Tuple[int, int, int, int]  # (Nx, Ny, Nz, Nt)
    precisions: Tuple[int, ...]
    start: str  # "hot" | "cold"
    seed: int
    betas: Tuple[float, ...]
    sweeps: int
    measure: Tuple[str, ...] = field(default=("plaquette",))

    @property
    def volume(self) -> int:
        return int(np.prod(self.dims))

    @property
    def links(self) -> int:
        return 4 * self.volume


# BASELINE.json configs[0..4]; seeds and sweep indices per SURVEY.md §8(d).
C1 = Workload("C1_8^4", (8, 8, 8, 8), (64,), "hot", 1, (2.3,), 10)
C2 = Workload("C2_16^3x4", (16, 16, 16, 4), (32,), "hot", 100, (2.2, 2.3, 2.4, 2.5, 2.6), 200,
              ("plaquette", "polyakov"))
C3 = Workload("C3_32^4", (32, 32, 32, 32), (32, 64), "hot", 1, (6.0,), 100)
C4 = tuple(Workload(f"C4_48^3x{nt}", (48, 48, 48, nt), (64,), "hot", 200 + nt, (2.5,), 500, ("polyakov",))
           for nt in (4, 6, 8))
C5 = Workload("C5_64^4", (64, 64, 64, 64), (32, 64), "cold", 1, (6.0,), 100)

BY_NAME = {w.name: w for w in (C1, C2, C3, *C4, C5)}


def random_links(dims, seed: int, dtype=np.float64) -> np.ndarray:
    """Haar-random unit quaternions in canonical order [site][mu][4] (site index
    x fastest), drawn with numpy's own generator (independent of Philox): a
    normalised 4-vector of standard normals is uniform on S^3."""
    V = int(np.prod(dims))
    D = len(dims)
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((V, D, 4))
    a /= np.linalg.norm(a, axis=-1, keepdims=True)
    return np.ascontiguousarray(a.astype(dtype))


def smooth_links(dims, seed: int, eps: float, dtype=np.float64) -> np.ndarray:
    """Unit quaternions close to the identity, (1, eps*g) normalised: the value
    structure of a thermalised weak-coupling lattice (large staple norm k)."""
    V = int(np.prod(dims))
    D = len(dims)
    rng = np.random.default_rng(seed)
    a = np.empty((V, D, 4))
    a[..., 0] = 1.0
    a[..., 1:] = eps * rng.standard_normal((V, D, 3))
    a /= np.linalg.norm(a, axis=-1, keepdims=True)
    return np.ascontiguousarray(a.astype(dtype))


def degenerate_staple_links(dims, s: int, mu: int, dtype=np.float64) -> np.ndarray:
    """Cold lattice in which the staple sum of link (site s, direction mu) vanishes
    exactly: U_mu(x - nu) = -1 for the three nu != mu turns every backward term into
    -1 against the +1 of the forward terms (the [R8] measure-zero case, built by hand).
    Needs every extent >= 4 so that the flipped links are distinct from the others."""
    D = len(dims)
    V = int(np.prod(dims))
    a = np.zeros((V, D, 4), dtype=dtype)
    a[..., 0] = 1.0
    x = []
    r = s
    for n in dims:
        x.append(r % n)
        r //= n
    for nu in range(D):
        if nu == mu:
            continue
        y = list(x)
        y[nu] = (y[nu] - 1) % dims[nu]
        sy = 0
        for d in reversed(range(D)):
            sy = sy * dims[d] + y[d]
        a[sy, mu, 0] = -1.0
    return a
