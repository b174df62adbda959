"""Seeded, synthetic workloads: the ONLY module both the CUDA path's tests/bench and the oracle's tests use.

Holds configuration data and crafted start lattices, none of the method's arithmetic (no Philox, no threshold,
no neighbour tables).  The paper (arXiv 1110.0899) measures on no dataset: its workload is a
self-generated periodic Ising lattice at T_c, so these configs ARE the paper's workload, not a stand-in.

Configs are BASELINE.json's `configs` (C1..C5b).  Temperatures are reading R14 of
DESIGN.md: T_c(2D) = 2/ln(1+sqrt 2) evaluated in double; T_c(3D) = 4.511528 (BASELINE.json; the paper prints
4.510).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

TC_2D = 2.0 / math.log(1.0 + math.sqrt(2.0))   # 2.269185314213022
TC_3D = 4.511528
TC_3D_PAPER = 4.510                            # PAPER.md:126, context only


@dataclass(frozen=True)
class Config:
    name: str
    dim: int
    L: int
    J: float
    T: float
    seed: int
    n_equil: int
    n_meas: int

    @property
    def N(self) -> int:
        return self.L ** self.dim

    def create_args(self):
        return (self.dim, self.L, self.J, self.T, self.seed)


CONFIGS = {
    "C1": Config("C1: 2D L=64 T_c", 2, 64, 1.0, TC_2D, 1, 0, 1000),
    "C2": Config("C2: 2D L=1024 T_c", 2, 1024, 1.0, TC_2D, 1, 1000, 10000),
    "C3": Config("C3: 2D L=4096 T_c", 2, 4096, 1.0, TC_2D, 1, 1000, 10000),
    "C4": Config("C4: 3D L=128 T_c", 3, 128, 1.0, TC_3D, 1, 1000, 10000),
    "C5a": Config("C5a: 3D L=256 T_c", 3, 256, 1.0, TC_3D, 1, 1000, 10000),
    "C5b": Config("C5b: 3D L=256 T=5.0", 3, 256, 1.0, 5.0, 1, 1000, 10000),
}


# ---------------------------------------------------------------- crafted start lattices (for set_spins)

def cold(N: int, sign: int = +1) -> np.ndarray:
    """All spins equal: the 'equilibrated' benchmark variant starts here (SURVEY.md 8(d) 'Start state')."""
    return np.full(N, sign, dtype=np.int8)


def random_pm1(N: int, seed: int, p_up: float = 0.5) -> np.ndarray:
    """i.i.d. +/-1 from numpy's PCG64 (NOT the method's Philox start; that one each side computes itself)."""
    rng = np.random.default_rng(seed)
    return np.where(rng.random(N) < p_up, 1, -1).astype(np.int8)


def checkerboard(dim: int, L: int) -> np.ndarray:
    idx = np.indices((L,) * dim).sum(axis=0)
    return np.where(idx % 2 == 0, 1, -1).astype(np.int8).reshape(-1)


def stripes(dim: int, L: int, width: int = 1, axis: int = 0) -> np.ndarray:
    """Stripes of `width` sites alternating along coordinate `axis` (0 = x, the fastest index)."""
    coords = np.indices((L,) * dim)          # coords[k] varies along numpy axis k; numpy axis dim-1 is x
    c = coords[dim - 1 - axis]
    return np.where((c // width) % 2 == 0, 1, -1).astype(np.int8).reshape(-1)


def blobs(dim: int, L: int, seed: int, n_blobs: int = 6) -> np.ndarray:
    """A few periodic balls of -1 in a +1 sea: large same-sign components with ragged boundaries."""
    rng = np.random.default_rng(seed)
    grid = np.indices((L,) * dim).astype(np.int64)
    s = np.ones((L,) * dim, dtype=np.int8)
    for _ in range(n_blobs):
        centre = rng.integers(0, L, size=dim)
        radius = rng.integers(max(1, L // 8), max(2, L // 3))
        d2 = np.zeros((L,) * dim, dtype=np.int64)
        for k in range(dim):
            dk = np.abs(grid[k] - centre[k])
            dk = np.minimum(dk, L - dk)
            d2 += dk * dk
        s[d2 <= radius * radius] *= -1
    return s.reshape(-1)
