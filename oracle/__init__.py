"""CPU oracle for the Wolff single-cluster hot path -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_1110_0899_b200`` (the CUDA path) and never imports it.

The arithmetic lives in plain C (``wolff_oracle.c``: the sequential stack-based
Wolff update of PAPER.md:42-50 with bond-keyed Philox4x32-10; ``ising_enum.c``:
brute-force enumeration used to pin it).  This module only compiles the two
files with gcc and marshals arguments through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SOURCES = ("wolff_oracle.c", "ising_enum.c")
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, no tuning) and return the .so path."""
    srcs = [os.path.join(_HERE, s) for s in _SOURCES]
    if not force and os.path.exists(_LIB_PATH):
        if os.path.getmtime(_LIB_PATH) >= max(os.path.getmtime(s) for s in srcs):
            return _LIB_PATH
    tmp = _LIB_PATH + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-std=c11", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp] + srcs + ["-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


def lib() -> ctypes.CDLL:
    global _lib
    with _lock:
        if _lib is not None:
            return _lib
        L = ctypes.CDLL(build())
        u64, u32, i64, i32, dbl, vp = (ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int64,
                                       ctypes.c_int, ctypes.c_double, ctypes.c_void_p)
        P = ctypes.POINTER
        L.oracle_philox4x32_10.argtypes = [P(u32), P(u32), P(u32)]
        L.oracle_philox4x32_10.restype = None
        L.oracle_threshold.argtypes = [dbl, dbl]
        L.oracle_threshold.restype = u64
        L.oracle_nbr.argtypes = [i32, i32, u64, i32, i32]
        L.oracle_nbr.restype = u64
        L.oracle_site_draw.argtypes = [u64, u64, u64]
        L.oracle_site_draw.restype = u64
        L.oracle_bond_active.argtypes = [u64, u64, u64, i32, u64]
        L.oracle_bond_active.restype = i32
        L.oracle_init_spin.argtypes = [u64, u64]
        L.oracle_init_spin.restype = i32
        L.oracle_create.argtypes = [i32, i32, dbl, dbl, u64]
        L.oracle_create.restype = vp
        L.oracle_destroy.argtypes = [vp]
        L.oracle_destroy.restype = None
        L.oracle_get_spins.argtypes = [vp, vp]
        L.oracle_get_spins.restype = None
        L.oracle_set_spins.argtypes = [vp, vp]
        L.oracle_set_spins.restype = None
        L.oracle_get_threshold.argtypes = [vp]
        L.oracle_get_threshold.restype = u64
        L.oracle_get_update_index.argtypes = [vp]
        L.oracle_get_update_index.restype = u64
        L.oracle_set_update_index.argtypes = [vp, u64]
        L.oracle_set_update_index.restype = None
        L.oracle_observables.argtypes = [vp, P(i64), P(i64)]
        L.oracle_observables.restype = None
        L.oracle_run.argtypes = [vp, u64, vp]
        L.oracle_run.restype = i32
        L.oracle_run_logged.argtypes = [vp, u64, vp, vp, vp]
        L.oracle_run_logged.restype = i32
        L.oracle_moments.argtypes = [u64, vp, vp, vp, vp]
        L.oracle_moments.restype = None
        L.oracle_binder.argtypes = [vp]
        L.oracle_binder.restype = dbl
        L.ising_enum_joint_dos.argtypes = [i32, i32, vp]
        L.ising_enum_joint_dos.restype = i32
        _lib = L
        return L


# ------------------------------------------------------------------ scalar helpers

def philox4x32_10(ctr, key):
    c = (ctypes.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (ctypes.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    out = (ctypes.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, out)
    return tuple(int(x) for x in out)


def threshold(J: float, T: float) -> int:
    return int(lib().oracle_threshold(float(J), float(T)))


def nbr(dim: int, L: int, i: int, d: int, sign: int) -> int:
    return int(lib().oracle_nbr(dim, L, int(i), d, sign))


def site_draw(seed: int, u: int, N: int) -> int:
    return int(lib().oracle_site_draw(int(seed), int(u), int(N)))


def bond_active(seed: int, u: int, owner: int, d: int, thr: int) -> bool:
    return bool(lib().oracle_bond_active(int(seed), int(u), int(owner), d, int(thr)))


def init_spin(seed: int, i: int) -> int:
    return int(lib().oracle_init_spin(int(seed), int(i)))


# ------------------------------------------------------------------ the oracle object

class OracleWolff:
    """Sequential Wolff single-cluster chain; mirrors the C-ABI of include/wolff.h."""

    def __init__(self, dim: int, L: int, J: float, T: float, seed: int):
        self._L = lib()
        self._h = self._L.oracle_create(dim, L, float(J), float(T), int(seed))
        if not self._h:
            raise ValueError("oracle_create rejected (dim=%r, L=%r, J=%r, T=%r)" % (dim, L, J, T))
        self.dim, self.L, self.N = dim, L, L ** dim

    def close(self):
        if getattr(self, "_h", None):
            self._L.oracle_destroy(self._h)
            self._h = None

    __del__ = close

    @property
    def threshold(self) -> int:
        return int(self._L.oracle_get_threshold(self._h))

    @property
    def update_index(self) -> int:
        return int(self._L.oracle_get_update_index(self._h))

    @update_index.setter
    def update_index(self, u: int):
        self._L.oracle_set_update_index(self._h, int(u))

    def run(self, n_updates: int) -> np.ndarray:
        sizes = np.empty(int(n_updates), dtype=np.uint32)
        self._L.oracle_run(self._h, int(n_updates), sizes.ctypes.data)
        return sizes

    def run_logged(self, n_updates: int):
        n = int(n_updates)
        sizes = np.empty(n, dtype=np.uint32)
        E = np.empty(n, dtype=np.int64)
        M = np.empty(n, dtype=np.int64)
        self._L.oracle_run_logged(self._h, n, sizes.ctypes.data, E.ctypes.data, M.ctypes.data)
        return sizes, E, M

    def observables(self):
        E, M = ctypes.c_int64(), ctypes.c_int64()
        self._L.oracle_observables(self._h, ctypes.byref(E), ctypes.byref(M))
        return int(E.value), int(M.value)

    def get_spins(self) -> np.ndarray:
        out = np.empty(self.N, dtype=np.int8)
        self._L.oracle_get_spins(self._h, out.ctypes.data)
        return out

    def set_spins(self, spins):
        a = np.ascontiguousarray(spins, dtype=np.int8).reshape(-1)
        if a.size != self.N or not np.all(np.abs(a) == 1):
            raise ValueError("need N spins of +/-1")
        self._L.oracle_set_spins(self._h, a.ctypes.data)


MOMENT_NAMES = ("n", "sum_E", "sum_absM", "sum_E2", "sum_M2", "sum_M4")


def moments_raw(E, M, acc=None) -> np.ndarray:
    """oracle_moments: the ten 64-bit words (layout in wolff_oracle.c) over the series (E_k, M_k), continuing `acc`."""
    E = np.ascontiguousarray(E, dtype=np.int64)
    M = np.ascontiguousarray(M, dtype=np.int64)
    assert E.shape == M.shape and E.ndim == 1
    out = np.zeros(10, dtype=np.uint64)
    a = None if acc is None else np.ascontiguousarray(acc, dtype=np.uint64)
    lib().oracle_moments(E.size, E.ctypes.data, M.ctypes.data, None if a is None else a.ctypes.data, out.ctypes.data)
    return out


def moments_dict(raw) -> dict:
    """The ten words as exact Python integers."""
    w = [int(x) for x in raw]
    sum_E = w[1] - (1 << 64) if w[1] >> 63 else w[1]
    return {"n": w[0], "sum_E": sum_E, "sum_absM": w[2], "sum_E2": w[3] | (w[4] << 64),
            "sum_M2": w[5] | (w[6] << 64), "sum_M4": w[7] | (w[8] << 64)}


def binder(raw) -> float:
    """oracle_binder: Eq. 3 of the paper from the accumulated sums."""
    a = np.ascontiguousarray(raw, dtype=np.uint64)
    return float(lib().oracle_binder(a.ctypes.data))


def joint_density_of_states(dim: int, L: int) -> np.ndarray:
    """g[E + dim*N, M + N] by brute-force enumeration of all 2^N states (ising_enum.c)."""
    N = L ** dim
    g = np.zeros((2 * dim * N + 1, 2 * N + 1), dtype=np.uint64)
    rc = lib().ising_enum_joint_dos(dim, L, g.ctypes.data)
    if rc != 0:
        raise ValueError("enumeration refused (dim=%d, L=%d)" % (dim, L))
    return g
