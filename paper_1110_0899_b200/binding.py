"""ctypes binding of include/wolff.h -- argument marshalling only; every step runs in the CUDA library.

PyTorch appears here only as a source of device pointers (`tensor.data_ptr()`) and streams
(`torch.cuda.current_stream().cuda_stream`).  If `libwolff_b200.so` is missing this module raises; there is no
CPU fallback.
"""
from __future__ import annotations

import ctypes
import os
import threading

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
# WOLFF_B200_LIB: another build of the same library (the bounds-checked one: `python -m paper_1110_0899_b200.build --checked`)
LIB_PATH = os.environ.get("WOLFF_B200_LIB") or os.path.join(HERE, "libwolff_b200.so")

WOLFF_OK, WOLFF_EINVAL, WOLFF_ENOMEM, WOLFF_ECUDA, WOLFF_EINTERNAL = 0, -1, -2, -3, -4
NSTATS = 16
STAT_NAMES = ("updates", "flipped", "levels_cta", "levels_cluster", "levels_grid", "cluster_wakeups",
              "levels_rebalanced", "claim_attempts", "widest_frontier", "monitor_polls",
              "inline_passes", "messages", "ring_pushes", "warp_passes", "spills", "fill_chunks")

# every symbol include/wolff.h declares (tests/test_abi.py checks the header against this table)
_SIGNATURES = {
    "wolff_create": (ctypes.c_void_p, [ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_uint64]),
    "wolff_run": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p]),
    "wolff_observables": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "wolff_get_spins": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "wolff_set_spins": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "wolff_get_state": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64)]),
    "wolff_set_update_index": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_uint64]),
    "wolff_set_option": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_char_p, ctypes.c_int64]),
    "wolff_get_series": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "wolff_get_moments": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_double)]),
    "wolff_reset_moments": (ctypes.c_int, [ctypes.c_void_p]),
    "wolff_get_stats": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint64)]),
    "wolff_microbench": (ctypes.c_int, [ctypes.POINTER(ctypes.c_double), ctypes.c_int]),
    "wolff_destroy": (ctypes.c_int, [ctypes.c_void_p]),
    "wolff_batch_create": (ctypes.c_void_p, [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                             ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_uint64)]),
    "wolff_batch_run": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p]),
    "wolff_batch_observables": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "wolff_batch_get_spins": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "wolff_batch_set_spins": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "wolff_batch_get_state": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64)]),
    "wolff_batch_set_update_index": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_uint64]),
    "wolff_batch_set_option": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_char_p, ctypes.c_int64]),
    "wolff_batch_get_series": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "wolff_batch_get_moments": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_double)]),
    "wolff_batch_reset_moments": (ctypes.c_int, [ctypes.c_void_p]),
    "wolff_batch_get_stats": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint64)]),
    "wolff_batch_destroy": (ctypes.c_int, [ctypes.c_void_p]),
    "wolff_energy_magnetisation_noalloc": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                                         ctypes.c_void_p, ctypes.c_void_p]),
    "wolff_last_error": (ctypes.c_char_p, []),
}
NOALLOC_MAX_SITES = 1 << 28

_lock = threading.Lock()
_lib = None


class WolffError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__("wolff error %d: %s" % (code, message))
        self.code = code


def load() -> ctypes.CDLL:
    """Load libwolff_b200.so (built in-tree by `paper_1110_0899_b200.build`).  Fails loudly when absent."""
    global _lib
    with _lock:
        if _lib is None:
            if not os.path.exists(LIB_PATH):
                raise ImportError(
                    "%s is missing: build it with `python -m paper_1110_0899_b200.build` "
                    "(needs nvcc; there is no CPU fallback)" % LIB_PATH)
            lib = ctypes.CDLL(LIB_PATH)
            for name, (restype, argtypes) in _SIGNATURES.items():
                fn = getattr(lib, name)        # AttributeError if the symbol is not exported
                fn.restype, fn.argtypes = restype, argtypes
            _lib = lib
        return _lib


def last_error() -> str:
    return load().wolff_last_error().decode()


def _ptr(buf):
    """Raw address of a torch tensor (host or device), a numpy array, an int address, or None."""
    if buf is None:
        return None
    if isinstance(buf, int):
        return buf
    if isinstance(buf, np.ndarray):
        return buf.ctypes.data
    if hasattr(buf, "data_ptr"):
        return buf.data_ptr()
    raise TypeError("expected a torch tensor, numpy array, int address or None")


def _stream_handle(stream):
    if stream is None:
        return None
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream            # torch.cuda.Stream


MICRO_NAMES = ("l2_load_lane_ns", "l2_load_warp_ns", "l2_atomic_lane_ns", "l2_atomic_warp_ns", "syncthreads_ns",
               "philox_x3_ns", "grid_barrier_ns", "smem_pass_floor_ns", "smem_pass_win_fraction",
               "dsmem_load_lane_ns", "dsmem_atomic_lane_ns", "dsmem_atomic_warp_ns", "dsmem_store_to_poll_ns")


def microbench() -> dict:
    """wolff_microbench: the dependent latencies that bound one BFS level (nanoseconds)."""
    buf = (ctypes.c_double * len(MICRO_NAMES))()
    rc = load().wolff_microbench(buf, len(MICRO_NAMES))
    if rc != WOLFF_OK:
        raise WolffError(rc, "wolff_microbench failed")
    return dict(zip(MICRO_NAMES, (float(x) for x in buf)))


def energy_magnetisation_noalloc(spins, dim: int, L: int, E_out=None, M_out=None, stream=None):
    """wolff_energy_magnetisation_noalloc: E and M of a lattice the caller already holds on the current device, for
    programs that cannot let the library allocate there (the card belongs to their own arena, their memory budget is
    fixed after start-up, or a cudaMalloc would stall their other streams).  `spins`: device tensor (or address) of
    L**dim int8 values +1 / -1; `E_out`, `M_out`: one int64 each in device, managed or pinned host memory, either may be
    None.  Nothing is allocated and nothing is waited for: the values are there once `stream` has run the kernel.  At
    most NOALLOC_MAX_SITES sites; calls that can overlap on the GPU race on the shared scratch memory (see wolff.h)."""
    rc = load().wolff_energy_magnetisation_noalloc(_ptr(spins), int(dim), int(L), _ptr(E_out), _ptr(M_out), _stream_handle(stream))
    if rc != WOLFF_OK:
        raise WolffError(rc, last_error())


class Wolff:
    """One Wolff single-cluster chain on the current CUDA device (wolff_create .. wolff_destroy)."""

    def __init__(self, dim: int, L: int, J: float, T: float, seed: int):
        self._lib = load()
        self._h = self._lib.wolff_create(int(dim), int(L), float(J), float(T), int(seed))
        if not self._h:
            raise WolffError(WOLFF_EINVAL, last_error())
        self.dim, self.L, self.N = int(dim), int(L), int(L) ** int(dim)
        self.last_n = 0

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            self._lib.wolff_destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != WOLFF_OK:
            raise WolffError(rc, last_error())

    # -- the four calls north_star names
    def run(self, n_updates: int, stream=None):
        """wolff_run: enqueue n_updates updates on `stream` (torch.cuda.Stream, raw handle or None) and return."""
        self._check(self._lib.wolff_run(self._h, int(n_updates), _stream_handle(stream)))
        if n_updates:
            self.last_n = int(n_updates)

    def observables_into(self, E=None, M=None, cluster_sizes=None):
        """wolff_observables with caller-owned buffers (torch tensors on host/device, numpy arrays, or None)."""
        self._check(self._lib.wolff_observables(self._h, _ptr(E), _ptr(M), _ptr(cluster_sizes)))

    def observables(self, sizes: bool = False):
        """(E, M) of the current lattice, plus the last run's cluster sizes when sizes=True (numpy, host)."""
        em = np.zeros(2, dtype=np.int64)
        out = np.empty(self.last_n, dtype=np.uint32) if sizes and self.last_n else None
        self._check(self._lib.wolff_observables(self._h, em.ctypes.data, em.ctypes.data + 8, _ptr(out)))
        if sizes:
            return int(em[0]), int(em[1]), (out if out is not None else np.empty(0, dtype=np.uint32))
        return int(em[0]), int(em[1])

    def get_spins_into(self, dst):
        self._check(self._lib.wolff_get_spins(self._h, _ptr(dst)))

    def get_spins(self) -> np.ndarray:
        out = np.empty(self.N, dtype=np.int8)
        self.get_spins_into(out)
        return out

    # -- hooks
    def set_spins(self, src):
        if isinstance(src, np.ndarray):
            src = np.ascontiguousarray(src, dtype=np.int8).reshape(-1)
            if src.size != self.N:
                raise ValueError("need N = %d spins" % self.N)
        self._check(self._lib.wolff_set_spins(self._h, _ptr(src)))

    @property
    def update_index(self) -> int:
        u = ctypes.c_uint64()
        self._check(self._lib.wolff_get_state(self._h, ctypes.byref(u), None))
        return int(u.value)

    @update_index.setter
    def update_index(self, u: int):
        self._check(self._lib.wolff_set_update_index(self._h, int(u)))

    @property
    def threshold(self) -> int:
        t = ctypes.c_uint64()
        self._check(self._lib.wolff_get_state(self._h, None, ctypes.byref(t)))
        return int(t.value)

    def set_option(self, key: str, value: int):
        self._check(self._lib.wolff_set_option(self._h, key.encode(), int(value)))

    # -- in-kernel measurement (set_option("measure", 1))
    def series_into(self, E=None, M=None, update_ns=None):
        """wolff_get_series with caller-owned buffers (host or device)."""
        self._check(self._lib.wolff_get_series(self._h, _ptr(E), _ptr(M), _ptr(update_ns)))

    def series(self):
        """(E, M) after every update of the most recent (measured) run, numpy int64 arrays on the host."""
        E = np.empty(self.last_n, dtype=np.int64)
        M = np.empty(self.last_n, dtype=np.int64)
        if self.last_n:
            self.series_into(E, M, None)
        return E, M

    def update_ns(self) -> np.ndarray:
        """Duration of every update of the most recent run in nanoseconds, as the kernel saw it."""
        ns = np.empty(self.last_n, dtype=np.uint32)
        if self.last_n:
            self.series_into(None, None, ns)
        return ns

    def moments(self):
        """(ten raw 64-bit words, Binder ratio): wolff_get_moments."""
        buf = (ctypes.c_uint64 * 10)()
        U = ctypes.c_double()
        self._check(self._lib.wolff_get_moments(self._h, buf, ctypes.byref(U)))
        return np.array([int(x) for x in buf], dtype=np.uint64), float(U.value)

    def reset_moments(self):
        self._check(self._lib.wolff_reset_moments(self._h))

    def stats(self) -> dict:
        buf = (ctypes.c_uint64 * NSTATS)()
        self._check(self._lib.wolff_get_stats(self._h, buf))
        return dict(zip(STAT_NAMES, (int(x) for x in buf)))


BATCH_STAT_NAMES = ("updates", "flipped", "levels", "claim_attempts")


class WolffBatch:
    """R independent chains of one shape in one launch (wolff_batch_create .. wolff_batch_destroy)."""

    def __init__(self, dim: int, L: int, J, T, seed):
        self._lib = load()
        T = [float(t) for t in np.atleast_1d(T)]
        R = len(T)
        J = [float(j) for j in np.broadcast_to(np.atleast_1d(J), (R,))]
        seed = [int(x) for x in np.broadcast_to(np.atleast_1d(np.asarray(seed, dtype=np.uint64)), (R,))]
        self._h = self._lib.wolff_batch_create(int(dim), int(L), R, (ctypes.c_double * R)(*J), (ctypes.c_double * R)(*T),
                                               (ctypes.c_uint64 * R)(*seed))
        if not self._h:
            raise WolffError(WOLFF_EINVAL, last_error())
        self.dim, self.L, self.N, self.R = int(dim), int(L), int(L) ** int(dim), R
        self.last_n = 0

    def close(self):
        if getattr(self, "_h", None):
            self._lib.wolff_batch_destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != WOLFF_OK:
            raise WolffError(rc, last_error())

    def run(self, n_updates: int, stream=None):
        self._check(self._lib.wolff_batch_run(self._h, int(n_updates), _stream_handle(stream)))
        if n_updates:
            self.last_n = int(n_updates)

    def observables_into(self, E=None, M=None, cluster_sizes=None):
        self._check(self._lib.wolff_batch_observables(self._h, _ptr(E), _ptr(M), _ptr(cluster_sizes)))

    def observables(self, sizes: bool = False):
        """(E[R], M[R]) of the current lattices, plus sizes[R, n] of the most recent run when sizes=True."""
        E = np.zeros(self.R, dtype=np.int64)
        M = np.zeros(self.R, dtype=np.int64)
        out = np.empty((self.R, self.last_n), dtype=np.uint32) if sizes and self.last_n else None
        self.observables_into(E, M, out)
        if sizes:
            return E, M, (out if out is not None else np.empty((self.R, 0), dtype=np.uint32))
        return E, M

    def get_spins_into(self, dst):
        self._check(self._lib.wolff_batch_get_spins(self._h, _ptr(dst)))

    def get_spins(self) -> np.ndarray:
        out = np.empty((self.R, self.N), dtype=np.int8)
        self.get_spins_into(out)
        return out

    def set_spins(self, src):
        if isinstance(src, np.ndarray):
            src = np.ascontiguousarray(src, dtype=np.int8).reshape(-1)
            if src.size != self.R * self.N:
                raise ValueError("need R * N = %d spins" % (self.R * self.N))
        self._check(self._lib.wolff_batch_set_spins(self._h, _ptr(src)))

    @property
    def update_index(self) -> int:
        u = ctypes.c_uint64()
        self._check(self._lib.wolff_batch_get_state(self._h, ctypes.byref(u), None))
        return int(u.value)

    @update_index.setter
    def update_index(self, u: int):
        self._check(self._lib.wolff_batch_set_update_index(self._h, int(u)))

    @property
    def thresholds(self) -> np.ndarray:
        buf = (ctypes.c_uint64 * self.R)()
        self._check(self._lib.wolff_batch_get_state(self._h, None, buf))
        return np.array([int(x) for x in buf], dtype=np.uint64)

    def set_option(self, key: str, value: int):
        self._check(self._lib.wolff_batch_set_option(self._h, key.encode(), int(value)))

    def series(self):
        """(E[R, n], M[R, n]) after every update of the most recent measured run."""
        E = np.empty((self.R, self.last_n), dtype=np.int64)
        M = np.empty((self.R, self.last_n), dtype=np.int64)
        self._check(self._lib.wolff_batch_get_series(self._h, _ptr(E), _ptr(M)))
        return E, M

    def moments(self):
        """(raw[R, 10], binder[R]): wolff_batch_get_moments."""
        buf = (ctypes.c_uint64 * (10 * self.R))()
        U = (ctypes.c_double * self.R)()
        self._check(self._lib.wolff_batch_get_moments(self._h, buf, U))
        return (np.array([int(x) for x in buf], dtype=np.uint64).reshape(self.R, 10), np.array([float(x) for x in U]))

    def reset_moments(self):
        self._check(self._lib.wolff_batch_reset_moments(self._h))

    def stats(self) -> dict:
        buf = (ctypes.c_uint64 * 4)()
        self._check(self._lib.wolff_batch_get_stats(self._h, buf))
        return dict(zip(BATCH_STAT_NAMES, (int(x) for x in buf)))
