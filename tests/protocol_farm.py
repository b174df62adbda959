"""Oracle side of the protocol-length parity tests (tests/test_gpu_protocol.py).

BASELINE.json's configs run 1,000 equilibration + up to 10,000 measured updates; at 2D L=4096 the sequential oracle
needs minutes for that.  The chains below are independent, so they run side by side in threads (the ctypes calls into
oracle/liboracle.so release the GIL) from the moment pytest has collected a protocol test, while the other GPU tests
run.  Everything stored here comes from `oracle/` alone; nothing is taken from the CUDA path.

A job is a chain (config, seed, start) and a list of batches, the launches the bench makes: `run(1000)` for the
equilibration, then batches of the bench's updates-per-step.  Kept per batch: every cluster size, E and M after the
batch, and the whole lattice as one bit per spin (spins are +/-1, so the bits ARE the lattice).  A job may end with a
stretch of single updates with E and M after every one (north_star: "integer E and M after every update").
"""
from __future__ import annotations

import threading
from concurrent.futures import Future, ThreadPoolExecutor

import numpy as np

import oracle
from paper_1110_0899_b200 import workloads as wl

# name -> config, seed (None = the config's), cold start?, batches, stretch of single logged updates at the end
JOBS = {
    # the bench's primary leg: C3 equilibrated variant, run(1000) then the first timed batches
    "C3": dict(cfg="C3", seed=None, cold=True, batches=[1000, 300], stretch=0),
    # E and M after every update on C3 once the chain is stationary (a few hundred updates after a cold start)
    "C3-stretch": dict(cfg="C3", seed=2, cold=True, batches=[300], stretch=200),
    # the bench's secondary leg: C5a, run(1000) then batches of 1000; then a stretch of single updates
    "C5a": dict(cfg="C5a", seed=None, cold=True, batches=[1000, 1000, 1000, 1000], stretch=200),
    "C2": dict(cfg="C2", seed=None, cold=True, batches=[1000, 1000, 1000, 1000], stretch=0),
    # the full 1,000 + 10,000 of BASELINE.json
    "C4": dict(cfg="C4", seed=None, cold=True, batches=[1000] + [1000] * 10, stretch=0),
    "C5b": dict(cfg="C5b", seed=None, cold=True, batches=[1000, 10000], stretch=0),
    "C5b-literal": dict(cfg="C5b", seed=None, cold=False, batches=[1000, 10000], stretch=0),
    "C2-literal": dict(cfg="C2", seed=None, cold=False, batches=[1000, 10000], stretch=0),
    # BASELINE.json's configs 3-5 exactly as written (random start from the seed, 1,000 + 10,000 updates): the clusters
    # stay at a handful of spins, so the oracle needs about a second per chain
    "C3-literal": dict(cfg="C3", seed=None, cold=False, batches=[1000, 10000], stretch=0),
    "C4-literal": dict(cfg="C4", seed=None, cold=False, batches=[1000, 10000], stretch=0),
    "C5a-literal": dict(cfg="C5a", seed=None, cold=False, batches=[1000, 10000], stretch=0),
}

_lock = threading.Lock()
_futures: dict[str, Future] = {}
_pool: ThreadPoolExecutor | None = None


def pack(spins: np.ndarray) -> np.ndarray:
    return np.packbits(np.asarray(spins).reshape(-1) > 0)


def _run_job(name: str) -> dict:
    job = JOBS[name]
    c = wl.CONFIGS[job["cfg"]]
    seed = c.seed if job["seed"] is None else job["seed"]
    ref = oracle.OracleWolff(c.dim, c.L, c.J, c.T, seed)
    if job["cold"]:
        ref.set_spins(wl.cold(c.N))
    out = {"threshold": ref.threshold, "batches": [], "stretch": None, "seed": seed}
    for n in job["batches"]:
        sizes = ref.run(n)
        E, M = ref.observables()
        out["batches"].append({"n": n, "sizes": sizes, "E": E, "M": M, "bits": pack(ref.get_spins()), "u": ref.update_index})
    if job["stretch"]:
        sizes, E, M = ref.run_logged(job["stretch"])
        out["stretch"] = {"sizes": sizes, "E": E, "M": M, "bits": pack(ref.get_spins()), "u": ref.update_index}
    ref.close()
    return out


def start(names=None):
    """Start the oracle chains (idempotent).  The longest job goes first."""
    global _pool
    with _lock:
        if _pool is None:
            _pool = ThreadPoolExecutor(max_workers=len(JOBS), thread_name_prefix="oracle-protocol")
        for name in (names or JOBS):
            if name not in _futures:
                _futures[name] = _pool.submit(_run_job, name)


def result(name: str) -> dict:
    start([name])
    return _futures[name].result()
