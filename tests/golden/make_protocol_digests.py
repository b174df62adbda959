#!/usr/bin/env python
"""Writes tests/golden/protocol_digests.json: the oracle's checkpoints over the WHOLE protocol of the equilibrated
headline chains, in the launch shape bench.py times.

    python tests/golden/make_protocol_digests.py [C3 C5a C2 ...]      (about 45 minutes of one core for C3, minutes for the others)

Everything in the file comes from `oracle/` alone (this script imports `oracle` and the shared, arithmetic-free
`workloads` module; nothing of the CUDA path).  BASELINE.json's configs run 1,000 equilibration + 10,000 measured
updates (steps i-v repeated).  bench.py runs them as: cold start, run(1000), W = 3 warm-up
steps and K = 20 timed steps of run(500) each -- updates 2,500 .. 12,499 are the timed region.  The chains here do
run(1000) and then 24 x run(500), i.e. updates 0 .. 12,999, and keep after every batch:
    u               the update index (updates done)
    E, M            integer energy and magnetisation of the lattice (PAPER.md:38 Eq. 2, :126)
    flipped         the sum of the batch's cluster sizes
    sizes_sha256    SHA-256 of the batch's cluster sizes as little-endian uint32
    lattice_sha256  SHA-256 of the lattice as one bit per spin (numpy.packbits of spin > 0; spins are +/-1, so the bits
                    ARE the lattice)
tests/test_gpu_protocol.py replays the same launches through the C-ABI and compares every checkpoint.
"""
from __future__ import annotations

import hashlib
import json
import os
import sys
from concurrent.futures import ThreadPoolExecutor

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle                                            # noqa: E402
from paper_1110_0899_b200 import workloads as wl         # noqa: E402

OUT = os.path.join(HERE, "protocol_digests.json")
BATCHES = [1000] + [500] * 24
JOBS = ("C3", "C5a", "C2")


def lattice_digest(spins: np.ndarray) -> str:
    return hashlib.sha256(np.packbits(np.asarray(spins).reshape(-1) > 0).tobytes()).hexdigest()


def sizes_digest(sizes: np.ndarray) -> str:
    return hashlib.sha256(np.ascontiguousarray(sizes, dtype="<u4").tobytes()).hexdigest()


def run_chain(name: str) -> dict:
    c = wl.CONFIGS[name]
    ref = oracle.OracleWolff(c.dim, c.L, c.J, c.T, c.seed)
    ref.set_spins(wl.cold(c.N))
    out = {"config": c.name, "dim": c.dim, "L": c.L, "J": c.J, "T": c.T, "seed": c.seed, "start": "cold (all +1)",
           "threshold": ref.threshold, "batches": BATCHES, "checkpoints": []}
    for n in BATCHES:
        sizes = ref.run(n)
        E, M = ref.observables()
        out["checkpoints"].append({"u": ref.update_index, "E": E, "M": M, "flipped": int(sizes.astype(np.int64).sum()),
                                   "sizes_sha256": sizes_digest(sizes), "lattice_sha256": lattice_digest(ref.get_spins())})
        sys.stderr.write("%s: %d updates done\n" % (name, ref.update_index))
    ref.close()
    return out


def main(argv):
    names = argv or list(JOBS)
    for n in names:
        if n not in wl.CONFIGS:
            raise SystemExit("unknown config %r" % n)
    data = {}
    if os.path.exists(OUT):
        with open(OUT) as f:
            data = json.load(f)
    with ThreadPoolExecutor(max_workers=len(names)) as pool:          # the ctypes calls into liboracle.so release the GIL
        for name, res in zip(names, pool.map(run_chain, names)):
            data[name] = res
    data["_written_by"] = "tests/golden/make_protocol_digests.py (oracle only)"
    tmp = OUT + ".tmp"
    with open(tmp, "w") as f:
        json.dump(data, f, indent=1, sort_keys=True)
        f.write("\n")
    os.replace(tmp, OUT)


if __name__ == "__main__":
    main(sys.argv[1:])
