"""Parity at PROTOCOL LENGTH on the full-size BASELINE configs, in the launch configuration bench.py times.

north_star: "match the oracle bit-exactly (spin lattices, per-update cluster sizes and integer E and M after every
update) ... on every config".  test_gpu_parity.py covers every kernel variant on short chains; here the default
kernel runs BASELINE.json's protocol -- cold start (the bench's 'equilibrated' variant) or the
literal random start, run(1000), then the bench's batches -- and every cluster size, E, M and the whole lattice are
compared with the oracle after each batch: the regime the bench times (T_c-sized fractal clusters, bond tables
double-buffered across thousands of updates, 148 CTAs x 28 tile slots).  The oracle chains are computed by
tests/protocol_farm.py in background threads while the other GPU tests run.
"""
import hashlib
import json
import os

import numpy as np
import pytest
import torch

import protocol_farm as farm
from paper_1110_0899_b200 import binding, workloads as wl

pytestmark = pytest.mark.gpu


def open_chain(name, options=None):
    job = farm.JOBS[name]
    c = wl.CONFIGS[job["cfg"]]
    seed = c.seed if job["seed"] is None else job["seed"]
    gpu = binding.Wolff(c.dim, c.L, c.J, c.T, seed)
    for k, v in (options or {}).items():
        gpu.set_option(k, v)
    if job["cold"]:
        gpu.set_spins(wl.cold(c.N))
    return gpu, c


def check_batch(gpu, c, b, what, lattice_dev):
    E, M, sz = gpu.observables(sizes=True)
    if not np.array_equal(sz, b["sizes"]):
        k = int(np.nonzero(sz != b["sizes"])[0][0])
        raise AssertionError("%s: cluster size differs at update %d of the batch: gpu %d oracle %d" % (what, k, sz[k], b["sizes"][k]))
    assert (E, M) == (b["E"], b["M"]), "%s: E/M differ: gpu %s oracle %s" % (what, (E, M), (b["E"], b["M"]))
    gpu.get_spins_into(lattice_dev)
    bits = farm.pack(lattice_dev.cpu().numpy())
    if not np.array_equal(bits, b["bits"]):
        raise AssertionError("%s: lattices differ in %d bytes of the bit image" % (what, int((bits != b["bits"]).sum())))
    assert gpu.update_index == b["u"]


@pytest.mark.parametrize("name", ["C2", "C4", "C5b", "C5b-literal", "C2-literal", "C3-literal", "C4-literal", "C5a-literal", "C5a", "C3"])
def test_protocol_batches(name):
    gpu, c = open_chain(name)
    stream = torch.cuda.Stream()
    lattice_dev = torch.empty(c.N, dtype=torch.int8, device="cuda")
    ref = farm.result(name)
    assert gpu.threshold == ref["threshold"]
    total = 0
    for k, b in enumerate(ref["batches"]):
        gpu.run(b["n"], stream=stream)           # one persistent launch per batch, as bench.py does
        check_batch(gpu, c, b, "%s batch %d (updates %d..%d)" % (name, k, total, total + b["n"] - 1), lattice_dev)
        total += b["n"]
    gpu.close()


@pytest.mark.parametrize("name", ["C5a", "C3-stretch"])
def test_protocol_energy_and_magnetisation_after_every_update(name):
    # the paper's '+ measurement' protocol on the equilibrated chain: run(1) + observables
    gpu, c = open_chain(name)
    ref = farm.result(name)
    for b in ref["batches"]:
        gpu.run(b["n"])
    E, M = gpu.observables()
    assert (E, M) == (ref["batches"][-1]["E"], ref["batches"][-1]["M"])
    st = ref["stretch"]
    for k in range(len(st["sizes"])):
        gpu.run(1)
        E, M, sz = gpu.observables(sizes=True)
        assert int(sz[0]) == int(st["sizes"][k]), "cluster size differs at stretch update %d" % k
        assert (E, M) == (int(st["E"][k]), int(st["M"][k])), "E/M differ at stretch update %d" % k
    assert np.array_equal(farm.pack(gpu.get_spins()), st["bits"])
    assert gpu.update_index == st["u"]
    gpu.close()


# ------------------------------------------------------------------ the whole protocol, and the region bench.py times
# tests/golden/protocol_digests.json is written by tests/golden/make_protocol_digests.py from the oracle alone: the
# equilibrated chains (cold start) of C3, C5a and C2 over run(1000) + 24 x run(500) = updates 0 .. 12,999, which contains
# BASELINE.json's 1,000 + 10,000 and the updates bench.py times (2,500 .. 12,499 with its 3 warm-up steps), in the
# bench's launch shape.  After every launch: E, M, the update index, the sum and the SHA-256 of the launch's cluster
# sizes, the SHA-256 of the lattice as one bit per spin.
DIGESTS_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "protocol_digests.json")


def _digests():
    with open(DIGESTS_PATH) as f:
        return json.load(f)


def _digest_chains():
    """The chains the golden file holds (C3 takes the oracle about 1.5 hours of one host core; C5a and C2 minutes)."""
    have = _digests() if os.path.exists(DIGESTS_PATH) else {}
    return [name for name in ("C2", "C5a", "C3") if name in have]


def test_the_golden_file_holds_the_secondary_headline_chain():
    assert {"C2", "C5a"} <= set(_digest_chains())


@pytest.mark.parametrize("chain", _digest_chains())
def test_whole_protocol_against_the_oracle_digests(chain):
    d = _digests()[chain]
    c = wl.CONFIGS[chain]
    assert (d["dim"], d["L"], d["J"], d["T"], d["seed"]) == (c.dim, c.L, c.J, c.T, c.seed)
    assert len(d["batches"]) == len(d["checkpoints"]) and sum(d["batches"]) >= c.n_equil + c.n_meas
    gpu = binding.Wolff(c.dim, c.L, c.J, c.T, c.seed)
    assert gpu.threshold == d["threshold"]
    gpu.set_spins(wl.cold(c.N))
    stream = torch.cuda.Stream()
    lattice_dev = torch.empty(c.N, dtype=torch.int8, device="cuda")
    for k, (n, cp) in enumerate(zip(d["batches"], d["checkpoints"])):
        what = "%s launch %d (updates %d..%d)" % (chain, k, cp["u"] - n, cp["u"] - 1)
        gpu.run(n, stream=stream)                 # one persistent launch, as bench.py does
        E, M, sz = gpu.observables(sizes=True)
        assert int(sz.astype(np.int64).sum()) == cp["flipped"], what + ": flipped spins"
        assert hashlib.sha256(np.ascontiguousarray(sz, dtype="<u4").tobytes()).hexdigest() == cp["sizes_sha256"], what + ": cluster sizes"
        assert (E, M) == (cp["E"], cp["M"]), what + ": E/M"
        gpu.get_spins_into(lattice_dev)
        bits = np.packbits(lattice_dev.cpu().numpy().reshape(-1) > 0)
        assert hashlib.sha256(bits.tobytes()).hexdigest() == cp["lattice_sha256"], what + ": lattice"
        assert gpu.update_index == cp["u"], what
    gpu.close()
