"""Shared driver of the GPU-vs-oracle parity tests: same seeded inputs to both sides, bit-exact comparison."""
import numpy as np

import oracle
from paper_1110_0899_b200 import binding


def make_pair(dim, L, J, T, seed, start=None, options=None):
    gpu = binding.Wolff(dim, L, J, T, seed)
    ref = oracle.OracleWolff(dim, L, J, T, seed)
    # reading R7: both sides compute the integer threshold independently; compare it before anything else
    assert gpu.threshold == ref.threshold, (gpu.threshold, ref.threshold)
    if start is not None:
        gpu.set_spins(start)
        ref.set_spins(start)
    for k, v in (options or {}).items():
        gpu.set_option(k, v)
    return gpu, ref


def assert_same_state(gpu, ref, what=""):
    a, b = gpu.get_spins(), ref.get_spins()
    if not np.array_equal(a, b):
        bad = np.nonzero(a != b)[0]
        raise AssertionError("%s lattices differ at %d sites, first %s" % (what, bad.size, bad[:8]))
    assert gpu.observables() == ref.observables(), what
    assert gpu.update_index == ref.update_index, what


def compare_stepwise(gpu, ref, n_updates, lattice_every=0):
    """run(1) + observables on both sides after EVERY update: sizes, E, M bit-exact."""
    for k in range(n_updates):
        gpu.run(1)
        E, M, sz = gpu.observables(sizes=True)
        rs = ref.run(1)
        rE, rM = ref.observables()
        assert sz.tolist() == rs.tolist(), "cluster size differs at update %d: gpu %s oracle %s" % (k, sz, rs)
        assert (E, M) == (rE, rM), "E/M differ at update %d" % k
        if lattice_every and (k + 1) % lattice_every == 0:
            assert_same_state(gpu, ref, "after update %d" % k)
    assert_same_state(gpu, ref, "final")


def compare_batched(gpu, ref, batches):
    """run(n) as one persistent launch per batch; per-update sizes, then E, M and the lattice after each batch."""
    for n in batches:
        gpu.run(n)
        E, M, sz = gpu.observables(sizes=True)
        rs = ref.run(n)
        if not np.array_equal(sz, rs):
            k = int(np.nonzero(sz != rs)[0][0])
            raise AssertionError("cluster size differs at update %d of batch %d: gpu %d oracle %d" % (k, n, sz[k], rs[k]))
        assert (E, M) == ref.observables()
        assert_same_state(gpu, ref, "after batch of %d" % n)
