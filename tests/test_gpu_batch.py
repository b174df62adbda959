"""A batch of independent chains in one launch (wolff_batch_*) against the oracle: every replica must equal ITS OWN
single-chain oracle bit for bit -- lattice, per-update cluster sizes, E and M (and, measured, E and M after every
update and the accumulated moments).  The sweeps over T (and L) of PAPER.md:149-168, Figs. 1-2, are what the batch is
for, so the replicas below differ in temperature and seed."""
import numpy as np
import pytest

import oracle
from paper_1110_0899_b200 import binding, workloads as wl

pytestmark = pytest.mark.gpu


def make_batch(dim, L, T, seeds, J=1.0, options=None, start=None):
    gpu = binding.WolffBatch(dim, L, J, T, seeds)
    J = np.broadcast_to(np.atleast_1d(J), (gpu.R,))
    refs = [oracle.OracleWolff(dim, L, float(J[r]), float(T[r]), int(seeds[r])) for r in range(gpu.R)]
    assert gpu.thresholds.tolist() == [r.threshold for r in refs]        # reading R7, compared first
    for k, v in (options or {}).items():
        gpu.set_option(k, v)
    if start is not None:
        gpu.set_spins(start)
        for r, ref in enumerate(refs):
            ref.set_spins(start[r])
    return gpu, refs


def assert_same_lattices(gpu, refs, what=""):
    spins = gpu.get_spins()
    E, M = gpu.observables()
    for r, ref in enumerate(refs):
        if not np.array_equal(spins[r], ref.get_spins()):
            raise AssertionError("%s: lattice of chain %d differs" % (what, r))
        assert (int(E[r]), int(M[r])) == ref.observables(), "%s: E/M of chain %d" % (what, r)
    assert gpu.update_index == refs[0].update_index


def compare(gpu, refs, batches, measured=False, acc=None):
    acc = acc if acc is not None else [None] * gpu.R
    for n in batches:
        gpu.run(n)
        _, _, sz = gpu.observables(sizes=True)
        if measured:
            Es, Ms = gpu.series()
            raw, U = gpu.moments()
        for r, ref in enumerate(refs):
            if measured:
                rs, rE, rM = ref.run_logged(n)
                assert np.array_equal(Es[r], rE), "E series of chain %d" % r
                assert np.array_equal(Ms[r], rM), "M series of chain %d" % r
                acc[r] = oracle.moments_raw(rE, rM, acc=acc[r])
                assert np.array_equal(raw[r], acc[r]), "moments of chain %d" % r
                Uo = oracle.binder(acc[r])
                assert (np.isnan(U[r]) and np.isnan(Uo)) or abs(U[r] - Uo) < 1e-12
            else:
                rs = ref.run(n)
            if not np.array_equal(sz[r], rs):
                k = int(np.nonzero(sz[r] != rs)[0][0])
                raise AssertionError("chain %d: cluster size differs at update %d: gpu %d oracle %d" % (r, k, sz[r][k], rs[k]))
        assert_same_lattices(gpu, refs, "after a batch of %d" % n)
    return acc


def sweep(R, lo, hi):
    return [lo + (hi - lo) * r / max(R - 1, 1) for r in range(R)]


# where a chain's lattice lives during its turn: the int8 lattice in global memory, or bit-packed in shared memory
RESIDENT = [1, 2]


@pytest.mark.parametrize("resident", RESIDENT)
@pytest.mark.parametrize("measured", [False, True])
@pytest.mark.parametrize("dim,L,Tlo,Thi", [(2, 32, 1.8, 3.2), (3, 12, 3.8, 5.4), (2, 20, 2.0, 2.6), (3, 8, 4.2, 4.8)])
def test_temperature_sweep_of_160_replicas(dim, L, Tlo, Thi, measured, resident):
    # more replicas than SMs: every CTA slot of the chip is in use, chains queue for CTAs; one T and seed per replica
    R = 160
    T = sweep(R, Tlo, Thi)
    seeds = [1000 + 7 * r for r in range(R)]
    gpu, refs = make_batch(dim, L, T, seeds, options={"measure": int(measured), "resident": resident})
    assert_same_lattices(gpu, refs, "start lattices (reading R9)")
    compare(gpu, refs, [1, 40, 200], measured=measured)
    gpu.close()


@pytest.mark.parametrize("options", [{"threads": 32}, {"threads": 64, "queue_cap": 8}, {"threads": 128, "queue_cap": 8, "measure": 1},
                                      {"threads": 256, "measure": 1}, {"threads": 32, "queue_cap": 16, "measure": 1},
                                      {"threads": 32, "resident": 2}, {"threads": 64, "queue_cap": 8, "resident": 2, "measure": 1},
                                      {"threads": 256, "resident": 2, "measure": 1}, {"threads": 128, "queue_cap": 8, "resident": 1}])
def test_launch_shapes_and_tiny_frontier_buffers(options):
    # queue_cap 8: every level wider than 8 sites is read back from the member list in global memory
    R = 24
    gpu, refs = make_batch(2, 48, sweep(R, 1.9, 2.5), [5 + r for r in range(R)], options=options,
                           start=np.stack([wl.cold(48 * 48) if r % 2 else wl.blobs(2, 48, seed=r) for r in range(R)]))
    compare(gpu, refs, [3, 60], measured=bool(options.get("measure")))
    gpu.close()


@pytest.mark.parametrize("resident", RESIDENT)
@pytest.mark.parametrize("measured", [False, True])
def test_wide_frontiers_p_one_and_p_zero(measured, resident):
    # chain 0: p = 1 from a cold start (the first cluster is the whole lattice); chain 1: p = 0 (only the seed flips);
    # chain 2: T_c; non-power-of-two L
    for dim, L in [(2, 100), (3, 20)]:
        N = L ** dim
        gpu, refs = make_batch(dim, L, [0.04, 1.0, wl.TC_2D if dim == 2 else wl.TC_3D], [3, 4, 5], J=[1.0, 0.0, 1.0],
                               options={"measure": int(measured), "resident": resident}, start=np.stack([wl.cold(N)] * 3))
        assert gpu.thresholds.tolist()[:2] == [1 << 32, 0]
        compare(gpu, refs, [1, 2, 10], measured=measured)
        gpu.close()


@pytest.mark.parametrize("resident", RESIDENT)
def test_medium_lattices_equilibrated_variant(resident):
    # C2-sized chains from a cold start: frontiers of hundreds of sites, clusters of 10^5..10^6 spins, in one CTA each.
    # resident 2: the 128 KiB sign plane of 2D L=1024 fills one SM's shared memory; the mark plane
    # of a measured run does not fit beside it, so the measured part runs 3D L=64 (two planes of 32 KiB)
    c = wl.CONFIGS["C2"]
    R = 3
    gpu, refs = make_batch(c.dim, c.L, [c.T, 2.2, 2.35], [1, 2, 3], start=np.stack([wl.cold(c.N)] * R), options={"resident": resident})
    compare(gpu, refs, [1, 12])
    if resident == 2:
        gpu.set_option("measure", 1)
        with pytest.raises(binding.WolffError):
            gpu.run(1)
        gpu.close()
        gpu, refs = make_batch(3, 64, [wl.TC_3D, 4.3, 4.7], [1, 2, 3], start=np.stack([wl.cold(64 ** 3)] * R), options={"resident": 2, "measure": 1})
        compare(gpu, refs, [2, 30], measured=True)
    else:
        gpu.set_option("measure", 1)
        compare(gpu, refs, [6], measured=True)
    gpu.close()


@pytest.mark.parametrize("dim,L,Tlo,Thi", [(2, 32, 1.8, 3.2), (3, 12, 3.8, 5.4), (2, 20, 2.0, 2.6), (3, 16, 4.2, 4.8)])
def test_one_cluster_per_chain_sweep(dim, L, Tlo, Thi):
    # "resident" = 3: every chain is grown by its own thread-block cluster (the cluster-resident bit-packed kernel), the
    # launches side by side on the library's streams; 40 replicas with their own T and seed, L a power of two and not
    R = 40
    gpu, refs = make_batch(dim, L, sweep(R, Tlo, Thi), [2000 + 3 * r for r in range(R)], options={"resident": 3})
    assert_same_lattices(gpu, refs, "start lattices (reading R9)")
    compare(gpu, refs, [1, 40, 200])
    st = gpu.stats()
    assert st["updates"] == R * 200
    gpu.set_option("measure", 1)
    if L % 32 == 0:
        acc = compare(gpu, refs, [2, 50], measured=True)          # E and M after every update, moments, Binder ratio
        gpu.set_option("resident", 1)                # the same chains continue on another kernel, the sums run on
        compare(gpu, refs, [30], measured=True, acc=acc)
    else:
        with pytest.raises(binding.WolffError):
            gpu.run(1)                               # this residency measures only when L is a multiple of 32
        gpu.set_option("measure", 0)
        gpu.set_option("resident", 1)
        compare(gpu, refs, [30])
    gpu.close()


def test_one_cluster_per_chain_full_size():
    # C5a-sized chains at T_c from a cold start (clusters of 10^5 .. 10^7 spins, 16 CTAs per chain, 7 chains side by side)
    # and p = 1 / p = 0 chains on a lattice that is not a power of two
    import torch
    c = wl.CONFIGS["C5a"]
    R = 9
    gpu, refs = make_batch(c.dim, c.L, [c.T] * R, [c.seed + r for r in range(R)], options={"resident": 3},
                           start=np.stack([wl.cold(c.N)] * R))
    gpu.run(3, stream=torch.cuda.Stream())
    _, _, sz = gpu.observables(sizes=True)
    for r, ref in enumerate(refs):
        assert np.array_equal(sz[r], ref.run(3))
    assert_same_lattices(gpu, refs, "C5a x 9")
    gpu.close()
    N = 100 * 100
    gpu, refs = make_batch(2, 100, [0.04, 1.0, wl.TC_2D], [3, 4, 5], J=[1.0, 0.0, 1.0], options={"resident": 3}, start=np.stack([wl.cold(N)] * 3))
    compare(gpu, refs, [1, 2, 10])
    gpu.close()


def test_split_runs_index_jumps_and_bad_input():
    R = 5
    T = sweep(R, 2.0, 2.6)
    seeds = [(0xABCDEF << 32) | r for r in range(R)]
    a, refs = make_batch(2, 16, T, seeds)
    b, _ = make_batch(2, 16, T, seeds)
    a.run(7); a.run(13); b.run(20)
    for ref in refs:
        ref.run(20)
    assert np.array_equal(a.get_spins(), b.get_spins())
    assert_same_lattices(a, refs)
    a.update_index = (1 << 40) + 99
    for ref in refs:
        ref.update_index = (1 << 40) + 99
    compare(a, refs, [30])
    bad = a.get_spins().copy()
    bad[3, 17] = 0
    with pytest.raises(binding.WolffError):
        a.set_spins(bad)
    assert_same_lattices(a, refs, "a rejected set_spins leaves the lattices alone")
    with pytest.raises(binding.WolffError):
        a.series()                                   # not a measured run
    a.close(); b.close()


def test_full_size_literal_random_start_replicas():
    # BASELINE's C5b as written (3D L=256, T=5.0, random start): 16 MiB per chain, clusters of a few spins
    c = wl.CONFIGS["C5b"]
    R = 6
    gpu, refs = make_batch(c.dim, c.L, [c.T] * R, [c.seed + r for r in range(R)])
    compare(gpu, refs, [1000])
    gpu.close()


def test_one_cluster_per_chain_abort_is_reported_by_every_synchronising_call():
    """resident = 3: a chain whose kernel aborted (here: a 1 ms watchdog on a cold-start update of four million spins,
    which one 16-CTA cluster cannot finish in that time) has a half-grown cluster and unfinished logs.  The single-chain
    API reports that at the next synchronising call (WOLFF_EINTERNAL, handle failed: wolff.h); the batch must too, from
    whichever call comes first -- not only from wolff_batch_get_stats."""
    L, R = 2048, 2
    cold = np.stack([wl.cold(L * L)] * R)
    for first_call in ("observables", "get_spins", "series", "moments", "set_spins", "reset_moments"):
        gpu = binding.WolffBatch(2, L, 1.0, [0.5] * R, [11, 12])
        gpu.set_option("resident", 3)
        gpu.set_option("measure", 1)
        gpu.set_spins(cold)
        gpu.set_option("watchdog_ms", 1)
        gpu.run(2)
        with pytest.raises(binding.WolffError) as info:
            {"observables": gpu.observables, "get_spins": gpu.get_spins, "series": gpu.series, "moments": gpu.moments,
             "set_spins": lambda: gpu.set_spins(cold), "reset_moments": gpu.reset_moments}[first_call]()
        assert info.value.code == binding.WOLFF_EINTERNAL, first_call
        assert "watchdog" in str(info.value)
        with pytest.raises(binding.WolffError):
            gpu.run(1)                              # the handle stays failed
        gpu.close()
    # the same start with the default watchdog finishes and is correct: both chains flip nearly the whole lattice
    gpu = binding.WolffBatch(2, L, 1.0, [0.5] * R, [11, 12])
    gpu.set_option("resident", 3)
    gpu.set_spins(cold)
    gpu.run(1)
    E, M, sz = gpu.observables(sizes=True)
    assert all(int(s) > 0.9 * L * L for s in sz[:, 0]) and all(int(m) < 0 for m in M)
    gpu.close()
