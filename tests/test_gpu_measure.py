"""In-kernel measurement ("measure" = 1) against the oracle: E and M after EVERY update, bit-exact.

PAPER.md:126, 138, 147 (the "+ measurement" columns) and Eq. 3.  The CUDA path evaluates E and M
inside the persistent kernel (growth_tiles.cu: every CTA sums the tiles it holds; growth_cluster.cu: population counts over
the bit lattice; growth.cu: running values from the cluster's boundary bonds); the oracle sums the whole lattice after every update (oracle_run_logged) and accumulates the
moments by their definition (oracle_moments).  Everything is integer: tolerance none, except the Binder ratio, a
double computed from identical integers on both sides (1e-12).
"""
import numpy as np
import pytest

import oracle
import protocol_farm as farm
from paper_1110_0899_b200 import binding, workloads as wl
from parity_util import assert_same_state, make_pair
from test_gpu_parity import MODES

pytestmark = pytest.mark.gpu


def compare_measured(gpu, ref, batches, acc=None):
    """run(n) with in-kernel measurement; sizes, E and M series, accumulated moments, lattice -- all against the oracle."""
    for n in batches:
        gpu.run(n)
        E, M = gpu.series()
        _, _, sz = gpu.observables(sizes=True)
        rs, rE, rM = ref.run_logged(n)
        assert np.array_equal(sz, rs), "cluster sizes differ"
        if not np.array_equal(E, rE):
            k = int(np.nonzero(E != rE)[0][0])
            raise AssertionError("E differs at update %d of %d: gpu %d oracle %d (size %d)" % (k, n, E[k], rE[k], rs[k]))
        if not np.array_equal(M, rM):
            k = int(np.nonzero(M != rM)[0][0])
            raise AssertionError("M differs at update %d of %d: gpu %d oracle %d" % (k, n, M[k], rM[k]))
        acc = oracle.moments_raw(rE, rM, acc=acc)
        raw, U = gpu.moments()
        assert np.array_equal(raw, acc), (oracle.moments_dict(raw), oracle.moments_dict(acc))
        Uo = oracle.binder(acc)
        assert (np.isnan(U) and np.isnan(Uo)) or abs(U - Uo) < 1e-12
        assert_same_state(gpu, ref, "after a measured batch of %d" % n)
    return acc


MEASURE_MODES = [dict(o, measure=1) for o in MODES]


@pytest.mark.parametrize("options", [{"mode": 0, "small_cluster": 0}, {"mode": 0}, {"mode": 4}, {"mode": 1},
                                      {"mode": 0, "small_cluster": 0, "fill": 2, "tile_log": 4}, {"mode": 5}])
def test_config_c1_measured_every_update(options):
    c = wl.CONFIGS["C1"]
    gpu, ref = make_pair(*c.create_args(), options=dict(options, measure=1))
    compare_measured(gpu, ref, [c.n_meas])
    gpu.close()


SMALL = [(2, 2, 2.0), (2, 3, 2.0), (2, 4, wl.TC_2D), (2, 6, 1.8), (3, 2, 4.0), (3, 3, wl.TC_3D), (3, 4, wl.TC_3D),
         (2, 16, wl.TC_2D), (3, 8, wl.TC_3D), (2, 48, 2.1), (3, 12, 4.2), (2, 64, 2.0), (3, 16, 4.3)]


@pytest.mark.parametrize("options", MEASURE_MODES)
@pytest.mark.parametrize("dim,L,T", SMALL)
def test_small_lattices_measured(dim, L, T, options):
    gpu, ref = make_pair(dim, L, 1.0, T, seed=70 + L, options=options)
    compare_measured(gpu, ref, [1, 2, 60])
    gpu.close()


@pytest.mark.parametrize("options", MEASURE_MODES)
@pytest.mark.parametrize("dim,L", [(2, 64), (2, 100), (3, 16), (3, 20)])
def test_p_one_cold_start_measured(dim, L, options):
    # every spin in one cluster: the member log of the level-synchronous kernel runs through every tier, the post-pass
    # sees a cluster without boundary; then ragged blobs (large boundaries)
    N = L ** dim
    gpu, ref = make_pair(dim, L, 1.0, 0.04, seed=3, start=wl.cold(N), options=options)
    compare_measured(gpu, ref, [1, 1, 3])
    gpu.set_spins(wl.blobs(dim, L, seed=5))
    ref.set_spins(wl.blobs(dim, L, seed=5))
    compare_measured(gpu, ref, [1] * 4, acc=gpu.moments()[0])
    gpu.close()


@pytest.mark.parametrize("options", [{"mode": 5}, {"mode": 5, "resident_ctas": 2, "ring_cap": 32}, {"mode": 5, "resident_ctas": 1, "idle_ns": 0},
                                      {"mode": 0, "small_cluster": 1 << 30}])
@pytest.mark.parametrize("dim,L,T", [(2, 32, wl.TC_2D), (2, 96, 2.2), (3, 32, wl.TC_3D), (2, 128, 2.0), (3, 64, 4.4), (2, 160, wl.TC_2D)])
def test_cluster_resident_kernel_measured(dim, L, T, options):
    # the cluster-resident kernel measures by population counts over its bit lattice when L is a multiple of 32 (L a power of
    # two and not; one word per row at L = 32); every spin in one cluster from a cold start, then ragged blobs
    gpu, ref = make_pair(dim, L, 1.0, T, seed=90 + L, options=dict(options, measure=1))
    acc = compare_measured(gpu, ref, [1, 2, 60])
    gpu.set_spins(wl.cold(L ** dim)); ref.set_spins(wl.cold(L ** dim))
    acc = compare_measured(gpu, ref, [1, 5], acc=acc)
    gpu.set_spins(wl.blobs(dim, L, seed=5)); ref.set_spins(wl.blobs(dim, L, seed=5))
    compare_measured(gpu, ref, [1] * 3 + [30], acc=acc)
    st = gpu.stats()
    if options["mode"] == 5:         # (mode 0 sends measured runs on clusters of a handful of spins to the level-synchronous kernel)
        assert st["levels_cta"] + st["levels_cluster"] + st["levels_grid"] + st["fill_chunks"] + st["inline_passes"] == 0    # it was this kernel
    gpu.close()


@pytest.mark.parametrize("options", [{"mode": 0, "small_cluster": 0}, {"mode": 4}, {"mode": 3}, {"mode": 1}, {"mode": 5}])
@pytest.mark.parametrize("name,n", [("C2", 150), ("C4", 100)])
def test_medium_configs_measured(name, n, options):
    c = wl.CONFIGS[name]
    gpu, ref = make_pair(*c.create_args(), start=wl.cold(c.N), options=dict(options, measure=1))
    compare_measured(gpu, ref, [3, n])
    gpu.close()


def test_moments_run_on_across_runs_and_reset():
    c = wl.CONFIGS["C1"]
    gpu, ref = make_pair(*c.create_args(), options={"measure": 1})
    acc = compare_measured(gpu, ref, [10, 40])
    gpu.set_option("measure", 0)                       # an unmeasured run leaves the accumulators alone
    gpu.run(25); ref.run(25)
    with pytest.raises(binding.WolffError):
        gpu.series()
    ns = gpu.update_ns()                               # durations are always recorded
    assert ns.shape == (25,) and np.all(ns > 0)
    assert np.array_equal(gpu.moments()[0], acc)
    gpu.set_option("measure", 1)
    acc = compare_measured(gpu, ref, [30], acc=acc)
    gpu.reset_moments()
    raw, U = gpu.moments()
    assert not raw.any() and np.isnan(U)
    compare_measured(gpu, ref, [20])
    gpu.close()


@pytest.mark.parametrize("name,options", [("C5a", {}), ("C5a", {"mode": 4}), ("C3-stretch", {}), ("C5a", {"mode": 5})])
def test_protocol_stretch_measured_in_kernel(name, options):
    # the stretch of single updates of the protocol tests, as ONE measured launch: same E, M after every update
    job = farm.JOBS[name]
    c = wl.CONFIGS[job["cfg"]]
    gpu = binding.Wolff(c.dim, c.L, c.J, c.T, c.seed if job["seed"] is None else job["seed"])
    for k, v in options.items():
        gpu.set_option(k, v)
    gpu.set_spins(wl.cold(c.N))
    ref = farm.result(name)
    for b in ref["batches"]:
        gpu.run(b["n"])
    st = ref["stretch"]
    gpu.set_option("measure", 1)
    gpu.run(len(st["sizes"]))
    E, M = gpu.series()
    _, _, sz = gpu.observables(sizes=True)
    assert np.array_equal(sz, st["sizes"])
    assert np.array_equal(E, st["E"]) and np.array_equal(M, st["M"])
    raw, U = gpu.moments()
    acc = oracle.moments_raw(st["E"], st["M"])
    assert np.array_equal(raw, acc) and abs(U - oracle.binder(acc)) < 1e-12
    assert np.array_equal(farm.pack(gpu.get_spins()), st["bits"])
    gpu.close()


def _measured_without_reevaluation(gpu, ref, n, acc):
    """A measured run followed ONLY by series() / moments(): no wolff_observables, so the next measured run must start from
    the running E and M the previous kernel left on the device (the em_valid carry-over of api.cu / batch_api.cu)."""
    gpu.run(n)
    E, M = gpu.series()
    rs, rE, rM = ref.run_logged(n)
    assert np.array_equal(E, rE) and np.array_equal(M, rM), "series differ"
    acc = oracle.moments_raw(rE, rM, acc=acc)
    assert np.array_equal(gpu.moments()[0], acc)
    return acc


@pytest.mark.parametrize("dim,L,T", [(2, 64, wl.TC_2D), (3, 32, wl.TC_3D), (2, 96, 2.2)])
def test_running_energy_carries_over_between_measured_runs_and_kernels(dim, L, T):
    gpu, ref = make_pair(dim, L, 1.0, T, seed=17 + L, options={"measure": 1})
    tiled = {"mode": 0, "small_cluster": 0}
    cluster = {"mode": 5}
    levels = {"mode": 4}
    acc = None
    for options, n in ((tiled, 20), (tiled, 15), (cluster, 20), (cluster, 10), (levels, 12), (levels, 9), (tiled, 7), (levels, 5),
                       (cluster, 6), (tiled, 4)):
        for k, v in options.items():
            gpu.set_option(k, v)
        acc = _measured_without_reevaluation(gpu, ref, n, acc)
    assert_same_state(gpu, ref, "after ten measured runs without a whole-lattice evaluation in between")
    gpu.close()


def test_running_energy_carries_over_in_a_batch():
    import test_gpu_batch as tb
    T = [2.0, wl.TC_2D, 2.6]
    gpu, refs = tb.make_batch(2, 64, T, [5, 6, 7], options={"measure": 1})
    acc = [None] * gpu.R
    for resident, n in ((3, 12), (3, 8), (1, 10), (2, 9), (3, 6), (1, 5)):
        gpu.set_option("resident", resident)
        gpu.run(n)
        Es, Ms = gpu.series()
        raw, _ = gpu.moments()
        for r, ref in enumerate(refs):
            _, rE, rM = ref.run_logged(n)
            assert np.array_equal(Es[r], rE) and np.array_equal(Ms[r], rM), "chain %d, resident %d" % (r, resident)
            acc[r] = oracle.moments_raw(rE, rM, acc=acc[r])
            assert np.array_equal(raw[r], acc[r])
    tb.assert_same_lattices(gpu, refs, "after six measured batch runs without an evaluation in between")
    gpu.close()


def test_measured_runs_that_would_wrap_the_moment_accumulators_are_refused():
    """sum M^4 is kept in 128 bits and |M| <= N, so the accumulators are exact while samples x N^4 < 2^128.  At N = 2^28
    that is 2^16 samples.  The oracle's accumulators would wrap in the same way, so parity cannot see an overflow: the
    library refuses the run instead (wolff.h, wolff_get_moments)."""
    L = 16384
    gpu = binding.Wolff(2, L, 1.0, 2.4, seed=1)
    gpu.set_option("measure", 1)
    with pytest.raises(binding.WolffError) as info:
        gpu.run(65537)
    assert info.value.code == binding.WOLFF_EINVAL and "overflow" in str(info.value)
    gpu.run(2)                                          # two samples in
    assert int(gpu.moments()[0][0]) == 2
    with pytest.raises(binding.WolffError):
        gpu.run(65535)                                  # 2 + 65535 > 2^16
    gpu.set_option("measure", 0)
    gpu.run(3)                                          # unmeasured runs are not counted
    gpu.set_option("measure", 1)
    gpu.reset_moments()
    gpu.run(65535)                                      # the count started again
    assert int(gpu.moments()[0][0]) == 65535
    with pytest.raises(binding.WolffError):
        gpu.run(2)
    gpu.close()
    batch = binding.WolffBatch(2, L, 1.0, [2.4], [3])
    batch.set_option("measure", 1)
    with pytest.raises(binding.WolffError) as info:
        batch.run(65537)
    assert info.value.code == binding.WOLFF_EINVAL and "overflow" in str(info.value)
    batch.close()
