"""GPU-vs-oracle parity through the C-ABI: lattice bytes, per-update cluster sizes, integer E and M, bit-exact.

Tolerance: none.  Everything on the path is integer (int8 spins, uint32 bond words against a uint32 threshold,
int64 sums); the one floating-point step, the threshold, is compared first (reading R7).
"""
import numpy as np
import pytest

from paper_1110_0899_b200 import workloads as wl
from parity_util import assert_same_state, compare_batched, compare_stepwise, make_pair

pytestmark = pytest.mark.gpu

# growth tiers forced in turn: auto, grid, one CTA, cluster; then threshold sets that make every tier switch fire
# on small lattices (CTA <-> cluster <-> grid), odd cluster sizes and grid sizes, and the rebalancing path
MODES = [{"mode": 0}, {"mode": 1}, {"mode": 2}, {"mode": 3},
         {"mode": 0, "up_threshold": 8, "down_threshold": 3, "cluster_up_threshold": 40, "grid_down_threshold": 20},
         {"mode": 1, "grid_ctas": 3, "cluster_ctas": 1},
         {"mode": 0, "up_threshold": 2, "down_threshold": 1, "cluster_ctas": 4, "balance_min": 0},
         {"mode": 3, "cluster_ctas": 8, "cluster_up_threshold": 100, "grid_down_threshold": 100, "grid_ctas": 16},
         {"mode": 3, "cluster_ctas": 2, "balance_min": 1000000, "cooperative": 0},
         # shared-memory-resident kernel (mode 0): tiny tiles on few CTAs (every hop crosses a border), a ring so small
         # that sites spill to global memory, bond tables never / always filled
         {"mode": 0, "tile_log": 2, "tile_ctas": 3, "fill": 2, "small_cluster": 0},
         {"mode": 0, "tile_log": 3, "ring_cap": 32, "fill": 2, "idle_ns": 0, "small_cluster": 0},
         {"mode": 0, "fill": 0, "small_cluster": 0},
         {"mode": 0, "fill": 2, "tile_ctas": 5, "tile_log": 4, "small_cluster": 0},
         {"mode": 0, "small_cluster": 1000000},
         # an inbox of 32 entries: senders wait for the receiver all the time (back-pressure path)
         {"mode": 0, "tile_log": 2, "tile_ctas": 4, "inbox_log": 5, "fill": 2, "small_cluster": 0},
         {"mode": 4, "speculative": 1, "up_threshold": 8, "down_threshold": 3, "cluster_up_threshold": 40, "grid_down_threshold": 20},
         # cluster-resident bit-packed kernel (mode 5; lattices it does not apply to fall through to mode 0): the largest
         # cluster, two CTAs with a 32-entry ring (sites spill to global memory, peers steal), one CTA alone
         {"mode": 5}, {"mode": 5, "resident_ctas": 2, "ring_cap": 32, "idle_ns": 0}, {"mode": 5, "resident_ctas": 1},
         {"mode": 5, "resident_ctas": 4, "ring_cap": 64}]


# ------------------------------------------------------------------ BASELINE config C1, exactly as written
@pytest.mark.parametrize("options", MODES[:4] + [{"mode": 5}])
def test_config_c1_every_update(options):
    c = wl.CONFIGS["C1"]
    gpu, ref = make_pair(*c.create_args(), options=options)
    assert_same_state(gpu, ref, "start lattice (reading R9)")
    compare_stepwise(gpu, ref, c.n_meas, lattice_every=100)


# ------------------------------------------------------------------ small and degenerate lattices, every growth mode
SMALL = [(2, 2, 2.0), (2, 3, 2.0), (2, 4, wl.TC_2D), (2, 6, 1.8), (2, 5, 3.0), (3, 2, 4.0), (3, 3, wl.TC_3D),
         (3, 4, wl.TC_3D), (3, 6, 4.0), (2, 16, wl.TC_2D), (3, 8, wl.TC_3D), (2, 48, 2.1), (3, 12, 4.2)]


@pytest.mark.parametrize("options", MODES)
@pytest.mark.parametrize("dim,L,T", SMALL)
def test_small_lattices_stepwise(dim, L, T, options):
    gpu, ref = make_pair(dim, L, 1.0, T, seed=7 + L, options=options)
    assert_same_state(gpu, ref, "start")
    compare_stepwise(gpu, ref, 60)


@pytest.mark.parametrize("options", MODES)
@pytest.mark.parametrize("dim,L", [(2, 64), (2, 100), (3, 16), (3, 20)])
def test_p_one_cold_start_widest_frontiers(dim, L, options):
    # thr = 2^32: the first update flips all N spins; frontiers are as wide as they get and every mode switch fires
    N = L ** dim
    gpu, ref = make_pair(dim, L, 1.0, 0.04, seed=3, start=wl.cold(N), options=options)
    assert gpu.threshold == 1 << 32
    compare_batched(gpu, ref, [1, 1, 3])
    gpu.set_spins(wl.blobs(dim, L, seed=5))
    ref.set_spins(wl.blobs(dim, L, seed=5))
    compare_batched(gpu, ref, [1] * 6)


@pytest.mark.parametrize("dim,L", [(2, 32), (3, 8)])
def test_p_zero_only_the_seed_site_flips(dim, L):
    gpu, ref = make_pair(dim, L, 0.0, 1.0, seed=11)
    assert gpu.threshold == 0
    gpu.run(200)
    E, M, sz = gpu.observables(sizes=True)
    assert np.all(sz == 1)
    assert np.array_equal(sz, ref.run(200))
    assert_same_state(gpu, ref)


@pytest.mark.parametrize("maker", ["checkerboard", "stripes", "blobs", "random"])
@pytest.mark.parametrize("dim,L,T", [(2, 64, 1.5), (3, 16, 3.0)])
def test_crafted_start_lattices(dim, L, T, maker):
    N = L ** dim
    start = {"checkerboard": lambda: wl.checkerboard(dim, L), "stripes": lambda: wl.stripes(dim, L, 3, axis=1),
             "blobs": lambda: wl.blobs(dim, L, 9), "random": lambda: wl.random_pm1(N, 4, 0.7)}[maker]()
    gpu, ref = make_pair(dim, L, 1.0, T, seed=21, start=start)
    compare_batched(gpu, ref, [1, 2, 17, 80])


@pytest.mark.parametrize("case_seed", range(4))
def test_randomised_knobs_shared_memory_resident_kernel(case_seed):
    # 25 short chains per seed with random lattice, temperature, start and every knob of the tiled kernel (tile size,
    # CTAs, ring size, bond tables never / adaptive / always, one or two buffers): the knobs never change the result
    import random
    rng = random.Random(1000 + case_seed)
    for _ in range(25):
        dim = rng.choice([2, 3])
        L = rng.choice([8, 16, 32, 64] if dim == 2 else [4, 8, 16])
        T = rng.choice([wl.TC_2D, 1.8, 3.0] if dim == 2 else [wl.TC_3D, 4.0, 5.0])
        opts = {"mode": 0, "small_cluster": 0, "tile_log": rng.choice([2, 3, 4, 5, 6]), "tile_ctas": rng.choice([0, 1, 2, 3, 7, 16, 64]),
                "fill": rng.choice([0, 1, 2, 2]), "ring_cap": rng.choice([32, 64, 2048]), "idle_ns": rng.choice([0, 100, 1000]),
                "fill_bufs": rng.choice([0, 1]), "fill_min_us": rng.choice([0, 30]), "inbox_log": rng.choice([0, 5, 6, 9])}
        start = rng.choice([None, wl.cold(L ** dim), wl.blobs(dim, L, seed=rng.randrange(1000))])
        gpu, ref = make_pair(dim, L, 1.0, T, seed=rng.randrange(1 << 40), start=start, options=opts)
        compare_batched(gpu, ref, [rng.choice([1, 2, 5]), rng.choice([50, 300]), rng.choice([1, 500])])
        gpu.close()


@pytest.mark.parametrize("case_seed", range(2))
def test_randomised_knobs_cluster_resident_kernel(case_seed):
    # 25 short chains per seed on the cluster-resident bit-packed kernel: random lattice (any L, a partial last word),
    # temperature, start, cluster size (1 .. 16 CTAs) and ring size (32 entries: sites spill to global memory and come
    # back; peers steal), in mode 5 and through the kernel choice of mode 0
    import random
    rng = random.Random(3000 + case_seed)
    for _ in range(25):
        dim = rng.choice([2, 3])
        L = rng.choice([8, 16, 32, 64, 128, 7, 30, 100] if dim == 2 else [4, 8, 16, 32, 5, 11, 24])
        T = rng.choice([wl.TC_2D, 1.8, 3.0] if dim == 2 else [wl.TC_3D, 4.0, 5.0])
        opts = {"mode": rng.choice([5, 5, 0]), "small_cluster": 1 << 30, "resident_ctas": rng.choice([1, 2, 4, 8, 16]),
                "ring_cap": rng.choice([32, 64, 2048]), "idle_ns": rng.choice([0, 100, 1000])}
        start = rng.choice([None, wl.cold(L ** dim), wl.blobs(dim, L, seed=rng.randrange(1000))])
        gpu, ref = make_pair(dim, L, 1.0, T, seed=rng.randrange(1 << 40), start=start, options=opts)
        compare_batched(gpu, ref, [rng.choice([1, 2, 5]), rng.choice([50, 300]), rng.choice([1, 500])])
        gpu.close()


def test_split_run_equivalence_and_resume():
    c = wl.CONFIGS["C1"]
    a, ref = make_pair(*c.create_args())
    b, _ = make_pair(*c.create_args())
    a.run(7); a.run(13); a.run(1)
    b.run(21)
    assert np.array_equal(a.get_spins(), b.get_spins()) and a.observables() == b.observables()
    ref.run(21)
    assert_same_state(a, ref)
    # resume: lattice + update index + seed is the whole state
    c2, _ = make_pair(*c.create_args())
    c2.set_spins(a.get_spins())
    c2.update_index = a.update_index
    a.run(50); c2.run(50); ref.run(50)
    assert np.array_equal(a.get_spins(), c2.get_spins())
    assert_same_state(c2, ref)


def test_seeds_and_large_update_index():
    gpu, ref = make_pair(2, 32, 1.0, wl.TC_2D, seed=(0xDEADBEEF << 32) | 0x12345678)
    gpu.update_index = ref.update_index = (1 << 40) + 12345        # exercises u_hi in the Philox counter
    compare_batched(gpu, ref, [40])


# ------------------------------------------------------------------ medium sizes: several tiles, ragged tails
@pytest.mark.parametrize("options", [{"mode": 0}, {"mode": 1}, {"mode": 3}, {"mode": 0, "fill": 2}, {"mode": 0, "fill": 0}])
@pytest.mark.parametrize("name,n", [("C2", 40), ("C4", 40)])
def test_medium_configs_equilibrated_variant(name, n, options):
    c = wl.CONFIGS[name]
    gpu, ref = make_pair(*c.create_args(), start=wl.cold(c.N), options=options)
    compare_batched(gpu, ref, [1, 4, n])


@pytest.mark.parametrize("name", ["C2", "C4"])
def test_medium_configs_literal_random_start(name):
    c = wl.CONFIGS[name]
    gpu, ref = make_pair(*c.create_args())
    assert_same_state(gpu, ref, "start lattice")
    compare_batched(gpu, ref, [1000])


# ------------------------------------------------------------------ BASELINE full sizes in the bench's launch configuration
@pytest.mark.parametrize("options", [{}, {"fill": 2}])
@pytest.mark.parametrize("name,batches", [("C3", [1, 5]), ("C5a", [1, 8]), ("C5b", [2, 30])])
def test_full_size_configs_equilibrated_variant(name, batches, options):
    # cold start (the bench's 'equilibrated' variant): the first clusters span the lattice, then shrink towards T_c sizes
    c = wl.CONFIGS[name]
    gpu, ref = make_pair(*c.create_args(), start=wl.cold(c.N), options=options)
    compare_batched(gpu, ref, batches)


@pytest.mark.parametrize("name", ["C3", "C5a", "C5b"])
def test_full_size_configs_literal_random_start(name):
    c = wl.CONFIGS[name]
    gpu, ref = make_pair(*c.create_args())
    assert_same_state(gpu, ref, "start lattice")
    compare_batched(gpu, ref, [1000, 2000])


def test_two_live_handles_with_different_plans_interleaved():
    # the kernel's shared-memory attribute belongs to the process, not to a handle: a second handle of the same dim
    # that makes a (smaller) plan must not break the launches of the first (regression: cudaErrorInvalidValue)
    big, ref_big = make_pair(2, 1024, 1.0, wl.TC_2D, seed=5, start=wl.cold(1024 * 1024), options={"small_cluster": 0})
    big.run(3)
    small, ref_small = make_pair(2, 64, 1.0, wl.TC_2D, seed=6, options={"small_cluster": 0, "tile_log": 3, "fill": 0})
    tiny, ref_tiny = make_pair(2, 16, 1.0, wl.TC_2D, seed=7, options={"small_cluster": 0, "tile_log": 2, "tile_ctas": 2})
    ref_big.run(3)
    for _ in range(3):
        small.run(20); ref_small.run(20)
        big.run(2); ref_big.run(2)
        tiny.run(20); ref_tiny.run(20)
        big.run(1); ref_big.run(1)
    for g, r in ((big, ref_big), (small, ref_small), (tiny, ref_tiny)):
        assert_same_state(g, r)
        g.close()
    # the same for the cluster-resident kernel: clusters of 16, 4 and 1 CTAs of one kernel function, interleaved
    a, ref_a = make_pair(3, 32, 1.0, wl.TC_3D, seed=8, options={"mode": 5})
    b, ref_b = make_pair(3, 16, 1.0, wl.TC_3D, seed=9, options={"mode": 5, "resident_ctas": 4})
    c, ref_c = make_pair(3, 8, 1.0, wl.TC_3D, seed=10, options={"mode": 5, "resident_ctas": 1, "ring_cap": 32})
    for _ in range(3):
        for g, r, n in ((a, ref_a, 30), (b, ref_b, 50), (c, ref_c, 70)):
            g.run(n); r.run(n)
    for g, r in ((a, ref_a), (b, ref_b), (c, ref_c)):
        assert_same_state(g, r)
        g.close()


def test_watchdog_abort_is_sticky_across_queued_runs():
    # a cold-start update of 2^24 spins takes milliseconds; with a 1 ms watchdog the first launch aborts.  The runs
    # queued behind it must not continue from a half-grown cluster, and the abort must still be reported.
    from paper_1110_0899_b200 import binding
    c = wl.CONFIGS["C3"]
    gpu = binding.Wolff(*c.create_args())
    gpu.set_option("small_cluster", 0)
    gpu.set_spins(wl.cold(c.N))
    gpu.set_option("watchdog_ms", 1)
    gpu.run(2)
    gpu.run(2)
    gpu.run(2)
    with pytest.raises(binding.WolffError) as info:
        gpu.observables()
    assert info.value.code == binding.WOLFF_EINTERNAL
    with pytest.raises(binding.WolffError):
        gpu.run(1)                                  # the handle stays failed
    gpu.close()
    # the device and the library are fine: a fresh handle works
    g2, ref = make_pair(2, 64, 1.0, wl.TC_2D, seed=3)
    compare_batched(g2, ref, [50])
    g2.close()


def test_microbench_pass_floor_runs_as_intended():
    # the latency-roofline floor (wolff_microbench [7]): every lane must have won every claim, else the chain timed is not
    # the one DESIGN.md section 6 describes
    from paper_1110_0899_b200 import binding
    m = binding.microbench()
    assert m["smem_pass_win_fraction"] == 1.0
    assert 20.0 < m["smem_pass_floor_ns"] < 2000.0
    assert m["l2_load_lane_ns"] > m["smem_pass_floor_ns"] / 10.0
    # the links of the cluster-resident kernel: a claim on a peer's shared memory is cheaper than one through L2
    assert 20.0 < m["dsmem_atomic_lane_ns"] < m["l2_atomic_lane_ns"]
    assert 20.0 < m["dsmem_load_lane_ns"] < 1000.0 and 20.0 < m["dsmem_store_to_poll_ns"] < 2000.0


@pytest.mark.parametrize("name", ["C1", "C2", "C4"])
def test_first_run_on_a_fresh_non_blocking_stream(name):
    # the very first wolff_run of a handle allocates and clears the tiled kernel's queues; a kernel launched on a
    # non-blocking stream must not start before that clearing has finished (regression: lost messages, watchdog abort)
    import torch
    c = wl.CONFIGS[name]
    for seed in range(3):
        gpu, ref = make_pair(c.dim, c.L, c.J, c.T, seed=100 + seed, options={"small_cluster": 0, "watchdog_ms": 5000})
        stream = torch.cuda.Stream()
        gpu.run(10, stream=stream)
        E, M, sz = gpu.observables(sizes=True)
        assert np.array_equal(sz, ref.run(10))
        assert (E, M) == ref.observables()
        assert_same_state(gpu, ref)
        gpu.close()


@pytest.mark.parametrize("case_seed", range(3))
def test_random_api_sequences(case_seed):
    # 40 chains per seed of randomly interleaved calls: runs on the default and on non-blocking streams, knob changes in
    # the middle of a chain (kernel, tiling, tables), lattices loaded and read back through device and host buffers,
    # update index jumps -- compared with the oracle after every step that returns something
    import random
    import torch
    rng = random.Random(2000 + case_seed)
    streams = [None, torch.cuda.Stream(), torch.cuda.Stream()]
    knobs = {"mode": [0, 0, 4, 1, 3, 5], "small_cluster": [0, 16, 100000], "resident_ctas": [1, 2, 4, 16], "tile_log": [0, 2, 3, 4, 5], "tile_ctas": [0, 1, 3, 16],
             "fill": [0, 1, 2], "fill_bufs": [0, 1], "ring_cap": [32, 2048], "idle_ns": [0, 1000], "fill_min_us": [0, 30],
             "inbox_log": [0, 5, 7]}
    for _ in range(40):
        dim = rng.choice([2, 3])
        L = rng.choice([8, 16, 32, 64] if dim == 2 else [4, 8, 16])
        gpu, ref = make_pair(dim, L, 1.0, rng.choice([wl.TC_2D, 1.9] if dim == 2 else [wl.TC_3D, 4.0]), seed=rng.randrange(1 << 40))
        for _step in range(rng.randrange(4, 12)):
            op = rng.choice(["run", "run", "run", "opt", "set", "obs_dev", "get_dev", "idx"])
            if op == "run":
                k = rng.choice([1, 2, 7, 60, 400])
                gpu.run(k, stream=rng.choice(streams))
                rs = ref.run(k)
                if rng.random() < 0.6:
                    E, M, sz = gpu.observables(sizes=True)
                    assert np.array_equal(sz, rs) and (E, M) == ref.observables()
            elif op == "opt":
                key = rng.choice(list(knobs))
                gpu.set_option(key, rng.choice(knobs[key]))
            elif op == "set":
                start = rng.choice([wl.cold(L ** dim), wl.blobs(dim, L, seed=rng.randrange(99)), wl.checkerboard(dim, L)])
                gpu.set_spins(start)
                ref.set_spins(start)
            elif op == "obs_dev":
                E = torch.zeros(1, dtype=torch.int64, device="cuda")
                M = torch.zeros(1, dtype=torch.int64, device="cuda")
                gpu.observables_into(E, M, None)
                assert (int(E.item()), int(M.item())) == ref.observables()
            elif op == "get_dev":
                d = torch.empty(L ** dim, dtype=torch.int8, device="cuda")
                gpu.get_spins_into(d)
                assert np.array_equal(d.cpu().numpy(), ref.get_spins())
            else:
                u = rng.randrange(1 << 45)
                gpu.update_index = u
                ref.update_index = u
        assert_same_state(gpu, ref, "end of a random call sequence")
        gpu.close()
