"""Small cases of every kernel of libwolff_b200, meant to be run under a memory / race checker:

    WOLFF_B200_LIB=paper_1110_0899_b200/libwolff_b200_checked.so python tests/sanitizer_cases.py    (the bounds-checked
        build, -DWOLFF_CHECKED: tests/test_gpu_checked.py runs exactly this)
    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py tiles
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py

(compute-sanitizer is closed on the pool this library was developed on -- profiles/r2_checked_build.md -- so the first
line is the one that has been run.)  Each case runs a short chain through the C-ABI and checks it against the oracle,
so a run that a tool slowed down by two orders of magnitude still proves that the kernels did their work.  Knobs make the small lattices exercise what the
large ones do: tiny tiles on few CTAs (every hop a message), a 32-entry ring (spills), a 32-entry inbox
(back-pressure), bond tables on and off, every tier of the level-synchronous kernel, the cluster-resident kernel on 1 to 16 CTAs,
in-kernel measurement, the batch.
Summaries of the runs are kept under profiles/ (SURVEY.md section 4 tier 4, section 5 "Race detection").
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import oracle                                                    # noqa: E402
from paper_1110_0899_b200 import binding, workloads as wl        # noqa: E402

SLOW = {"watchdog_ms": 3600000}      # the tools slow the kernels down a lot: the device watchdog must not fire

TILES = [
    (2, 16, wl.TC_2D, {"mode": 0, "small_cluster": 0, "tile_log": 2, "tile_ctas": 3, "ring_cap": 32, "fill": 2}),
    (2, 16, wl.TC_2D, {"mode": 0, "small_cluster": 0, "tile_log": 2, "tile_ctas": 3, "ring_cap": 32, "fill": 0, "inbox_log": 5}),
    (3, 8, wl.TC_3D, {"mode": 0, "small_cluster": 0, "tile_log": 2, "tile_ctas": 4, "ring_cap": 32, "fill": 2, "fill_bufs": 1}),
    (2, 32, 2.0, {"mode": 0, "small_cluster": 0, "tile_log": 4, "tile_ctas": 2, "fill": 2, "measure": 1}),
    (3, 8, 4.0, {"mode": 0, "small_cluster": 0, "tile_log": 2, "tile_ctas": 5, "fill": 1, "measure": 1, "inbox_log": 5}),
]
TIERS = [
    (2, 24, 2.0, {"mode": 4, "up_threshold": 8, "down_threshold": 3, "cluster_up_threshold": 40, "grid_down_threshold": 20}),
    (3, 6, 4.0, {"mode": 1, "grid_ctas": 3, "cluster_ctas": 1}),
    (2, 20, 2.1, {"mode": 3, "cluster_ctas": 4, "balance_min": 0}),
    (2, 24, 2.0, {"mode": 4, "up_threshold": 8, "down_threshold": 3, "cluster_up_threshold": 40, "grid_down_threshold": 20, "measure": 1}),
    (3, 6, 4.2, {"mode": 2, "measure": 1}),
    (2, 16, 2.2, {"mode": 4, "speculative": 1}),
]


CLUSTER = [
    (2, 16, wl.TC_2D, {"mode": 5}),
    (3, 8, wl.TC_3D, {"mode": 5, "resident_ctas": 4, "ring_cap": 32, "idle_ns": 0}),
    (2, 32, 2.0, {"mode": 5, "resident_ctas": 2, "ring_cap": 32}),
    (3, 8, 4.0, {"mode": 0, "small_cluster": 1 << 30, "resident_ctas": 1}),
    (2, 21, 2.1, {"mode": 0, "resident_ctas": 4, "ring_cap": 32}),          # L not a power of two, a partial last word
]


def single_chain(dim, L, T, options, n=12):
    gpu = binding.Wolff(dim, L, 1.0, T, 11)
    ref = oracle.OracleWolff(dim, L, 1.0, T, 11)
    for k, v in dict(options, **SLOW).items():
        gpu.set_option(k, v)
    start = wl.blobs(dim, L, seed=3)
    gpu.set_spins(start)
    ref.set_spins(start)
    gpu.run(n)
    E, M, sz = gpu.observables(sizes=True)
    if options.get("measure"):
        rs, rE, rM = ref.run_logged(n)
        Es, Ms = gpu.series()
        assert np.array_equal(Es, rE) and np.array_equal(Ms, rM)
    else:
        rs = ref.run(n)
    assert np.array_equal(sz, rs) and (E, M) == ref.observables()
    assert np.array_equal(gpu.get_spins(), ref.get_spins())
    gpu.stats()                                  # a checked build reports an index out of its bounds here (WOLFF_EINTERNAL)
    gpu.close()


def batch(measure, threads, resident):
    R = 6
    T = [2.0 + 0.1 * r for r in range(R)]
    gpu = binding.WolffBatch(2, 16, 1.0, T, list(range(40, 40 + R)))
    refs = [oracle.OracleWolff(2, 16, 1.0, T[r], 40 + r) for r in range(R)]
    gpu.set_option("measure", measure)
    gpu.set_option("threads", threads)
    gpu.set_option("queue_cap", 8)
    gpu.set_option("resident", resident)
    gpu.run(15)
    E, M, sz = gpu.observables(sizes=True)
    spins = gpu.get_spins()
    for r, ref in enumerate(refs):
        assert np.array_equal(sz[r], ref.run(15)) and (int(E[r]), int(M[r])) == ref.observables()
        assert np.array_equal(spins[r], ref.get_spins())
    gpu.stats()
    gpu.close()


def main(which):
    done = []
    if which in ("all", "tiles"):
        for case in TILES:
            single_chain(*case)
            done.append("tiles %s" % (case[3],))
    if which in ("all", "tiers"):
        for case in TIERS:
            single_chain(*case)
            done.append("tiers %s" % (case[3],))
    if which in ("all", "cluster"):
        for case in CLUSTER:
            single_chain(*case)
            done.append("cluster %s" % (case[3],))
    if which in ("all", "batch"):
        for measure, threads, resident in [(0, 32, 1), (1, 64, 1), (1, 256, 2), (0, 64, 2), (0, 64, 3)]:
            batch(measure, threads, resident)
            done.append("batch measure=%d threads=%d resident=%d" % (measure, threads, resident))
    for d in done:
        print("ok:", d)
    print("sanitizer cases passed: %d" % len(done))


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else "all")
