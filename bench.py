#!/usr/bin/env python
"""bench.py -- throughput of the Wolff single-cluster hot path on B200, one JSON line.

A "step" is one pass of the whole hot path over one batch:
    wolff_run(h, U, stream)           -- U single-cluster updates as ONE persistent kernel launch (A1-A7)
    wolff_observables(h, E, M, sizes) -- the whole-lattice E/M reduction (A8) + read-back of the size log (A9)
on the workload BASELINE.json's metric is quoted on: 2D L=4096 at T_c (primary; `value`) and 3D L=256 at T_c
(reported under "secondary").  Start state: the 'equilibrated' variant of SURVEY.md 8(d) -- cold start followed by
`--equil` untimed updates -- because the literal random start never reaches T_c-sized clusters within the configured
1,000 + 10,000 updates; the literal variant is reported as updates/s under "literal_random_start".  With the default
U = 500 the driver's 20 steps are BASELINE.json's 10,000 measured updates.

Every GPU figure has the oracle beside it, timed on the SAME clusters: the lattice and update index at the start of
the timed region are copied out of the library and loaded into the oracle, which then runs a bounded prefix of exactly
those updates on one host core (the algorithm is sequential; `cores` says so).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--workload C3] [--updates U]
                    [--opt key=value ...]

N > 1 (torchrun): replicas only -- every rank runs its own independent chain (seed + rank), no
data-path collective; value = flipped spins of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "flipped spins/sec & Wolff updates/sec, 2D L=4096 and 3D L=256 at T_c"
UNIT = "flipped spins/s"
DTYPE = "int8 spins / uint32 bond words / int64 sums"
L2_FLUSH_BYTES = 256 << 20          # > 126 MB L2


def measured_peak_hbm():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, STREAM-style copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ncu `--set full` DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of the growth kernel, by
# (workload, growth mode): taken offline from the committed captures under profiles/ (the launch shape of each capture
# is stated there).  Any other workload / mode / knob setting prints null -- never a figure from another configuration.
NCU_TRAFFIC = {
    ("C3", 0): {"bytes": 26623488 + 1387264, "source": "profiles/r2_growth_tiles_C3.md (50-update launch; the traffic is the one lattice "
                                                        "load per launch plus the queues, and does not grow with the updates)"},
    ("C5a", 0): {"bytes": 54497536 + 8451584, "source": "profiles/r2_growth_tiles_C5a.md (200-update launch)"},
}


def kernel_of(stats: dict) -> str:
    """Which growth kernel the most recent run used, from its counters (wolff_get_stats)."""
    if stats["levels_cta"] + stats["levels_cluster"] + stats["levels_grid"] > 0:
        return "growth_kernel (level-synchronous tiers)"
    if stats["fill_chunks"] + stats["inline_passes"] > 0:
        return "growth_tiles_kernel (int8 tiles in the shared memory of all SMs)"
    return "growth_cluster_kernel (bit-packed lattice in one cluster's distributed shared memory)"


def ncu_traffic(workload: str, mode: int, options: dict):
    if options:
        return None
    return NCU_TRAFFIC.get((workload, mode))


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 200 ms while the timed region runs."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.QUERY,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for name, flag in zip(names, parts[3:7]):
                if flag.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def algorithmic_bytes(dim: int, flipped: int, attempts: int) -> int:
    """Bytes the growth kernel must touch: per added spin 2*dim neighbour bytes, one 4-byte
    list write and one 4-byte list read; plus one 4-byte atomic read-modify-write per claim attempt."""
    return flipped * (2 * dim + 8) + 4 * attempts


def workload_config(c, equil: int, updates: int, world: int):
    """The `config` object of the JSON line: the same for the CUDA arm and the reference arm."""
    return {"workload": "%s, equilibrated variant: cold start + %d untimed updates, seed %d(+rank)" % (c.name, equil, c.seed),
            "updates_per_step": updates, "step": "wolff_run(U) + wolff_observables (E, M, size log)",
            "l2": "flushed between steps by a %d MiB write, outside the timed events" % (L2_FLUSH_BYTES >> 20),
            "parallelism": "replicas only" if world > 1 else "single GPU"}


# ====================================================================== N > 1: replicas only

def all_reduce_scalar(x, op: str, world: int, device=None):
    """Sum / max of one number over the ranks (no-op at world 1).  The only collective of the bench: the data path
    has none, every rank runs its own chain."""
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM if op == "sum" else dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_replicas(flipped: int, updates: int, total_ms: float, world: int, device=None):
    """Whole-job throughput of N independent replicas: units of all ranks / the slowest rank's device time."""
    ms = all_reduce_scalar(total_ms, "max", world, device)
    f = all_reduce_scalar(flipped, "sum", world, device)
    u = all_reduce_scalar(updates, "sum", world, device)
    return {"total_ms": ms, "flipped": f, "updates": u, "value": f / (ms * 1e-3), "updates_per_s": u / (ms * 1e-3)}


# ====================================================================== the oracle beside every figure

def oracle_on_same_clusters(c, seed: int, lattice, update_index: int, budget_s: float, max_updates: int, measured: bool = False):
    """The oracle as it stands, one host core, started from the very state the GPU's timed region started from
    (lattice bytes + update index + seed = the whole state), running a bounded prefix of exactly those updates.
    measured=True: E and M by whole-lattice summation after every update, as the paper's CPU '+ measurement' column."""
    import oracle
    ref = oracle.OracleWolff(c.dim, c.L, c.J, c.T, seed)
    ref.set_spins(lattice)
    ref.update_index = update_index
    flipped = n = 0
    all_sizes = []
    t0 = time.perf_counter()
    while n < max_updates and time.perf_counter() - t0 < budget_s:
        if measured:
            sizes, _, _ = ref.run_logged(1)
        else:
            sizes = ref.run(1)
        flipped += int(sizes[0])
        all_sizes.append(int(sizes[0]))
        n += 1
    dt = time.perf_counter() - t0
    ref.close()
    return {"sizes": all_sizes, "value": flipped / dt, "unit": UNIT, "updates_per_s": n / dt, "cores": 1, "kind": "oracle",
            "sample": "%s, the first %d updates of the GPU's timed region (from update index %d, same lattice, same seed): "
                      "%.1f s of CPU work, %d spins flipped%s" % (c.name, n, update_index, dt, flipped,
                                                                  ", E and M summed over the lattice after every update" if measured else ""),
            "host_cores_available": os.cpu_count()}


def oracle_replicas(c, seeds, n_updates: int, budget_s: float, threads: int, equil: int = 0):
    """`threads` independent oracle chains side by side (one per host core; the ctypes calls release the GIL): the
    aggregate the host can reach on replicas.  Literal start (the oracle's own seed-derived lattice), then the same
    `equil` untimed updates the batch ran before its timed call, so that both sides time the same clusters."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor

    def one(seed):
        ref = oracle.OracleWolff(c.dim, c.L, c.J, c.T, seed)
        if equil:
            ref.run(equil)
        t0 = time.perf_counter()
        n = f = 0
        while n < n_updates and time.perf_counter() - t0 < budget_s:
            f += int(ref.run(100).sum())
            n += 100
        dt = time.perf_counter() - t0
        ref.close()
        return n, f, dt

    with ThreadPoolExecutor(max_workers=threads) as pool:
        res = list(pool.map(one, seeds[:threads]))
    dt = max(r[2] for r in res)
    return {"updates_per_s": sum(r[0] for r in res) / dt, "value": sum(r[1] for r in res) / dt, "unit": UNIT, "cores": threads,
            "kind": "oracle", "one_core_updates_per_s": res[0][0] / res[0][2],
            "sample": "%s literal random start + %d untimed updates, %d chains of up to %d updates side by side (the updates the batch times)" % (
                c.name, equil, threads, n_updates)}


# ====================================================================== the CUDA arm

def run_b200(args, rank: int, world: int):
    import numpy as np
    import torch
    from paper_1110_0899_b200 import build as cuda_build
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        cuda_build.build()              # no-op when libwolff_b200.so is up to date; the .so is not in the history
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    from paper_1110_0899_b200 import binding, workloads as wl

    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    options = dict(args.opt)
    launches = [0]
    parity_checks = []                  # one entry per leg whose oracle sample was compared with the kernel's size log

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    def open_chain(cfg_name: str, seed: int, cold: bool, equil: int, extra=None):
        c = wl.CONFIGS[cfg_name]
        h = binding.Wolff(c.dim, c.L, c.J, c.T, seed)
        if args.mode:
            h.set_option("mode", args.mode)
        for k, v in list(options.items()) + list((extra or {}).items()):
            h.set_option(k, v)
        if cold:
            h.set_spins(wl.cold(c.N))
        if equil:
            h.run(equil, stream=stream)
            h.observables()
        return c, h

    def measure(cfg_name: str, updates: int, equil: int, steps: int, warmup: int, cold: bool, seed_offset: int = 0,
                depth_steps: int = 1, sample_clocks: bool = False):
        """One timed leg.  Returns per-step device times, the kernel's own per-update durations, counters, the BFS depth
        of the first `depth_steps` timed steps, and the state at the start of the timed region (for the oracle)."""
        c = wl.CONFIGS[cfg_name]
        seed = c.seed + rank + seed_offset
        c, h = open_chain(cfg_name, seed, cold, equil)
        E_d = torch.zeros(1, dtype=torch.int64, device=dev)
        M_d = torch.zeros(1, dtype=torch.int64, device=dev)
        sizes_d = torch.zeros(updates, dtype=torch.int32, device=dev)
        ns_d = torch.zeros(updates, dtype=torch.int32, device=dev)
        res = {"cfg": c, "h": h, "seed": seed, "flipped": 0, "attempts": 0, "levels": 0, "depth_updates": 0, "updates": updates * steps,
               "step_ms": [], "growth_ms": [], "update_ns": [], "sizes": []}
        # BFS depth of the clusters the timed steps grow (a property of the workload): the
        # level-synchronous kernel (mode 4) replays the same updates from the same lattice, untimed, and counts levels
        twin = None
        if args.mode == 0 and not args.no_depth and depth_steps > 0:
            twin = binding.Wolff(c.dim, c.L, c.J, c.T, seed)
            twin.set_option("mode", 4)
            snapshot = torch.empty(c.N, dtype=torch.int8, device=dev)

        def one_step(timed: bool, index: int):
            replay = timed and twin is not None and index < depth_steps
            if replay:
                h.get_spins_into(snapshot)
                twin.set_spins(snapshot)
                twin.update_index = h.update_index
            with torch.cuda.stream(stream):
                flush.fill_(1)                     # L2 flush between steps, outside the timed events
                e0 = torch.cuda.Event(enable_timing=True)
                e1 = torch.cuda.Event(enable_timing=True)
                e2 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                h.run(updates, stream=stream)      # A1-A7: one persistent kernel
                e1.record(stream)
                h.observables_into(E_d, M_d, sizes_d)   # A8 + A9 (device buffers); blocks
                e2.record(stream)
            e2.synchronize()
            if timed:
                launches[0] += 2
                res["step_ms"].append(e0.elapsed_time(e2))
                res["growth_ms"].append(e0.elapsed_time(e1))
                st = h.stats()
                res["kernel"] = kernel_of(st)
                res["flipped"] += st["flipped"]; res["attempts"] += st["claim_attempts"]
                assert int(sizes_d.sum().item()) == st["flipped"]
                res["sizes"].append(sizes_d.cpu().numpy().astype(np.uint32))
                h.series_into(None, None, ns_d)
                res["update_ns"].append(ns_d.cpu().numpy().astype(np.uint32).astype(np.float64))
                if replay:
                    twin.run(updates, stream=stream)
                    ts = twin.stats()
                    assert ts["flipped"] == st["flipped"]
                    res["levels"] += ts["levels_cta"] + ts["levels_cluster"] + ts["levels_grid"]
                    res["depth_updates"] += updates
                    res["depth_growth_ms"] = res.get("depth_growth_ms", 0.0) + e0.elapsed_time(e1)

        for i in range(warmup):
            one_step(False, i)
        # the state the timed region starts from: lattice + update index (+ seed) is the whole state of a chain
        res["start_lattice"] = h.get_spins()
        res["start_index"] = h.update_index
        barrier()
        if sample_clocks:
            with ClockSampler(local_rank) as clocks:
                for i in range(steps):
                    one_step(True, i)
                barrier()
            res["clocks"] = clocks.summary()
        else:
            for i in range(steps):
                one_step(True, i)
        if twin is not None:
            twin.close()
        ns = np.concatenate(res["update_ns"]) if res["update_ns"] else np.zeros(1)
        res["ms_per_update_mean_in_kernel"] = float(ns.mean()) * 1e-6
        res["ms_per_update_median_in_kernel"] = float(np.median(ns)) * 1e-6
        return res

    def leg_summary(r, oracle_budget: float, oracle_max: int = 10 ** 9):
        ms = sum(r["step_ms"])
        out = {"value": r["flipped"] / (ms * 1e-3), "unit": UNIT, "updates_per_s": r["updates"] / (ms * 1e-3), "kernel": r.get("kernel"),
               "updates_timed": r["updates"], "mean_cluster": r["flipped"] / max(r["updates"], 1),
               "ms_per_update_mean": ms / max(r["updates"], 1), "ms_per_update_median": r["ms_per_update_median_in_kernel"],
               "ms_per_update_note": "mean = device time of the steps / updates; median = the kernel's own per-update durations (wolff_get_series)"}
        if r["depth_updates"]:
            out["bfs_depth_per_update"] = r["levels"] / r["depth_updates"]
            out["us_per_bfs_level"] = r["depth_growth_ms"] * 1e3 / max(r["levels"], 1)
            out["bfs_depth_sample"] = "the first %d timed updates, replayed untimed by the level-synchronous kernel" % r["depth_updates"]
        if rank == 0 and not args.no_cpu_baseline and oracle_budget > 0:
            base = oracle_on_same_clusters(r["cfg"], r["seed"], r["start_lattice"], r["start_index"], oracle_budget,
                                           min(oracle_max, r["updates"]))
            # the oracle ran the first n updates of the timed region from the same state: its cluster sizes must be the
            # ones the kernel logged for those updates (north_star: bit-exact per-update cluster sizes)
            ref_sizes = base.pop("sizes")
            gpu_sizes = np.concatenate(r["sizes"])[:len(ref_sizes)].tolist() if r["sizes"] else []
            out["parity_in_timed_region"] = {"updates": len(ref_sizes), "equal": gpu_sizes == ref_sizes,
                                             "compared": "per-update cluster sizes, oracle vs the kernel's log, from update index %d" % r["start_index"]}
            parity_checks.append(out["parity_in_timed_region"]["equal"])
            out["cpu_baseline"] = base
            out["gpu_over_one_cpu_core"] = out["value"] / out["cpu_baseline"]["value"] if out["cpu_baseline"]["value"] else None
        return out

    def measurement_legs(cfg_name: str, seed: int, lattice, index: int, n_updates: int, oracle_budget: float):
        """Row A8 on its own, and the paper's '+ measurement' protocol (E and M after EVERY
        update) three ways on the SAME updates, from the same state: update only; measured inside the persistent kernel
        ("measure" = 1, ONE launch); and the host loop run(1) + observables per update (one launch per update)."""
        c, h = open_chain(cfg_name, seed, False, 0)
        lat_d = torch.from_numpy(lattice).to(dev)
        E_d = torch.zeros(1, dtype=torch.int64, device=dev)
        M_d = torch.zeros(1, dtype=torch.int64, device=dev)

        def timed_observables(cold: bool):
            best = None
            for _ in range(5):
                with torch.cuda.stream(stream):
                    if cold:
                        flush.fill_(1)
                    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    h.observables_into(E_d, M_d, None)
                    e1.record(stream)
                e1.synchronize()
                ms = e0.elapsed_time(e1)
                best = ms if best is None else min(best, ms)
            return best

        def reset():
            h.set_spins(lat_d)
            h.update_index = index

        def timed_run(measure: int, n: int):
            reset()
            h.set_option("measure", measure)
            h.run(3, stream=stream); h.observables()       # first launch of this kernel variant (module load, attributes, logs)
            # reset() loads the lattice again, which clears the handle's run history: the timed run below uses the kernel
            # mode 0 picks WITHOUT a mean cluster size to go by.  Which one that was is read back and reported.
            reset()
            with torch.cuda.stream(stream):
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                h.run(n, stream=stream)
                e1.record(stream)
            e1.synchronize()
            launches[0] += 1
            st = h.stats()
            return e0.elapsed_time(e1), st["flipped"], kernel_of(st)

        reset()
        cold_ms, warm_ms = timed_observables(True), timed_observables(False)
        plain_ms, flipped, plain_kernel = timed_run(0, n_updates)
        meas_ms, flipped_m, meas_kernel = timed_run(1, n_updates)
        assert flipped == flipped_m
        # host loop: one launch + one whole-lattice reduction per update
        h.set_option("measure", 0)
        reset()
        n_loop = min(n_updates, 50 if c.N > (1 << 22) and cfg_name == "C3" else 200)
        sz = torch.zeros(1, dtype=torch.int32, device=dev)
        loop_flipped = 0
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(n_loop):
            h.run(1, stream=stream)
            h.observables_into(E_d, M_d, sz)
            loop_flipped += int(sz.item())
        loop_dt = time.perf_counter() - t0
        launches[0] += 2 * n_loop
        peak, _ = measured_peak_hbm()
        out = {"a8_energy_magnetisation": {"bound": "hbm", "bytes": c.N, "cold_l2_us": cold_ms * 1e3, "warm_l2_us": warm_ms * 1e3,
                                           "cold_l2_gbs": c.N / (cold_ms * 1e-3) / 1e9, "warm_l2_gbs": c.N / (warm_ms * 1e-3) / 1e9,
                                           "peak": peak, "frac_cold": c.N / (cold_ms * 1e-3) / 1e9 / peak,
                                           "note": "wolff_observables(E, M) as a call, device destinations written by the reduction kernel "
                                                   "itself: launch + kernel + one small read-back of the control block + one synchronise"},
               "with_measurement_every_update": {
                   "updates": n_updates, "same_updates_same_state": True,
                   "update_only_ms_per_update": plain_ms / n_updates, "update_only_kernel": plain_kernel, "in_kernel_kernel": meas_kernel,
                   "in_kernel_ms_per_update": meas_ms / n_updates, "in_kernel_over_update_only": meas_ms / plain_ms,
                   "in_kernel_value": flipped / (meas_ms * 1e-3), "unit": UNIT,
                   "in_kernel_protocol": "set_option('measure', 1); run(%d): ONE launch, E and M after every update on the device" % n_updates,
                   "host_loop_updates": n_loop, "host_loop_ms_per_update": loop_dt * 1e3 / n_loop,
                   "host_loop_value": loop_flipped / loop_dt,
                   "host_loop_protocol": "run(1) + observables(E, M, size) per update, host wall clock"}}
        if rank == 0 and not args.no_cpu_baseline and oracle_budget > 0:
            base = oracle_on_same_clusters(c, seed, lattice, index, oracle_budget, n_updates, measured=True)
            base.pop("sizes")
            out["with_measurement_every_update"]["cpu_baseline"] = base
        h.close()
        return out

    def batch_leg(cfg_name: str, R: int, n: int, cold: bool, equil: int, oracle_budget: float, batch_options=None):
        """R independent chains in ONE call (wolff_batch_run): aggregate updates/s and flipped spins/s."""
        c = wl.CONFIGS[cfg_name]
        seeds = [c.seed + 1000 * rank + r for r in range(R)]
        b = binding.WolffBatch(c.dim, c.L, c.J, [c.T] * R, seeds)
        for k, v in (batch_options or {}).items():
            b.set_option(k, v)
        if cold:
            b.set_spins(torch.ones(R * c.N, dtype=torch.int8, device=dev))
        if equil:
            b.run(equil, stream=stream)
            b.stats()
        best = None
        for _ in range(2):
            with torch.cuda.stream(stream):
                flush.fill_(1)
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                b.run(n, stream=stream)
                e1.record(stream)
            e1.synchronize()
            launches[0] += R if (batch_options or {}).get("resident") == 3 else 1
            st = b.stats()
            ms = e0.elapsed_time(e1)
            if best is None or ms < best[0]:
                best = (ms, st)
        b.close()
        ms, st = best
        agg = aggregate_replicas(st["flipped"], st["updates"], ms, world, dev)
        out = {"workload": "%s, %s, %d chains (seeds %d..) in one %s, %d updates each after %d untimed" %
                           (c.name, "cold start" if cold else "random start", R, seeds[0],
                            "call: one thread-block cluster per chain, 7 chains side by side" if (batch_options or {}).get("resident") == 3 else "launch",
                            n, equil),
               "replicas": R * world, "updates_per_s": agg["updates_per_s"], "value": agg["value"], "unit": UNIT,
               "mean_cluster": st["flipped"] / max(st["updates"], 1), "bfs_levels_per_update": st["levels"] / max(st["updates"], 1),
               "ms": ms}
        if rank == 0 and not args.no_cpu_baseline and oracle_budget > 0 and not cold:
            cores = os.cpu_count() or 1
            out["cpu_baseline_one_core"] = oracle_replicas(c, seeds, n, oracle_budget, 1, equil)
            out["cpu_baseline_all_cores"] = oracle_replicas(c, seeds, n, oracle_budget, cores, equil)
        return out

    def reduce_sum(x):
        return all_reduce_scalar(x, "sum", world, dev)

    def reduce_max(x):
        return all_reduce_scalar(x, "max", world, dev)

    # ------------------------------------------------------------------ primary leg
    primary = measure(args.workload, args.updates, args.equil, args.steps, args.warmup, cold=True, sample_clocks=True)
    c = primary["cfg"]
    agg = aggregate_replicas(primary["flipped"], primary["updates"], sum(primary["step_ms"]), world, dev)
    total_ms, updates_all, value = agg["total_ms"], agg["updates"], agg["value"]

    def e2e(h):
        """Same metric through the C-ABI with HOST buffers: every step copies the lattice in from pinned host
        memory, runs, and reads E, M, the size log and the lattice back to the host."""
        updates = args.updates
        lattice = torch.empty(c.N, dtype=torch.int8).pin_memory()
        sizes = torch.empty(updates, dtype=torch.int32).pin_memory()
        em = torch.zeros(2, dtype=torch.int64).pin_memory()
        h.get_spins_into(lattice)
        flipped = 0

        def step():
            h.set_spins(lattice)                                   # H2D: N bytes
            h.run(updates, stream=stream)
            h.observables_into(em.data_ptr(), em.data_ptr() + 8, sizes)   # D2H: 16 + 4*updates bytes
            h.get_spins_into(lattice)                              # D2H: N bytes
            return int(sizes.sum().item())
        for _ in range(args.warmup):
            step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            flipped += step()
        barrier()
        dt = time.perf_counter() - t0
        launches[0] += 3 * args.steps                              # validation, growth, E/M reduction
        return {"flipped": flipped, "seconds": dt, "h2d": c.N, "d2h": c.N + 16 + 4 * updates}

    e = e2e(primary["h"])
    e2e_value = reduce_sum(e["flipped"]) / reduce_max(e["seconds"])
    primary["h"].close()

    peak, peak_src = measured_peak_hbm()
    alg_bytes = algorithmic_bytes(c.dim, primary["flipped"], primary["attempts"]) / args.steps
    avg_growth_s = sum(primary["growth_ms"]) / args.steps * 1e-3
    achieved = alg_bytes / avg_growth_s / 1e9
    traffic = ncu_traffic(args.workload, args.mode, options)
    summary = leg_summary(primary, args.cpu_seconds if world == 1 else 0.0)

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": DTYPE, "data": "synthetic",
        "config": workload_config(c, args.equil, args.updates, world),
        "options": options,
        "updates_per_s": updates_all / (total_ms * 1e-3),
        "updates_timed": primary["updates"],
        "mean_cluster": primary["flipped"] / primary["updates"],
        "ms_per_update_mean": summary["ms_per_update_mean"], "ms_per_update_median": summary["ms_per_update_median"],
        "clocks": primary["clocks"],
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": e["h2d"], "d2h_bytes_per_step": e["d2h"]},
        "roofline": {"bound": "hbm", "kernel": primary.get("kernel", "?") + " (persistent, one launch per step)",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic["bytes"] if traffic else None,
                     "traffic_source": traffic["source"] if traffic else "no committed ncu capture for this workload / mode / options",
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                     "note": "the fraction is ~1e-3 by the nature of the path: a chain of dependent hops (BFS depth x hop latency) on a "
                             "lattice that lives in shared memory, not a stream; latency_roofline is the bound that describes it"},
    }
    for key in ("bfs_depth_per_update", "us_per_bfs_level", "bfs_depth_sample", "cpu_baseline", "gpu_over_one_cpu_core", "parity_in_timed_region"):
        if key in summary:
            out[key] = summary[key]

    single = rank == 0 and world == 1
    if single and not args.no_depth and args.mode == 0 and "bfs_depth_per_update" in summary:
        # latency roofline: T_update >= BFS depth x t_pass, t_pass floor from wolff_microbench [7]
        micro = binding.microbench()
        depth = summary["bfs_depth_per_update"]
        floor_ms = depth * micro["smem_pass_floor_ns"] * 1e-6
        achieved_ms = primary["depth_growth_ms"] / primary["depth_updates"]
        out["latency_roofline"] = {"bound": "latency", "bfs_depth_per_update": depth, "t_pass_floor_ns": micro["smem_pass_floor_ns"],
                                   "bound_ms_per_update": floor_ms, "achieved_ms_per_update": achieved_ms,
                                   "frac": floor_ms / achieved_ms if achieved_ms else None, "sample": summary["bfs_depth_sample"],
                                   "microbench_ns": {k: v for k, v in micro.items()}}
    if single and not args.no_secondary:
        osec = args.leg_cpu_seconds
        # spread over seeds (SURVEY.md 8(d) "Timing protocol"): the same leg on seeds +1, +2, fewer steps
        seeds = {"seed %d" % c.seed: {"value": value, "updates": primary["updates"], "ms_per_update_mean": summary["ms_per_update_mean"],
                                      "ms_per_update_median": summary["ms_per_update_median"], "mean_cluster": out["mean_cluster"]}}
        for off in (1, 2):
            r = measure(args.workload, args.updates, args.equil, max(2, args.steps // 5), 1, cold=True, seed_offset=off, depth_steps=0)
            s = leg_summary(r, 0.0)
            seeds["seed %d" % r["seed"]] = {k: s[k] for k in ("value", "ms_per_update_mean", "ms_per_update_median", "mean_cluster")}
            seeds["seed %d" % r["seed"]]["updates"] = r["updates"]
            r["h"].close()
        out["seeds"] = seeds
        out.update(measurement_legs(args.workload, primary["seed"], primary["start_lattice"], primary["start_index"], args.updates, osec))

        sec = measure(args.secondary, args.secondary_updates, args.equil, args.steps, args.warmup, cold=True)
        sc = sec["cfg"]
        out["secondary"] = dict(workload=sc.name + ", equilibrated variant: cold start + %d untimed updates" % args.equil,
                                updates_per_step=args.secondary_updates, ms_per_step=sum(sec["step_ms"]) / args.steps, **leg_summary(sec, osec))
        sec["h"].close()
        out["secondary"].update(measurement_legs(args.secondary, sec["seed"], sec["start_lattice"], sec["start_index"],
                                                 args.secondary_updates, osec))
        lit = {}
        for name in (args.workload, args.secondary, "C5b"):
            r = measure(name, 1000, 1000, max(1, args.steps // 2), 1, cold=False, depth_steps=0)
            lit[wl.CONFIGS[name].name] = leg_summary(r, osec, oracle_max=r["updates"])
            r["h"].close()
        out["literal_random_start"] = lit
        # the other BASELINE configs ("reported for all five configs"), equilibrated variant
        others = {}
        for name, upd in (("C1", 1000), ("C2", 1000), ("C4", 1000)):
            r = measure(name, upd, args.equil, max(2, args.steps // 2), 1, cold=name != "C1", depth_steps=0)
            others[wl.CONFIGS[name].name] = leg_summary(r, osec, oracle_max=r["updates"])
            r["h"].close()
        out["other_configs_equilibrated"] = others
        # C5b (T = 5.0, disordered phase) from a cold start: equilibrium clusters of a few tens of spins
        r = measure("C5b", 10000, 1000, max(1, args.steps // 2), 1, cold=True, depth_steps=0)
        out["c5b_equilibrated"] = dict(workload=wl.CONFIGS["C5b"].name + ", cold start + 1000 untimed updates", **leg_summary(r, osec, oracle_max=r["updates"]))
        r["h"].close()
    if not args.no_batch and (single or world > 1):
        # f1: independent replicas in one launch -- the small-cluster regime is where one chain
        # cannot fill the chip
        osec = args.leg_cpu_seconds if single else 0.0
        out["batch_replicas"] = {
            "C5b_literal": batch_leg("C5b", args.batch_replicas, 2000, False, 200, osec),
            "C2_literal": batch_leg("C2", 4 * args.batch_replicas, 2000, False, 200, osec),
            "C1_equilibrated": batch_leg("C1", 4 * args.batch_replicas, 2000, False, 1000, 0.0),
            "C2_equilibrated": batch_leg("C2", args.batch_replicas // 2, 40, True, 300, 0.0),
            # the metric's own workloads as replicas: every chain in one 16-CTA cluster (cluster-resident kernel)
            "C3_equilibrated_one_cluster_per_chain": batch_leg("C3", 14, 50, True, 300, 0.0, {"resident": 3}),
            "C5a_equilibrated_one_cluster_per_chain": batch_leg("C5a", 14, 300, True, 300, 0.0, {"resident": 3}),
        }
    out["gpu_launches"] = launches[0]
    out["parity_all_legs"] = {"legs_compared": len(parity_checks), "all_equal": all(parity_checks)}
    return out


# ====================================================================== row A8 on its own (--a8)

def run_a8(args):
    """The one bandwidth-bound kernel of the path, the whole-lattice E/M reduction, at
    the two headline lattices (16 MiB) and at sizes where the launch ramp no longer dominates (256 MiB, 1 GiB), two ways:
    wolff_observables as a call (launch + kernel + read-back of the control block + one synchronise, device destinations)
    and wolff_energy_magnetisation_noalloc on a copy of the same lattice (asynchronous: memset + kernel between the two
    events).  Algorithmic bytes = N (every spin byte read once); the fraction is against the measured HBM peak.  Cold =
    L2 flushed by a 256 MiB write before the timed call (the two large lattices do not fit L2 either way)."""
    import torch
    from paper_1110_0899_b200 import binding, build as cuda_build, workloads as wl
    cuda_build.build()
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    peak, peak_src = measured_peak_hbm()
    out_d = torch.zeros(4, dtype=torch.int64, device=dev)

    def timed(fn, cold: bool, reps: int = 7):
        times = []
        for _ in range(reps):
            with torch.cuda.stream(stream):
                if cold:
                    flush.fill_(1)
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                fn()
                e1.record(stream)
            e1.synchronize()
            times.append(e0.elapsed_time(e1))
        return min(times), statistics.median(times)

    def figures(N, ms_pair):
        best, med = ms_pair
        return {"best_us": best * 1e3, "median_us": med * 1e3, "gbs": N / (best * 1e-3) / 1e9, "frac": N / (best * 1e-3) / 1e9 / peak}

    rows = []
    for dim, L in args.a8_lattices:
        N = L ** dim
        h = binding.Wolff(dim, L, 1.0, wl.TC_2D if dim == 2 else wl.TC_3D, 1)
        call = lambda: h.observables_into(out_d[0:1], out_d[1:2], None)
        call()
        row = {"lattice": "%dD L=%d" % (dim, L), "bytes": N,
               "wolff_observables_call": {"cold": figures(N, timed(call, True)), "warm": figures(N, timed(call, False))}}
        if N <= binding.NOALLOC_MAX_SITES:
            spins = torch.empty(N, dtype=torch.int8, device=dev)
            h.get_spins_into(spins)
            na = lambda: binding.energy_magnetisation_noalloc(spins, dim, L, out_d[2:3], out_d[3:4], stream)
            na()
            row["noalloc_kernel"] = {"cold": figures(N, timed(na, True)), "warm": figures(N, timed(na, False))}
            torch.cuda.synchronize()
            vals = out_d.cpu().tolist()
            assert vals[0:2] == vals[2:4], vals
            del spins
        h.close()
        rows.append(row)
    return {"a8_only": True, "bound": "hbm", "peak": peak, "peak_source": peak_src, "unit": "GB/s", "algorithmic_bytes": "N (one byte per spin)",
            "rows": rows}


# ====================================================================== pass counters of a -DWOLFF_PROFILE build (--profile-counters)

def run_profile_counters(args):
    """What one warp pass of the barrier-free growth kernels costs, from counters compiled in with -DWOLFF_PROFILE
    (libwolff_b200_profile.so, built here; main() points the binding at it).  Not a timing of the product: the counters
    cost cycles themselves.  Per workload (equilibrated C3 and C5a): one launch of `updates` updates on the tiled kernel
    and one on the cluster-resident kernel, and from wolff_get_stats the cycles spent inside passes, the passes, the
    sites expanded, hand-overs / messages / spills, and the launch's prologue / growth / epilogue times."""
    import torch
    from paper_1110_0899_b200 import binding, workloads as wl
    torch.cuda.set_device(0)
    stream = torch.cuda.Stream()
    rows = []
    for name, updates in ((args.workload, args.updates), (args.secondary, args.secondary_updates)):
        c = wl.CONFIGS[name]
        for label, opts in (("growth_tiles_kernel", {"mode": 0, "small_cluster": 0}), ("growth_cluster_kernel", {"mode": 5})):
            h = binding.Wolff(c.dim, c.L, c.J, c.T, c.seed)
            for k, v in opts.items():
                h.set_option(k, v)
            h.set_spins(wl.cold(c.N))
            h.run(args.equil, stream=stream)
            h.observables()
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(stream):
                e0.record(stream)
                h.run(updates, stream=stream)
                e1.record(stream)
            e1.synchronize()
            raw = (ctypes_stats(h))
            row = {"workload": c.name, "kernel": label, "updates": raw[0], "flipped": raw[1], "launch_ms": e0.elapsed_time(e1),
                   "warp_passes": raw[13], "cycles_in_passes": raw[2], "sites_expanded": raw[3],
                   "cycles_per_pass": raw[2] / max(raw[13], 1), "sites_per_pass": raw[3] / max(raw[13], 1),
                   "claim_attempts": raw[7], "ring_pushes": raw[12], "spills": raw[14]}
            if label == "growth_tiles_kernel":
                row.update({"messages": raw[11], "inline_philox_passes": raw[10], "prologue_us": raw[4] * 1e-3, "growth_us": raw[5] * 1e-3,
                            "epilogue_us": raw[6] * 1e-3, "messages_per_spin": raw[11] / max(raw[1], 1)})
            else:
                row.update({"steals": raw[11], "hand_overs": raw[10], "cycles_per_hand_over": raw[4] / max(raw[10], 1),
                            "takes": raw[8], "cycles_per_take": raw[6] / max(raw[8], 1)})
            h.close()
            rows.append(row)
    return {"profile_counters": True, "build": "-DWOLFF_PROFILE (libwolff_b200_profile.so)", "equil": args.equil, "rows": rows}


def ctypes_stats(h):
    """The raw WOLFF_NSTATS words of wolff_get_stats (a profiling build reuses some slots, so no names here)."""
    import ctypes
    from paper_1110_0899_b200 import binding
    buf = (ctypes.c_uint64 * binding.NSTATS)()
    rc = binding.load().wolff_get_stats(h._h, buf)
    if rc != binding.WOLFF_OK:
        raise binding.WolffError(rc, binding.last_error())
    return [int(x) for x in buf]


# ====================================================================== the oracle arm (CPU)

def run_reference(args):
    """--impl reference: the oracle, as it stands, on one host core, on the CUDA arm's workload and config.  The
    chain is brought to the state the CUDA arm's timed region starts from -- cold start, `--equil` updates, the warm-up
    steps -- by the CUDA library when a GPU is there (untimed: the sequential oracle needs minutes for it), else by
    the oracle itself with a shorter equilibration; the timed steps run the oracle alone, each on a bounded number of
    the very updates the CUDA arm times."""
    import oracle
    from paper_1110_0899_b200 import workloads as wl
    c = wl.CONFIGS[args.workload]
    seed = c.seed
    ref = oracle.OracleWolff(c.dim, c.L, c.J, c.T, seed)
    start = None
    try:
        import torch
        if torch.cuda.is_available():
            from paper_1110_0899_b200 import binding, build as cuda_build
            cuda_build.build()
            torch.cuda.set_device(0)
            h = binding.Wolff(c.dim, c.L, c.J, c.T, seed)
            h.set_spins(wl.cold(c.N))
            h.run(args.equil + args.warmup * args.updates)          # what precedes the CUDA arm's timed region
            ref.set_spins(h.get_spins())
            ref.update_index = h.update_index
            start = "state at update index %d taken from the CUDA library (cold start + %d + %d warm-up updates, untimed)" % (
                h.update_index, args.equil, args.warmup * args.updates)
            h.close()
    except Exception as exc:                                       # no GPU / no library: the oracle equilibrates itself
        sys.stderr.write("reference arm: CUDA equilibration unavailable (%s)\n" % exc)
    if start is None:
        ref.set_spins(wl.cold(c.N))
        ref.run(args.reference_equil)
        start = "cold start + %d oracle updates (no GPU for the equilibration: NOT the CUDA arm's clusters)" % args.reference_equil
    per_step = args.reference_updates
    for _ in range(args.warmup):
        ref.run(1)                                                 # warm the caches; the chain moves on by W updates
    flipped = 0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        flipped += int(ref.run(per_step).sum())
    dt = time.perf_counter() - t0
    value = flipped / dt
    sample = "%s; each step = %d consecutive updates of that chain (bounded sample of the %d-update step), %d steps timed" % (
        start, per_step, args.updates, args.steps)
    return {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": DTYPE, "data": "synthetic",
            "config": workload_config(c, args.equil, args.updates, 1),
            "updates_per_s": per_step * args.steps / dt, "mean_cluster": flipped / (per_step * args.steps),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def parse_opt(text: str):
    key, _, value = text.partition("=")
    if not key or not value:
        raise argparse.ArgumentTypeError("expected key=value")
    return key, int(value)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--updates", type=int, default=500, help="updates per step (primary workload); 20 steps = BASELINE's 10,000")
    ap.add_argument("--secondary", default="C5a")
    ap.add_argument("--secondary-updates", type=int, default=1000)
    ap.add_argument("--equil", type=int, default=1000, help="untimed equilibration updates after the cold start")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="oracle budget beside the primary leg")
    ap.add_argument("--leg-cpu-seconds", type=float, default=3.0, help="oracle budget beside each of the other legs")
    ap.add_argument("--reference-updates", type=int, default=20, help="--impl reference: oracle updates per step")
    ap.add_argument("--reference-equil", type=int, default=100, help="--impl reference without a GPU: oracle equilibration updates")
    ap.add_argument("--batch-replicas", type=int, default=296, help="chains of the batch legs at 3D L=256 (x4 at the small lattices)")
    ap.add_argument("--mode", type=int, default=0, help="growth kernel: 0 = default (shared-memory-resident), 4 = level-synchronous tiers")
    ap.add_argument("--opt", type=parse_opt, action="append", default=[], help="wolff_set_option key=value for every chain of the bench")
    ap.add_argument("--no-depth", action="store_true", help="skip the untimed BFS-depth replay of the timed updates")
    ap.add_argument("--no-secondary", action="store_true")
    ap.add_argument("--no-batch", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--profile-counters", action="store_true",
                    help="build with -DWOLFF_PROFILE and print the pass counters of the growth kernels (not a timing of the product)")
    ap.add_argument("--a8", action="store_true", help="only row A8 (the E/M reduction) on its own, at 16 MiB .. 1 GiB lattices")
    ap.add_argument("--a8-lattices", type=lambda t: [tuple(int(x) for x in item.split(":")) for item in t.split(",")],
                    default=[(2, 4096), (3, 256), (2, 16384), (3, 1024)], help="dim:L,dim:L,... for --a8")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        sys.stderr.write("note: fewer than 3 warm-up steps; the timing rules ask for W >= 3\n")

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args)), flush=True)
        return 0
    if args.profile_counters:
        if rank == 0:
            from paper_1110_0899_b200 import build as cuda_build
            os.environ["WOLFF_B200_LIB"] = cuda_build.build(profile=True)      # before the binding is imported
            print(json.dumps(run_profile_counters(args)), flush=True)
        return 0
    if args.a8:
        if rank == 0:
            print(json.dumps(run_a8(args)), flush=True)
        return 0

    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        dist.init_process_group("nccl")
    out = run_b200(args, rank, world)
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    if rank == 0 and not out["parity_all_legs"]["all_equal"]:
        sys.stderr.write("bench: the oracle's cluster sizes differ from the kernel's inside a timed region\n")
        return 1
    return 0


if __name__ == "__main__":
    sys.exit(main())
