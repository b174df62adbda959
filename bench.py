#!/usr/bin/env python
"""bench.py -- throughput of the Wolff single-cluster hot path on B200, one JSON line.

A "step" is one pass of the whole hot path over one batch:
    wolff_run(h, U, stream)          -- U single-cluster updates as ONE persistent kernel launch (A1-A7)
    wolff_observables(h, E, M, sizes) -- the whole-lattice E/M reduction (A8) + read-back of the size log (A9)
on the workload BASELINE.json's metric is quoted on: 2D L=4096 at T_c (primary; `value`) and 3D L=256 at T_c
(reported under "secondary").  Start state: the 'equilibrated' variant of SURVEY.md 8(d) -- cold start followed by
`--equil` untimed updates -- because the literal random start never reaches T_c-sized clusters within the configured
1,000 + 10,000 updates; the literal variant is reported as updates/s under "literal_random_start".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--workload C3] [--updates U]

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
L2_FLUSH_BYTES = 256 << 20          # > 126 MB L2


def measured_peak_hbm():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, STREAM-style copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ncu `--set full` DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum) of one launch of the growth kernel,
# bytes: profiles/r1_growth_tiles_C3.md (a 10-update C3 launch: the 16 MiB lattice is read once in the prologue; the
# write-back and all queue traffic stay in L2).  It does not grow with the updates per launch.
NCU_TRAFFIC_BYTES_PER_LAUNCH = 22624256 + 493056


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

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    def measure(cfg_name: str, updates: int, equil: int, steps: int, warmup: int, cold: bool):
        c = wl.CONFIGS[cfg_name]
        seed = c.seed + rank
        h = binding.Wolff(c.dim, c.L, c.J, c.T, seed)
        if args.mode:
            h.set_option("mode", args.mode)
        if cold:
            h.set_spins(wl.cold(c.N))
        if equil:
            h.run(equil, stream=stream)
            h.observables()
        E_d = torch.zeros(1, dtype=torch.int64, device=dev)
        M_d = torch.zeros(1, dtype=torch.int64, device=dev)
        sizes_d = torch.zeros(updates, dtype=torch.int32, device=dev)
        flipped = attempts = levels = 0
        step_ms, growth_ms = [], []
        # BFS depth of the clusters the timed steps grow (a property of the workload): the
        # level-synchronous kernel (mode 4) replays the same updates from the same lattice, untimed, and counts levels
        twin = None
        if args.mode == 0 and not args.no_depth:
            twin = binding.Wolff(c.dim, c.L, c.J, c.T, seed)
            twin.set_option("mode", 4)
            snapshot = torch.empty(c.N, dtype=torch.int8, device=dev)

        def one_step(timed: bool):
            nonlocal flipped, attempts, levels
            if timed and twin is not None:
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
                step_ms.append(e0.elapsed_time(e2))
                growth_ms.append(e0.elapsed_time(e1))
                st = h.stats()
                flipped += st["flipped"]; attempts += st["claim_attempts"]
                assert int(sizes_d.sum().item()) == st["flipped"]
                if twin is not None:
                    twin.run(updates, stream=stream)
                    ts = twin.stats()
                    assert ts["flipped"] == st["flipped"]
                    st = ts
                levels += st["levels_cta"] + st["levels_cluster"] + st["levels_grid"]

        for _ in range(warmup):
            one_step(False)
        barrier()
        t0 = time.perf_counter()
        with ClockSampler(local_rank) as clocks:
            for _ in range(steps):
                one_step(True)
            barrier()
        wall = time.perf_counter() - t0
        if twin is not None:
            twin.close()
        res = {"cfg": c, "h": h, "flipped": flipped, "attempts": attempts, "levels": levels, "updates": updates * steps,
               "step_ms": step_ms, "growth_ms": growth_ms, "wall_s": wall, "clocks": clocks.summary()}
        return res

    def measurement_legs(h, cfg, n_updates: int):
        """Row A8 on its own (the E/M reduction through the C-ABI, L2 flushed / warm) and the paper's '+ measurement'
        protocol: E and M after EVERY update, i.e. run(1) + observables in a loop."""
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
        cold_ms, warm_ms = timed_observables(True), timed_observables(False)
        sz = torch.zeros(1, dtype=torch.int32, device=dev)
        flipped = 0
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(n_updates):
            h.run(1, stream=stream)
            h.observables_into(E_d, M_d, sz)
            flipped += int(sz.item())
        dt = time.perf_counter() - t0
        peak, _ = measured_peak_hbm()
        return {"a8_energy_magnetisation": {"bound": "hbm", "bytes": cfg.N, "cold_l2_us": cold_ms * 1e3, "warm_l2_us": warm_ms * 1e3,
                                            "cold_l2_gbs": cfg.N / (cold_ms * 1e-3) / 1e9, "warm_l2_gbs": cfg.N / (warm_ms * 1e-3) / 1e9,
                                            "peak": peak, "frac_cold": cfg.N / (cold_ms * 1e-3) / 1e9 / peak,
                                            "note": "wolff_observables(E, M) with device pointers: the reduction kernel, two 8-byte copies and "
                                                    "a stream synchronise; at 16 MiB the call is launch-latency bound"},
                "with_measurement_every_update": {"updates": n_updates, "updates_per_s": n_updates / dt, "value": flipped / dt, "unit": UNIT,
                                                  "ms_per_update": dt * 1e3 / n_updates, "protocol": "run(1) + observables(E, M, size) per update, host wall clock"}}

    def e2e(cfg_name: str, updates: int, steps: int, warmup: int, h):
        """Same metric through the C-ABI with HOST buffers: every step copies the lattice in from pinned host
        memory, runs, and reads E, M, the size log and the lattice back to the host."""
        c = wl.CONFIGS[cfg_name]
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
        for _ in range(warmup):
            step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            flipped += step()
        barrier()
        dt = time.perf_counter() - t0
        return {"flipped": flipped, "seconds": dt, "h2d": c.N, "d2h": c.N + 16 + 4 * updates}

    def reduce_sum(x):
        return all_reduce_scalar(x, "sum", world, dev)

    def reduce_max(x):
        return all_reduce_scalar(x, "max", world, dev)

    primary = measure(args.workload, args.updates, args.equil, args.steps, args.warmup, cold=True)
    c = primary["cfg"]
    agg = aggregate_replicas(primary["flipped"], primary["updates"], sum(primary["step_ms"]), world, dev)
    total_ms, updates_all, value = agg["total_ms"], agg["updates"], agg["value"]

    e = e2e(args.workload, args.updates, args.steps, args.warmup, primary["h"])
    e2e_value = reduce_sum(e["flipped"]) / reduce_max(e["seconds"])

    peak, peak_src = measured_peak_hbm()
    alg_bytes = algorithmic_bytes(c.dim, primary["flipped"], primary["attempts"]) / args.steps
    avg_growth_s = sum(primary["growth_ms"]) / args.steps * 1e-3
    achieved = alg_bytes / avg_growth_s / 1e9

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int8 spins / uint32 bond words / int64 sums", "data": "synthetic",
        "config": {"workload": "%s, equilibrated variant: cold start + %d untimed updates, seed %d(+rank)" % (c.name, args.equil, c.seed),
                   "updates_per_step": args.updates, "step": "wolff_run(U) + wolff_observables (E, M, size log)",
                   "l2": "flushed between steps by a %d MiB write, outside the timed events" % (L2_FLUSH_BYTES >> 20),
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "updates_per_s": updates_all / (total_ms * 1e-3),
        "mean_cluster": primary["flipped"] / primary["updates"],
        "bfs_depth_per_update": primary["levels"] / primary["updates"],
        "us_per_bfs_level": sum(primary["growth_ms"]) * 1e3 / max(primary["levels"], 1),
        "clocks": primary["clocks"],
        "gpu_launches": 2 * args.steps,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": e["h2d"], "d2h_bytes_per_step": e["d2h"]},
        "roofline": {"bound": "hbm", "kernel": ("growth_tiles_kernel" if args.mode == 0 else "growth_kernel") + " (persistent, one launch per step)",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": alg_bytes,
                     "note": "latency-bound by design: the path is a chain of dependent hops (BFS depth x hop latency), not a stream; "
                             "see bfs_depth_per_update and us_per_bfs_level"},
    }

    if rank == 0 and world == 1 and not args.no_depth and args.mode == 0:
        # latency roofline: T_update >= BFS depth x t_pass, t_pass floor from wolff_microbench [7]
        micro = binding.microbench()
        depth = primary["levels"] / primary["updates"]
        floor_ms = depth * micro["smem_pass_floor_ns"] * 1e-6
        achieved_ms = sum(primary["growth_ms"]) / primary["updates"]
        out["latency_roofline"] = {"bfs_depth_per_update": depth, "t_pass_floor_ns": micro["smem_pass_floor_ns"],
                                   "bound_ms_per_update": floor_ms, "achieved_ms_per_update": achieved_ms,
                                   "frac": floor_ms / achieved_ms if achieved_ms else None,
                                   "microbench_ns": {k: v for k, v in micro.items()}}
    if rank == 0 and world == 1 and not args.no_secondary:
        out.update(measurement_legs(primary["h"], c, 50))
        primary["h"].close()
        sec = measure(args.secondary, args.secondary_updates, args.equil, args.steps, args.warmup, cold=True)
        sc = sec["cfg"]
        ms = sum(sec["step_ms"])
        out["secondary"] = {"workload": sc.name + ", equilibrated variant", "value": sec["flipped"] / (ms * 1e-3), "unit": UNIT,
                            "updates_per_s": sec["updates"] / (ms * 1e-3), "ms_per_step": ms / args.steps,
                            "updates_per_step": args.secondary_updates, "mean_cluster": sec["flipped"] / sec["updates"],
                            "bfs_depth_per_update": sec["levels"] / sec["updates"],
                            "us_per_bfs_level": sum(sec["growth_ms"]) * 1e3 / max(sec["levels"], 1)}
        out["secondary"].update(measurement_legs(sec["h"], sc, 500))
        sec["h"].close()
        lit = {}
        for name in (args.workload, args.secondary, "C5b"):
            r = measure(name, 1000, 1000, max(1, args.steps // 2), 1, cold=False)
            ms = sum(r["step_ms"])
            lit[wl.CONFIGS[name].name] = {"updates_per_s": r["updates"] / (ms * 1e-3), "mean_cluster": r["flipped"] / r["updates"]}
            r["h"].close()
        out["literal_random_start"] = lit
        # C5b (T = 5.0, disordered phase) from a cold start: equilibrium clusters of a few tens of spins
        r = measure("C5b", 10000, 1000, max(1, args.steps // 2), 1, cold=True)
        ms = sum(r["step_ms"])
        out["c5b_equilibrated"] = {"workload": wl.CONFIGS["C5b"].name + ", cold start + 1000 untimed updates", "updates_per_s": r["updates"] / (ms * 1e-3),
                                   "value": r["flipped"] / (ms * 1e-3), "unit": UNIT, "mean_cluster": r["flipped"] / r["updates"]}
        r["h"].close()

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, budget_s=args.cpu_seconds)
    return out


# ====================================================================== the oracle arm (CPU)

def cpu_baseline(cfg_name: str, budget_s: float):
    """The oracle as it stands, one host core, on a bounded sample of the same workload."""
    import oracle
    from paper_1110_0899_b200 import workloads as wl
    c = wl.CONFIGS[cfg_name]
    ref = oracle.OracleWolff(*c.create_args())
    ref.set_spins(wl.cold(c.N))
    flipped = n = 0
    t0 = time.perf_counter()
    while time.perf_counter() - t0 < budget_s:
        flipped += int(ref.run(1)[0])
        n += 1
    dt = time.perf_counter() - t0
    return {"value": flipped / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "%s cold start, first %d updates (%.1f s of CPU work, %d spins flipped)" % (c.name, n, dt, flipped),
            "updates_per_s": n / dt, "host_cores_available": os.cpu_count()}


def run_reference(args):
    """--impl reference: the oracle timed on the host; each step is a bounded sample of the workload."""
    import oracle
    from paper_1110_0899_b200 import workloads as wl
    c = wl.CONFIGS[args.workload]
    ref = oracle.OracleWolff(*c.create_args())
    ref.set_spins(wl.cold(c.N))
    per_step = args.reference_updates
    for _ in range(args.warmup):
        ref.run(per_step)
    flipped = 0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        flipped += int(ref.run(per_step).sum())
    dt = time.perf_counter() - t0
    value = flipped / dt
    sample = "%s cold start, updates %d..%d (%d per step)" % (c.name, args.warmup * per_step,
                                                             (args.warmup + args.steps) * per_step - 1, per_step)
    return {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int8 spins / uint32 bond words / int64 sums", "data": "synthetic",
            "config": {"workload": "%s, cold start (bounded sample)" % c.name, "updates_per_step": per_step,
                       "step": "oracle_run(U)", "parallelism": "one host core"},
            "updates_per_s": per_step * args.steps / dt,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--updates", type=int, default=100, help="updates per step (primary workload)")
    ap.add_argument("--secondary", default="C5a")
    ap.add_argument("--secondary-updates", type=int, default=1000)
    ap.add_argument("--equil", type=int, default=1000, help="untimed equilibration updates after the cold start")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--reference-updates", type=int, default=3)
    ap.add_argument("--mode", type=int, default=0, help="growth kernel: 0 = default (shared-memory-resident), 4 = level-synchronous tiers")
    ap.add_argument("--no-depth", action="store_true", help="skip the untimed BFS-depth replay of the timed updates")
    ap.add_argument("--no-secondary", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        sys.stderr.write("note: fewer than 3 warm-up steps; the timing rules ask for W >= 3\n")

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args)), flush=True)
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
    return 0


if __name__ == "__main__":
    sys.exit(main())
