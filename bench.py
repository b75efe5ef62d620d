#!/usr/bin/env python
"""bench.py -- XY spin updates/ns of the coloured Metropolis + over-relaxation + PT hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--impl ours|reference]

One STEP = one parallel-tempering cycle of the whole hot path over the synthetic workload (SURVEY.md 8(a)
rows a2-a6): sweeps_per_swap x (Metropolis sweep + OR sweep + measure) and one swap round, replayed from
the captured CUDA graph (xy_run).  `value` = spin updates (one Metropolis OR one over-relaxation update of
one spin of one replica) per nanosecond over all replicas, samples and GPUs, inputs resident in HBM.
Default workload: BASELINE.json configs[4] (L=512, R=64, S=8; 537 MB of angles), the configuration the
metric's target is quoted on.  Samples are independent (Eq. 12), so N GPUs each run their
own S samples (global sample ids rank*S ..) with no data-path collective: weak scaling.

Timing: CUDA events on the library's stream, barrier + synchronize on both sides, max over ranks.  The
working set (537 MB) is larger than the 126 MB L2, so no explicit flush is needed (config.l2 says so).

Roofline objects (all from live CUDA-event timings of this run):
  roofline            the dominant kernel k_phase in the DEFAULT schedule.  The library time-blocks a cycle by sample
                      group (config 4: one 67 MB sample at a time, all 10 sweeps), so the gathers are served by L2:
                      bound = "l2", peak = the L2 read bandwidth measured in this run (xy_l2_bandwidth), and the
                      north star's HBM-equivalent fraction (algorithmic bytes / time / HBM peak) in a field of its own.
  roofline_streaming  the same kernels with xy_set_schedule(S): every launch streams one colour class of ALL samples
                      (537 MB of angles per sweep, no reuse in L2) -- bound = "hbm" against MEASURED_PEAKS.json.
The oracle (oracle/) is used only by the cpu_baseline leg and by --impl reference.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "XY spin updates/ns over all PT replicas+samples"
UNIT = "updates/ns"


# ------------------------------------------------------------------------------------------------------
def measured_peak():
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------------
def host_cpu():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return model, os.cpu_count()


def oracle_replicas(w):
    """replicas of the bounded oracle sample: all of them up to 16 (config 4: 16 of 64, 16.8 MB of angles -- far beyond
    the host's caches like the full state; a step of all 64 would take 14 s)"""
    return min(w.R, 16)


def oracle_sample_run(w, n_steps, n_warmup, seed=0xBA5E, reduce_colours=0):
    """The ONE cpu_baseline definition used by both arms: the oracle as it stands (gcc -O2, fp64, one thread pinned to
    one core) on graph sample 0 of workload w restricted to the first oracle_replicas(w) temperature slots; each step =
    one Metropolis sweep + or_per_sweep over-relaxation sweeps + one measurement + one swap round (orc_run_order with
    sweeps_per_swap = 1).  Returns (updates/ns, seconds of the timed steps, description)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as O
    from paper_1211_3991_b200 import levy
    n_rep = oracle_replicas(w)
    g = levy.build(w.L, w.rho, w.z, w.seed, S=1, reduce_colours=reduce_colours)
    T = w.temperatures()[:n_rep]
    ch = O.Chain(g.row_ptr[0], g.col_idx[0], g.class_ptr(0), T, seed)
    O.lib()
    old = None
    try:                                            # one thread pinned to one core
        old = os.sched_getaffinity(0)
        os.sched_setaffinity(0, {max(old)})
    except (AttributeError, OSError):
        old = None
    try:
        if n_warmup > 0:
            ch.run(n_warmup, 1, w.or_per_sweep, 1)
        t0 = time.perf_counter()
        ch.run(n_steps, 1, w.or_per_sweep, 1)
        dt = time.perf_counter() - t0
    finally:
        if old is not None:
            os.sched_setaffinity(0, old)
    updates = n_steps * (1 + w.or_per_sweep) * w.N * n_rep
    what = (f"graph sample 0 of {w.S}, first {n_rep} of {w.R} replicas; per step one Metropolis + {w.or_per_sweep} OR sweep(s) + "
            f"measure + swap round; fp64 oracle as it stands, gcc -O2, 1 thread pinned to 1 core")
    return updates / dt * 1e-9, dt, what


def workload_config(w, world, measure_every, colours, max_degree, colouring, class_sizes):
    """the `config` object -- identical in both arms"""
    return {"colouring": colouring, "class_sizes_sample0": class_sizes, "workload": w.name, "L": w.L, "N": w.N, "rho": w.rho, "z": w.z, "R": w.R, "S_per_gpu": w.S,
            "T_min": w.T_min, "T_max": w.T_max, "sweeps_per_step": w.sweeps_per_swap, "or_per_sweep": w.or_per_sweep,
            "measure_every": measure_every, "colours": colours, "max_degree": max_degree,
            "step": "one PT cycle: sweeps_per_step x (Metropolis + OR + measure) + one swap round",
            "l2": "inputs larger than L2 (no flush)" if w.S * w.N * w.R * 4 > 126e6 else
                  "working set fits the 126 MB L2 (L2-resident by design; no flush)",
            "parallelism": f"samples x{world}"}


def run_reference(args, w, rank, world):
    """--impl reference: the oracle on the host cores (single pinned thread), a bounded sample per step."""
    if rank != 0:
        return
    from paper_1211_3991_b200 import levy, workloads
    g = levy.build(w.L, w.rho, w.z, w.seed, S=w.S, reduce_colours=workloads.REDUCE_COLOURS if args.colouring == "reduced" else 0)
    val, dt, what = oracle_sample_run(w, args.steps, args.warmup, reduce_colours=workloads.REDUCE_COLOURS if args.colouring == "reduced" else 0)
    model, cores = host_cpu()
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / max(args.steps, 1) * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, world, args.measure_every, int(g.n_colours.max()), int(np.diff(g.row_ptr, axis=1).max()),
                                      args.colouring, np.bincount(g.colour[0]).tolist()),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": what, "steps": args.steps,
                             "seconds": dt, "host_cpu": model, "host_cores": cores},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--samples-per-group", type=int, default=0, help="0 = library default")
    ap.add_argument("--measure-every", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-interleaved", action="store_true", help="skip the interleaved-order measurement")
    ap.add_argument("--colouring", default="reduced", choices=["reduced", "smallest-last"],
                    help="reduced = smallest-last followed by the builder's colour-reducing local search (default)")
    ap.add_argument("--no-aux", action="store_true", help="skip every auxiliary stderr line")
    ap.add_argument("--no-lscan", action="store_true", help="skip config 3's L scan (auxiliary JSON lines on stderr)")
    ap.add_argument("--no-table3", action="store_true", help="skip the paper's Table III workload (auxiliary lines on stderr)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    from paper_1211_3991_b200 import workloads
    w = workloads.CONFIGS[args.config]

    if args.impl == "reference":
        run_reference(args, w, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_1211_3991_b200 import binding as B
    from paper_1211_3991_b200 import levy

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- synthetic inputs: this rank's S samples (global ids rank*S ..), built by the shared builder ----
    sample_base = rank * w.S
    reduce_colours = workloads.REDUCE_COLOURS if args.colouring == "reduced" else 0
    g = levy.build(w.L, w.rho, w.z, w.seed, S=w.S, sample_base=sample_base, reduce_colours=reduce_colours)
    T = w.temperatures()
    seed = 0xB200_1211_3991
    ens = B.Ensemble(g.row_ptr, g.col_idx, g.colour, T, seed, sample_base=sample_base, device=f"cuda:{local_rank}")
    if args.samples_per_group:
        ens.set_schedule(args.samples_per_group)
    sps, orps, me = w.sweeps_per_swap, w.or_per_sweep, args.measure_every
    upd_per_step = sps * (1 + orps) * w.N * w.R * w.S            # per rank

    def timed(fn, n):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record(ens.stream)
        fn(n)
        ev1.record(ens.stream)
        ens.synchronize()
        barrier()
        ms = ev0.elapsed_time(ev1)
        if world > 1:
            t = torch.tensor([ms], device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms

    # ---- warm-up, then the timed region: K full PT cycles ----
    ens.run(args.warmup, sps, orps, me)
    ens.synchronize()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    l0 = ens.launch_count()
    t_wall0 = time.time()
    ms = timed(lambda n: ens.run(n, sps, orps, me), args.steps)
    t_wall1 = time.time()
    launches = ens.launch_count() - l0
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    value = upd_per_step * world * args.steps / (ms * 1e6)

    # ---- dominant kernel (k_phase: the Metropolis / OR colour-class kernel): same launches, same
    #      schedule, without measure/swap, timed with CUDA events on the same stream ----
    peak_hbm, peak_src = measured_peak()
    bpu = w.bytes_per_update()

    def sweep_roofline():
        """MET+OR sweeps in the schedule in force: algorithmic GB/s of the colour-class launches"""
        ens.run_sweeps(2, sps, orps)
        lk0 = ens.launch_count()
        ms_k = timed(lambda n: ens.run_sweeps(n, sps, orps), args.steps)
        n_launch = ens.launch_count() - lk0 - args.steps             # minus the tick kernels
        ach = bpu * upd_per_step * args.steps / (ms_k * 1e-3) * 1e-9  # GB/s, per rank
        return {"achieved": ach, "avg_launch_us": ms_k * 1e3 / max(n_launch, 1), "launches_timed": n_launch,
                "updates_per_launch_avg": upd_per_step * args.steps / max(n_launch, 1),
                "met_or_updates_per_ns": upd_per_step * world * args.steps / (ms_k * 1e6)}

    group, group_bytes = ens.get_schedule()
    l2_stream = B.xy_l2_bandwidth(32 << 20, 0, 5, ens.stream.cuda_stream)      # measured here, on this GPU, in this run
    l2_gather = B.xy_l2_bandwidth(32 << 20, 1, 5, ens.stream.cuda_stream)
    k = sweep_roofline()
    resident = group_bytes <= 126e6 and sps > 1
    roofline = {"bound": "l2" if resident else "hbm", "achieved": k["achieved"], "peak": l2_stream if resident else peak_hbm,
                "unit": "GB/s", "frac": k["achieved"] / (l2_stream if resident else peak_hbm), "traffic": None,
                "kernel": "k_phase<G,CB,0|1> (Metropolis and over-relaxation colour-class launches)",
                "peak_source": ("measured in this run: xy_l2_bandwidth(32 MiB, linear 16-byte loads, L1 bypassed)" if resident
                                else peak_src),
                "schedule": f"time-blocked: {group} sample(s) = {group_bytes / 1e6:.0f} MB per launch group, all {sps} sweeps "
                            f"of the cycle before the next group" + (" -- the group stays resident in the 126 MB L2" if resident else ""),
                "l2_stream_gbs": l2_stream, "l2_gather256_gbs": l2_gather, "frac_of_l2_gather256": k["achieved"] / l2_gather,
                "hbm_peak_gbs": peak_hbm, "hbm_peak_source": peak_src,
                "hbm_equivalent_frac": k["achieved"] / peak_hbm,
                "hbm_equivalent_note": "north star's counting (algorithmic bytes / time / HBM peak); the gathers of this "
                                       "schedule are served by L2, so this is not an HBM utilisation",
                "traffic_note": "dram__bytes per launch: profiles/ (ncu --set full at the benched commit); not read at run time",
                "bytes_per_update": bpu, **{kk: k[kk] for kk in ("updates_per_launch_avg", "avg_launch_us", "launches_timed",
                                                                  "met_or_updates_per_ns")}}
    roofline["path"] = ens.path_name(orps)
    if ens.get_path(orps)[0] == 2:
        roofline["kernel"] = "k_cycle<G,ORDER> (cluster path: whole cycles per launch)"
        roofline["schedule"] = ("cluster path: every sample stays in the distributed shared memory of its thread-block cluster for the "
                                "whole launch; neither L2 nor HBM carries the gathers, the bound is the latency chain of a colour "
                                "class (DESIGN.md 7.2) -- frac is the algorithmic bytes against the L2 bandwidth, for reference only")

    # ---- what actually bounds k_phase: ISSUE SLOTS.  peak = 4 warp schedulers per SM x SMs x SM clock warp
    #      instructions per second; the warp instructions per row (one row = 64 spin updates: 32 lanes x 2 slots) of the
    #      Metropolis launch and of the over-relaxation + measurement launch are ncu counts of smsp__inst_executed.sum /
    #      rows (profiles/r2a_full_warm.md, r2f_full_warm.md: G = 32; profiles/r2d_cfg2_full_warm.md: G = 16), constants of
    #      the kernels as built, not of this run.  One PT-cycle step executes one row of each per 128 updates. ----
    if ens.get_path(orps)[0] == 1 and w.R % 2 == 0 and w.R >= 32 and orps == 1:
        inst_met, inst_orm = (238.8, 199.9) if w.R % 64 == 0 else (338.7, 428.4)
        props = torch.cuda.get_device_properties(local_rank)
        sm_ghz = (clocks["sm_mhz"] if clocks and clocks.get("sm_mhz") else 1965.0) * 1e-3
        peak_inst = 4.0 * props.multi_processor_count * sm_ghz                      # G warp instructions / s
        peak_upd = peak_inst / (inst_met + inst_orm) * 128.0                         # updates / ns of the full cycle
        roofline["issue"] = {"bound": "alu", "achieved": value / world, "peak": peak_upd, "unit": UNIT, "frac": value / world / peak_upd,
                             "peak_derivation": f"4 schedulers x {props.multi_processor_count} SMs x {sm_ghz:.3f} GHz = {peak_inst:.0f} G warp "
                                                f"instructions/s; {inst_met} (Metropolis) + {inst_orm} (over-relaxation + measurement) warp "
                                                "instructions per 128 updates (ncu, profiles/); applies to `value` (the full cycle)"}

    # ---- the genuinely streaming schedule: one launch per colour class over ALL samples (every sweep re-reads the whole
    #      state from HBM) -- the number "fraction of the HBM roofline" is literally about ----
    streaming = None
    if group < w.S:
        ens.set_schedule(w.S)
        ens.run(2, sps, orps, me)
        ms_s = timed(lambda n: ens.run(n, sps, orps, me), args.steps)
        ks = sweep_roofline()
        ens.set_schedule(args.samples_per_group)
        streaming = {"bound": "hbm", "achieved": ks["achieved"], "peak": peak_hbm, "unit": "GB/s", "frac": ks["achieved"] / peak_hbm,
                     "peak_source": peak_src, "schedule": f"xy_set_schedule({w.S}): every launch covers all {w.S} samples "
                     f"({w.S * w.N * w.R * 4 / 1e6:.0f} MB of angles per sweep, no L2 reuse across sweeps)",
                     "value_full_cycle": upd_per_step * world * args.steps / (ms_s * 1e6),
                     **{kk: ks[kk] for kk in ("updates_per_launch_avg", "avg_launch_us", "launches_timed", "met_or_updates_per_ns")}}

    # ---- the interleaved sweep order (xy_set_order(1)): per colour class Metropolis then
    #      over-relaxation from ONE gather -- a different valid chain with its own oracle mode and parity tests.
    #      `value` and `roofline` above stay on the default order; this object reports the same two measurements.
    #      Its bytes: one own-angle read, one write, z gathers and z/R indices per update PAIR. ----
    interleaved = None
    if not args.no_interleaved and orps == 1:
        ens.set_order(1)
        ens.run(args.warmup, sps, orps, me)
        ms_i = timed(lambda n: ens.run(n, sps, orps, me), args.steps)
        ki = sweep_roofline()
        ens.set_order(0)
        ach_i = ki["achieved"] * 0.5                  # bpu per update pair
        interleaved = {"value": upd_per_step * world * args.steps / (ms_i * 1e6), "unit": UNIT, "ms_per_step": ms_i / args.steps,
                       "met_or_updates_per_ns": ki["met_or_updates_per_ns"], "bytes_per_update": bpu / 2,
                       "roofline": {"bound": "l2" if resident else "hbm", "achieved": ach_i, "peak": l2_stream if resident else peak_hbm,
                                    "unit": "GB/s", "frac": ach_i / (l2_stream if resident else peak_hbm),
                                    "hbm_equivalent_frac": ach_i / peak_hbm}}

    # ---- end to end through the C ABI with HOST buffers: every step uploads the step's input state from pinned host
    #      memory (xy_set_theta_async: one copy per sample group on a second stream; group g+1 uploads while group g
    #      sweeps), runs one PT cycle and reads the step's result -- the accumulated observables [S][R][8] fp64 and the
    #      temperature labels -- back to the host ----
    e2e = None
    if not args.no_e2e:
        nbytes = w.S * w.N * w.R * 4
        host = torch.empty((w.S, w.N, w.R), dtype=torch.float32, pin_memory=True).numpy()
        ens.get_theta(out=host)
        n_e2e = max(2, args.steps)
        sink = []

        def e2e_steps(n):
            for _ in range(n):
                ens.set_theta_async(host)                 # H2D, pinned, group by group
                ens.run(1, sps, orps, me)
                sink.append(ens.read_accumulators())      # D2H result (synchronises)
                sink.append(ens.get_labels())
                del sink[:-2]
        e2e_steps(2)
        barrier()
        t0 = time.perf_counter()
        e2e_steps(n_e2e)
        barrier()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": upd_per_step * world * n_e2e / (dt * 1e9), "unit": UNIT, "steps": n_e2e,
               "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": w.S * w.R * 8 * 8 + w.S * w.R * 4,
               "what": "xy_set_theta_async(pinned host state, copy of sample group g+1 overlapping the sweeps of group g) + "
                       "xy_run(1 cycle) + xy_read_accumulators + xy_get_labels (host)"}

    # ---- CPU baseline: the oracle on a bounded sample of the same workload (rank 0, N = 1 only); the SAME definition
    #      as the reference arm (oracle_sample_run), fewer steps so that the default run stays short ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        per_step = (1 + orps) * w.N * oracle_replicas(w) / 2.4e6          # seconds, at the oracle's ~2.4e6 updates/s
        n_cpu = int(min(args.steps, max(2, 12.0 / per_step)))
        v, dt, what = oracle_sample_run(w, n_cpu, 1, reduce_colours=reduce_colours)
        model, cores = host_cpu()
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt, "steps": n_cpu, "sample": what,
               "host_cpu": model, "host_cores": cores}

    if rank == 0:
        info = B.xy_graph_info(ens.graph)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": workload_config(w, world, me, info["q_max"], info["max_degree"], args.colouring,
                                          np.bincount(g.colour[0]).tolist()),
                "roofline": roofline, "roofline_streaming": streaming, "interleaved": interleaved, "cpu_baseline": cpu, "e2e": e2e,
                "gpu_launches": int(launches), "clocks": clocks}
        print(json.dumps(line), flush=True)

    def aux(obj):
        print(json.dumps(obj), file=sys.stderr, flush=True)

    def event_timed(e, fn, n):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e.synchronize()
        ev0.record(e.stream)
        fn(n)
        ev1.record(e.stream)
        e.synchronize()
        return ev0.elapsed_time(ev1)

    # ---- auxiliary row: structure factor at k_min, one streaming pass over theta; its own
    #      roofline line goes to stderr so that stdout keeps the single contract line ----
    if rank == 0 and not args.no_aux:
        x = (g.new_to_old % w.L).astype(np.int32)
        y = (g.new_to_old // w.L).astype(np.int32)
        ens.set_coords(w.L, w.L, x, y)
        for _ in range(3):
            ens.measure_fourier()
        n_f = 20
        ms_f = event_timed(ens, lambda n: [ens.measure_fourier() for _ in range(n)], n_f) / n_f
        bytes_f = w.S * w.N * (4.0 * w.R + 4.0)                 # theta once + packed coordinates
        aux({"aux": "xy_measure_fourier (k_fourier2)", "workload": w.name, "us_per_launch": ms_f * 1e3,
             "spins_per_ns": w.S * w.N * w.R / (ms_f * 1e6),
             "roofline": {"bound": "hbm", "achieved": bytes_f / (ms_f * 1e-3) * 1e-9, "peak": peak_hbm, "unit": "GB/s",
                          "frac": bytes_f / (ms_f * 1e-3) * 1e-9 / peak_hbm, "bytes_per_spin": 4.0 + 4.0 / w.R}})

    # ---- auxiliary row: random-walk self-return histogram, the paper's 4e4 walkers per graph;
    #      kernel time from CUDA events around the k_random_walk launch alone (xy_random_walk_kernel_us) ----
    if rank == 0 and not args.no_aux:
        n_w, n_t = 40_000, 1024
        rng = np.random.default_rng(1)
        st = np.stack([rng.choice(np.where(np.diff(g.row_ptr[s]) > 2)[0], n_w) for s in range(w.S)]).astype(np.int32)
        B.xy_random_walk(ens.graph, st, 16, seed)
        t0 = time.perf_counter()
        hist = B.xy_random_walk(ens.graph, st, n_t, seed)
        dt = time.perf_counter() - t0
        us = B.xy_random_walk_kernel_us()
        aux({"aux": "xy_random_walk (k_random_walk)", "workload": w.name, "walkers_per_graph": n_w, "steps": n_t,
             "kernel_us": us, "walker_steps_per_ns": w.S * n_w * n_t / (us * 1e3), "seconds_call_incl_alloc_and_copies": dt,
             "bound": "latency (two dependent random 32-byte reads per step, served by L2: one sample's graph is 8.4 MB)",
             "sector_gbs": w.S * n_w * n_t * 64 / (us * 1e3), "returns_at_t2": int(hist[:, 2].sum())})
    ens.close()

    # ---- auxiliary rows: BASELINE.json configs[3]'s throughput sweep over L at 512 replica-samples (R = 32 x S = 16) ----
    if rank == 0 and world == 1 and not args.no_aux and not args.no_lscan:
        for L in (32, 64, 128, 256):
            wl = workloads.lscan(L)
            gl = levy.build(wl.L, wl.rho, wl.z, wl.seed, S=wl.S, reduce_colours=reduce_colours)
            el = B.Ensemble(gl.row_ptr, gl.col_idx, gl.colour, wl.temperatures(), seed)
            el.run(5, sps, orps, me)
            n = max(10, int(2000 * 64 * 64 / (L * L)))
            msl = event_timed(el, lambda k_: el.run(k_, sps, orps, me), n)
            msk = event_timed(el, lambda k_: el.run_sweeps(k_, sps, orps), n)
            el.set_order(1)
            el.run(2, sps, orps, me)
            msi = event_timed(el, lambda k_: el.run(k_, sps, orps, me), n)
            upd = sps * (1 + orps) * wl.N * wl.R * wl.S * n
            gl_, gb_ = el.get_schedule()
            aux({"lscan": wl.name, "updates_per_ns": upd / (msl * 1e6), "met_or_updates_per_ns": upd / (msk * 1e6),
                 "interleaved_updates_per_ns": upd / (msi * 1e6), "ms_per_step": msl / n, "steps": n, "path": el.path_name(),
                 "roofline": {"bound": "l2" if gb_ <= 126e6 else "hbm", "achieved": wl.bytes_per_update() * upd / (msk * 1e6),
                              "peak": l2_stream if gb_ <= 126e6 else peak_hbm, "unit": "GB/s",
                              "frac": wl.bytes_per_update() * upd / (msk * 1e6) / (l2_stream if gb_ <= 126e6 else peak_hbm),
                              "hbm_equivalent_frac": wl.bytes_per_update() * upd / (msk * 1e6) / peak_hbm}})
            el.close()

    # ---- auxiliary rows: the paper's own timing workload (Table III): periodic square lattice,
    #      N = 2^14, z = 4, two colours; time per spin = run time / (N * N_T * MCS) for Metropolis alone, over-relaxation
    #      alone and Metropolis + a parallel-tempering swap round EVERY sweep, fp32 + fast intrinsics.  The
    #      paper's GTX480 numbers are context, not a target. ----
    if rank == 0 and world == 1 and not args.no_aux and not args.no_table3:
        for (R3, S3) in ((64, 1), (64, 8)):
            w3 = workloads.square_lattice(128, R3, 0.7, 1.3, S3)
            g3 = levy.build(w3.L, w3.rho, w3.z, w3.seed, S=1)
            e3 = B.Ensemble(np.tile(g3.row_ptr, (S3, 1)), np.tile(g3.col_idx, (S3, 1)), np.tile(g3.colour, (S3, 1)),
                            w3.temperatures(), seed)
            n = 200
            spins = w3.N * R3 * S3
            e3.run_sweeps(5, 10, 0); t_met = event_timed(e3, lambda k_: e3.run_sweeps(k_, 10, 0), n) * 1e6 / (n * 10 * spins)
            e3.run(5, 1, 0, 0); t_pt = event_timed(e3, lambda k_: e3.run(k_, 1, 0, 0), n * 10) * 1e6 / (n * 10 * spins)
            e3.run_sweeps(5, 10, 1)           # OR alone = (Metropolis + OR sweeps) - (Metropolis sweeps), both from captured graphs
            t_or = event_timed(e3, lambda k_: e3.run_sweeps(k_, 10, 1), n) * 1e6 / (n * 10 * spins) - t_met
            aux({"aux": "paper Table III workload (square lattice N = 2^14, PBC, z = 4, Q = 2)", "R": R3, "S": S3,
                 "ns_per_spin": {"MET": t_met, "OR (MET+OR minus MET)": t_or, "MET+PT every sweep": t_pt}, "path": e3.path_name(),
                 "paper_gtx480_ns_per_spin": {"MET": 0.635, "OR": 0.36, "MET+PT": 1.88, "source": "PAPER.md:474-480"}})
            e3.close()
    if world > 1:
        dist.barrier()          # rank 0 may still be in its auxiliary measurements
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
