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
def oracle_sample_run(w, n_replicas, n_steps, seed, with_measure=True):
    """Time the oracle, as it stands, on ONE graph sample of workload w restricted to the first n_replicas
    slots: each step = one Metropolis sweep + or_per_sweep OR sweeps (+ one measure).  Returns (updates/ns, s)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as O
    from paper_1211_3991_b200 import levy
    g = levy.build(w.L, w.rho, w.z, w.seed, S=1)
    T = w.temperatures()[:n_replicas]
    ch = O.Chain(g.row_ptr[0], g.col_idx[0], g.class_ptr(0), T, seed)
    O.lib()
    t0 = time.perf_counter()
    # sweeps_per_swap = 1 cycle = 1 Metropolis + or_per_sweep OR sweeps + measure + (cheap) swap round
    ch.run(n_steps, 1, w.or_per_sweep, 1 if with_measure else 0)
    dt = time.perf_counter() - t0
    updates = n_steps * (1 + w.or_per_sweep) * w.N * n_replicas
    return updates / dt * 1e-9, dt


def run_reference(args, w, rank):
    """--impl reference: the oracle on the host cores (single thread), bounded sample per step."""
    if rank != 0:
        return
    n_rep = min(w.R, max(1, int(2.0e6 / (w.N * (1 + w.or_per_sweep)))))     # ~2e6 updates (~1 s) per step
    if args.warmup > 0:
        oracle_sample_run(w, n_rep, args.warmup, 0xBA5E)
    val, dt = oracle_sample_run(w, n_rep, args.steps, 0xBA5E)
    sample = (f"1 of {w.S} samples, first {n_rep} of {w.R} replicas, per step one Metropolis + {w.or_per_sweep} OR "
              f"sweep(s) + measure + swap round (fp64 oracle, gcc -O2, 1 thread)")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / max(args.steps, 1) * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "L": w.L, "rho": w.rho, "z": w.z, "R": w.R, "S": w.S, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
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
    ap.add_argument("--no-aux", action="store_true", help="skip the structure-factor kernel's stderr line")
    ap.add_argument("--lscan", action="store_true", help="also time config 3's L scan (extra JSON lines, stderr)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    from paper_1211_3991_b200 import workloads
    w = workloads.CONFIGS[args.config]

    if args.impl == "reference":
        run_reference(args, w, rank)
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
    g = levy.build(w.L, w.rho, w.z, w.seed, S=w.S, sample_base=sample_base)
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
    ens.run_sweeps(2, sps, orps)
    lk0 = ens.launch_count()
    ms_k = timed(lambda n: ens.run_sweeps(n, sps, orps), args.steps)
    n_class_launches = ens.launch_count() - lk0 - args.steps         # minus the tick kernels
    bytes_alg = w.bytes_per_update() * upd_per_step * args.steps      # per rank
    achieved = bytes_alg / (ms_k * 1e-3) * 1e-9                       # GB/s
    peak, peak_src = measured_peak()
    traffic = None          # ncu dram__bytes per launch of this kernel on this workload (profiles/roofline_traffic.md)
    tc = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if os.path.exists(tc):
        try:
            import csv
            for row in csv.DictReader(open(tc)):
                if row["workload"] == w.name:
                    traffic = float(row["dram_bytes_per_launch"])
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "kernel": "k_phase<G,CB,0|1> (Metropolis and over-relaxation colour-class launches)",
                "peak_source": peak_src, "bytes_per_update": w.bytes_per_update(),
                "updates_per_launch_avg": upd_per_step * args.steps / max(n_class_launches, 1),
                "avg_launch_us": ms_k * 1e3 / max(n_class_launches, 1), "launches_timed": n_class_launches,
                "met_or_updates_per_ns": upd_per_step * world * args.steps / (ms_k * 1e6)}

    # ---- the interleaved sweep order (xy_set_order(1)): per colour class Metropolis then
    #      over-relaxation from ONE gather -- a different valid chain with its own oracle mode and parity tests.
    #      `value` and `roofline` above stay on the default order; this object reports the same two measurements. ----
    interleaved = None
    if not args.no_interleaved and orps == 1:
        ens.set_order(1)
        ens.run(args.warmup, sps, orps, me)
        ms_i = timed(lambda n: ens.run(n, sps, orps, me), args.steps)
        ens.run_sweeps(2, sps, orps)
        ms_ik = timed(lambda n: ens.run_sweeps(n, sps, orps), args.steps)
        ens.set_order(0)
        ach_i = bytes_alg / (ms_ik * 1e-3) * 1e-9
        interleaved = {"value": upd_per_step * world * args.steps / (ms_i * 1e6), "unit": UNIT, "ms_per_step": ms_i / args.steps,
                       "met_or_updates_per_ns": upd_per_step * world * args.steps / (ms_ik * 1e6),
                       "roofline_frac_algorithmic": ach_i / peak,
                       "note": "one gather serves the Metropolis and the over-relaxation update of a site, so the "
                               "north star's per-update byte count (32.375 B) overstates what is moved: frac may exceed 1"}

    # ---- end to end through the C ABI with HOST buffers: every step uploads the step's input state from pinned host
    #      memory (xy_set_theta), runs one PT cycle and reads the step's result -- the accumulated observables
    #      [S][R][8] fp64 and the temperature labels -- back to the host ----
    e2e = None
    if not args.no_e2e:
        nbytes = w.S * w.N * w.R * 4
        host = torch.empty((w.S, w.N, w.R), dtype=torch.float32, pin_memory=True).numpy()
        ens.get_theta(out=host)
        n_e2e = max(2, min(args.steps, 5))
        sink = []

        def e2e_steps(n):
            for _ in range(n):
                ens.set_theta(host)                       # H2D, pinned
                ens.run(1, sps, orps, me)
                sink.append(ens.read_accumulators())      # D2H result (synchronises)
                sink.append(ens.get_labels())
                del sink[:-2]
        e2e_steps(1)
        t0 = time.perf_counter()
        barrier()
        e2e_steps(n_e2e)
        barrier()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": upd_per_step * world * n_e2e / (dt * 1e9), "unit": UNIT, "steps": n_e2e,
               "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": w.S * w.R * 8 * 8 + w.S * w.R * 4,
               "what": "xy_set_theta(pinned host state) + xy_run(1 cycle) + xy_read_accumulators + xy_get_labels (host)"}

    # ---- CPU baseline: the oracle on a bounded sample of the same workload (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_rep = min(w.R, max(1, int(2.4e7 / (w.N * (1 + orps)))))       # ~2.4e7 updates: 10-30 s of one core
        v, dt = oracle_sample_run(w, n_rep, 1, 0xBA5E)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "sample": f"1 of {w.S} samples, first {n_rep} of {w.R} replicas, one Metropolis + {orps} OR sweep(s) + measure"}

    if rank == 0:
        info = B.xy_graph_info(ens.graph)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": w.name, "L": w.L, "N": w.N, "rho": w.rho, "z": w.z, "R": w.R, "S_per_gpu": w.S,
                           "T_min": w.T_min, "T_max": w.T_max, "sweeps_per_step": sps, "or_per_sweep": orps,
                           "measure_every": me, "colours": info["q_max"], "max_degree": info["max_degree"],
                           "step": "one PT cycle: sweeps_per_step x (Metropolis + OR + measure) + one swap round",
                           "l2": "inputs larger than L2 (no flush)" if w.S * w.N * w.R * 4 > 126e6 else
                                 "working set fits the 126 MB L2 (L2-resident by design; no flush)",
                           "parallelism": f"samples x{world}"},
                "roofline": roofline, "interleaved": interleaved, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks}
        print(json.dumps(line), flush=True)

    # ---- auxiliary row: structure factor at k_min, one streaming pass over theta; its own
    #      roofline line goes to stderr so that stdout keeps the single contract line ----
    if rank == 0 and not args.no_aux:
        x = (g.new_to_old % w.L).astype(np.int32)
        y = (g.new_to_old // w.L).astype(np.int32)
        ens.set_coords(w.L, w.L, x, y)
        for _ in range(3):
            ens.measure_fourier()
        n_f = 20
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ens.synchronize()
        ev0.record(ens.stream)
        for _ in range(n_f):
            ens.measure_fourier()
        ev1.record(ens.stream)
        ens.synchronize()
        ms_f = ev0.elapsed_time(ev1) / n_f
        bytes_f = w.S * w.N * (4.0 * w.R + 4.0)                 # theta once + packed coordinates
        peak, peak_src = measured_peak()
        print(json.dumps({"aux": "xy_measure_fourier (k_fourier)", "workload": w.name, "us_per_launch": ms_f * 1e3,
                          "spins_per_ns": w.S * w.N * w.R / (ms_f * 1e6),
                          "roofline": {"bound": "hbm", "achieved": bytes_f / (ms_f * 1e-3) * 1e-9, "peak": peak, "unit": "GB/s",
                                       "frac": bytes_f / (ms_f * 1e-3) * 1e-9 / peak, "bytes_per_spin": 4.0 + 4.0 / w.R}}),
              file=sys.stderr, flush=True)

    # ---- auxiliary row: random-walk self-return histogram, the paper's 4e4 walkers per graph ----
    if rank == 0 and not args.no_aux:
        n_w, n_t = 40_000, 1024
        rng = np.random.default_rng(1)
        st = np.stack([rng.choice(np.where(np.diff(g.row_ptr[s]) > 2)[0], n_w) for s in range(w.S)]).astype(np.int32)
        B.xy_random_walk(ens.graph, st, 16, seed)
        t0 = time.perf_counter()
        hist = B.xy_random_walk(ens.graph, st, n_t, seed)
        dt = time.perf_counter() - t0
        print(json.dumps({"aux": "xy_random_walk (k_random_walk)", "workload": w.name, "walkers_per_graph": n_w, "steps": n_t,
                          "walker_steps_per_ns": w.S * n_w * n_t / (dt * 1e9), "seconds_incl_copies": dt,
                          "bound": "latency (two dependent random 32-byte reads per step)",
                          "returns_at_t2": int(hist[:, 2].sum())}), file=sys.stderr, flush=True)

    if args.lscan and rank == 0 and world == 1:
        ens.close()
        for L in (32, 64, 128, 256):
            wl = workloads.lscan(L)
            gl = levy.build(wl.L, wl.rho, wl.z, wl.seed, S=wl.S)
            el = B.Ensemble(gl.row_ptr, gl.col_idx, gl.colour, wl.temperatures(), seed)
            el.run(5, sps, orps, me); el.synchronize()
            n = max(10, int(2000 * 64 * 64 / (L * L)))
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record(el.stream); el.run(n, sps, orps, me); ev1.record(el.stream); el.synchronize()
            msl = ev0.elapsed_time(ev1)
            print(json.dumps({"lscan": wl.name, "updates_per_ns": sps * (1 + orps) * wl.N * wl.R * wl.S * n / (msl * 1e6),
                              "ms_per_step": msl / n, "steps": n}), file=sys.stderr, flush=True)
            el.close()
    else:
        ens.close()
    if world > 1:
        dist.barrier()          # rank 0 may still be in its auxiliary measurements
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
