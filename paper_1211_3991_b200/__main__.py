"""python -m paper_1211_3991_b200 <workload> [options] -- run PT cycles of one synthetic workload on cuda:0 and print the
throughput as one JSON line.  A small front end to the C ABI for users and for profiling commands (ncu wraps it).

  workload:  config0 .. config4        the BASELINE.json configs
             lscan32 | lscan64 | lscan128 | lscan256   config 3's L scan (R = 32, S = 16)
             square<L>                 periodic square lattice, z = 4 (R, S from --replicas / --samples)
"""
import argparse
import json
import re
import sys

import numpy as np


def main(argv=None):
    ap = argparse.ArgumentParser(prog="python -m paper_1211_3991_b200")
    ap.add_argument("workload")
    ap.add_argument("--cycles", type=int, default=20, help="timed PT cycles (10 sweeps + swap round each)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--order", type=int, default=0, choices=[0, 1], help="1 = interleaved (xy_set_order)")
    ap.add_argument("--path", type=int, default=0, choices=[0, 1, 2], help="xy_set_path: 1 launch per class, 2 cluster per sample")
    ap.add_argument("--samples-per-group", type=int, default=0, help="xy_set_schedule")
    ap.add_argument("--sweeps-only", action="store_true", help="xy_run_sweeps instead of xy_run (no measurement, no swap)")
    ap.add_argument("--replicas", type=int, default=64)
    ap.add_argument("--samples", type=int, default=8)
    ap.add_argument("--seed", type=lambda v: int(v, 0), default=0xB200_1211_3991)
    ap.add_argument("--colouring", default="reduced", choices=["reduced", "smallest-last"],
                    help="reduced = smallest-last followed by the builder's colour-reducing local search (bench.py's default)")
    ap.add_argument("--no-pdl", action="store_true", help="xy_set_tuning: no programmatic-dependent-launch edges")
    ap.add_argument("--no-l2-window", action="store_true", help="xy_set_tuning: no persisting-L2 access window")
    ap.add_argument("--no-balance", action="store_true", help="xy_set_tuning: equal shares instead of cost-balanced ones")
    a = ap.parse_args(argv)

    import torch
    from . import binding as B
    from . import levy, workloads

    m = re.fullmatch(r"(config|lscan|square)(\d+)", a.workload)
    if not m:
        ap.error("unknown workload")
    kind, k = m.group(1), int(m.group(2))
    tile = 1
    if kind == "config":
        w = workloads.CONFIGS[k]
    elif kind == "lscan":
        w = workloads.lscan(k)
    else:
        w = workloads.square_lattice(k, a.replicas, 0.7, 1.3, a.samples)
        tile = w.S
    g = levy.build(w.L, w.rho, w.z, w.seed, S=1 if tile > 1 else w.S,
                   reduce_colours=workloads.REDUCE_COLOURS if a.colouring == "reduced" else 0)
    rp, ci, col = (np.tile(x, (tile, 1)) for x in (g.row_ptr, g.col_idx, g.colour))
    ens = B.Ensemble(rp, ci, col, w.temperatures(), a.seed)
    ens.set_order(a.order)
    ens.set_path(a.path)
    if a.samples_per_group:
        ens.set_schedule(a.samples_per_group)
    if a.no_pdl or a.no_l2_window or a.no_balance:
        ens.set_tuning(balance=0 if a.no_balance else 1, pdl=0 if a.no_pdl else 1, l2_persist=0 if a.no_l2_window else 1)
    sps, orps = w.sweeps_per_swap, w.or_per_sweep

    def run(n):
        ens.run_sweeps(n, sps, orps) if a.sweeps_only else ens.run(n, sps, orps, 1)

    run(a.warmup)
    ens.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(ens.stream)
    run(a.cycles)
    ev1.record(ens.stream)
    ens.synchronize()
    ms = ev0.elapsed_time(ev1)
    upd = sps * (1 + orps) * w.N * w.R * w.S * a.cycles
    print(json.dumps({"workload": w.name, "path": ens.path_name(orps), "order": a.order, "cycles": a.cycles,
                      "what": "xy_run_sweeps" if a.sweeps_only else "xy_run", "ms_per_cycle": ms / max(a.cycles, 1),
                      "updates_per_ns": upd / (ms * 1e6) if ms > 0 else None, "launches": ens.launch_count()}))
    ens.close()


if __name__ == "__main__":
    sys.exit(main())
