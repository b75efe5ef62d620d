#!/usr/bin/env python
"""Writes tests/golden/oracle_equilibrium_cfg{2,3,4}.npz: the ORACLE's observables on the FULL temperature ladder of
BASELINE.json configs 2, 3 and 4, for tests/test_gpu_equilibrium.py (north_star: "equilibrium E, <|m|> and the
Binder cumulant must agree within 3 combined jackknife sigma"; Eq. 13-16).

Calls ONLY oracle/ (orc_run_order through oracle.Chain, as it stands) and the shared seeded input generators
(paper_1211_3991_b200.levy / workloads: graph sample 0 of the config, the temperature ladder); never the CUDA path.

The oracle makes 2.4e6 updates/s on one core, so the configs' full sweep counts (1e4 / 5e3 / 2e3 sweeps of up to
3.4e7 updates) are out of reach; reading R13b: both sides run the SAME shortened protocol -- uniform
random initial angles (Philox domain 0), the bench protocol (10 sweeps + one swap round per cycle, one OR sweep per
Metropolis sweep, measurement every sweep), the same number of sweeps -- as several INDEPENDENT chains (seeds), and
the test compares the seed-averaged observables of the same time window.  That comparison is exact for two
implementations of one Markov chain whether or not the window is equilibrated at the coldest temperatures.

Stored per config: acc[seed][block][temperature][8] = the accumulator increments (n, E, E^2, |m|, m^2, m^4, Mx/N, My/N)
of consecutive blocks of `cycles_per_block` PT cycles, plus the swap counters and the run parameters.

  python tests/golden/make_oracle_equilibrium.py --configs 2 4 3 --workers 6        (hours; resumable)
"""
import argparse
import concurrent.futures as cf
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for p in (ROOT, os.path.join(ROOT, "oracle")):
    if p not in sys.path:
        sys.path.insert(0, p)

SEED0 = 0x0CAC1E00
# cfg -> (independent chains, PT cycles per chain, cycles per stored block); a cycle = 10 sweeps + 1 swap round
PLAN = {
    2: (12, 300, 30),
    3: (12, 150, 15),
    4: (6, 60, 6),
}


def chain_seed(cfg, k):
    return SEED0 + 0x100 * cfg + k


def run_chain(cfg, k, n_cycles, per_block, partial_dir):
    import oracle as O
    from paper_1211_3991_b200 import levy, workloads
    out = os.path.join(partial_dir, f"cfg{cfg}_seed{k}_c{n_cycles}_b{per_block}.npz")
    if os.path.exists(out):
        return out
    w = workloads.CONFIGS[cfg]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=1)                    # graph sample 0 of the config
    ch = O.Chain(g.row_ptr[0], g.col_idx[0], g.class_ptr(0), w.temperatures(), chain_seed(cfg, k))
    blocks = []
    t0 = time.time()
    for _ in range(n_cycles // per_block):
        ch.reset_acc()
        ch.run(per_block, w.sweeps_per_swap, w.or_per_sweep, 1)
        blocks.append(ch.acc.copy())
    np.savez(out + ".tmp.npz", acc=np.array(blocks), att=ch.swap_attempts, accepts=ch.swap_accepts, seconds=time.time() - t0)
    os.replace(out + ".tmp.npz", out)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="+", default=[2, 4, 3])
    ap.add_argument("--workers", type=int, default=max(1, (os.cpu_count() or 2) - 2))
    ap.add_argument("--partial-dir", default="/tmp/xy_oracle_equilibrium")
    ap.add_argument("--seeds", type=int, default=0, help="use only the first N chains of the plan (0 = all)")
    args = ap.parse_args()
    os.makedirs(args.partial_dir, exist_ok=True)
    import oracle as O
    from paper_1211_3991_b200 import workloads
    O.lib()                                                          # build once, before the workers start
    with cf.ProcessPoolExecutor(max_workers=args.workers) as pool:
        futs = {}
        for cfg in args.configs:
            n_seeds, n_cycles, per_block = PLAN[cfg]
            n_seeds = min(n_seeds, args.seeds) if args.seeds > 0 else n_seeds
            for k in range(n_seeds):
                futs[(cfg, k)] = pool.submit(run_chain, cfg, k, n_cycles, per_block, args.partial_dir)
        for cfg in args.configs:
            n_seeds, n_cycles, per_block = PLAN[cfg]
            n_seeds = min(n_seeds, args.seeds) if args.seeds > 0 else n_seeds
            w = workloads.CONFIGS[cfg]
            parts = [np.load(futs[(cfg, k)].result()) for k in range(n_seeds)]
            dst = os.path.join(HERE, f"oracle_equilibrium_cfg{cfg}.npz")
            np.savez_compressed(
                dst, acc=np.array([p["acc"] for p in parts]), swap_attempts=np.array([p["att"] for p in parts]),
                swap_accepts=np.array([p["accepts"] for p in parts]), seconds=np.array([float(p["seconds"]) for p in parts]),
                seeds=np.array([chain_seed(cfg, k) for k in range(n_seeds)], np.uint64), T=w.temperatures(),
                cycles_per_block=per_block, n_cycles=n_cycles, sweeps_per_swap=w.sweeps_per_swap, or_per_sweep=w.or_per_sweep,
                measure_every=1, order=0, workload=w.name, graph_sample=0)
            print(f"wrote {dst}: {n_seeds} chains x {n_cycles} cycles, {sum(float(p['seconds']) for p in parts):.0f} core-seconds",
                  flush=True)


if __name__ == "__main__":
    main()
