"""-m gpu parity at BASELINE.json's FULL sizes (configs 1-4), in the launch configuration bench.py times
(same sample groups / grids as the captured xy_run graph): after a few captured PT cycles, every colour
class is stepped in lockstep and SAMPLED sites are compared with the oracle one by one (all replicas of
the site); energies of sampled samples are compared with the oracle's fp64 sum; and properties that hold
at any size are checked on the whole state (range, untouched classes, OR energy conservation, labels)."""
import numpy as np
import pytest

import gpu_util as U
import oracle as O
from paper_1211_3991_b200 import levy, workloads

pytestmark = pytest.mark.gpu
SEED = 0xF0115123
SITES_PER_CLASS = 96          # sampled sites per (sample, colour class): x R replicas each


def near_bound(n):
    """near-threshold decisions (R6): P(|u2 - min(1, p)| < 1e-5) is 2e-5 for p < 1 and 1e-5 for p >= 1 per update;
    allow 3 x 2e-5 plus small-number slack (a kernel that mis-decides ten times more often must fail)."""
    return 6e-5 * n + 10


def illcond_bound(n):
    """ill-conditioned over-relaxation updates (R7): SURVEY C7 measured 0.17 % at T = infinity (the worst case) + 5 sigma"""
    return 1.7e-3 * n + 5 * np.sqrt(1.7e-3 * n) + 3


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_full_size_lockstep_sampled_sites_and_invariants(cfg):
    w = workloads.CONFIGS[cfg]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=w.S)
    T = w.temperatures()
    ens = U.ensemble_from_levy(g, T, SEED)
    graphs = U.graphs_of_levy(g)
    rng = np.random.default_rng(cfg)
    # the timed path first: two captured PT cycles (labels get permuted, angles decorrelate from the init)
    ens.run(2, w.sweeps_per_swap, w.or_per_sweep, 1)
    sw, rd, att, acc = ens.get_counters()
    assert (sw, rd) == (2 * w.sweeps_per_swap, 2)
    labels = ens.get_labels()
    assert np.array_equal(np.sort(labels, axis=1), np.tile(np.arange(w.R, dtype=np.int32), (w.S, 1)))
    assert acc.sum() > 0 and np.all(acc <= att)                       # some swaps were accepted
    n_acc = ens.read_accumulators()[..., 0]
    assert np.all(n_acc == 2 * w.sweeps_per_swap)

    samples = sorted(rng.choice(w.S, size=min(2, w.S), replace=False).tolist())
    Q = int(g.n_colours.max())
    tm = dict(updates=0, near=0, bad=0, accepted=0, disagree_near=0)
    to = dict(updates=0, illcond=0, bad=0)
    sweep = sw + 1
    for c in range(Q):
        st = U.lockstep_metropolis(ens, graphs, T, SEED, c, sweep, samples=samples, site_subset=SITES_PER_CLASS, rng=rng)
        assert st["bad"] == 0, (cfg, c, st)
        for k in tm: tm[k] += st[k]
    E_before = ens.get_energy()
    for c in range(Q):
        st = U.lockstep_overrelax(ens, graphs, c, samples=samples, site_subset=SITES_PER_CLASS, rng=rng)
        assert st["bad"] == 0, (cfg, c, st)
        for k in to: to[k] += st[k]
    E_after = ens.get_energy()
    print(f"\n[full size cfg {cfg}] metropolis {tm}  overrelax {to}")
    assert tm["updates"] >= 0.9 * len(samples) * (Q - 1) * SITES_PER_CLASS * w.R
    assert 0.2 < tm["accepted"] / tm["updates"] < 0.95
    assert tm["near"] <= near_bound(tm["updates"])
    assert to["illcond"] <= illcond_bound(to["updates"])

    # OR sweep conserves the energy of every replica (ref 66 via PAPER.md:460): fp32 round-off only
    assert np.all(np.abs(E_after - E_before) <= 1e-6 * w.N * 3), np.abs(E_after - E_before).max()

    # energies / magnetisation of one whole sample against the oracle's fp64 sums (all R slots)
    th = ens.get_theta()
    assert th.min() >= 0.0 and th.max() <= np.float32(6.2831855)
    s = samples[0]
    Eo, Mxo, Myo = O.measure(g.row_ptr[s], g.col_idx[s], th[s])
    assert np.all(np.abs(E_after[s] - Eo) <= 4e-7 * 3 * w.N), np.abs(E_after[s] - Eo).max()
    out = ens.measure(want=True)
    lab = ens.get_labels()
    assert np.all(np.abs(out[s, lab[s], 0] - Eo) <= 4e-7 * 3 * w.N)
    assert np.all(np.abs(out[s, lab[s], 1] - Mxo) <= 2e-7 * w.N) and np.all(np.abs(out[s, lab[s], 2] - Myo) <= 2e-7 * w.N)
    ens.close()


@pytest.mark.parametrize("cfg,reduce_colours", [(1, 0), (2, 0), (3, 0), (4, 0), (4, workloads.REDUCE_COLOURS), (3, workloads.REDUCE_COLOURS)])
def test_full_size_lockstep_every_site_of_one_sample_both_orders(cfg, reduce_colours):
    """EVERY site (all R replicas) of one whole sample of the full-size ensemble, in the bench's launch configuration:
    a Metropolis sweep and an over-relaxation sweep colour by colour (default order), then an interleaved sweep
    (Metropolis + over-relaxation of a class in one launch), each class compared with the oracle from the same
    pre-state.  Share, chunk and column-block boundaries, the degree > 8 tail and isolated sites are all covered.
    reduce_colours > 0: the graphs as bench.py builds them (colour-reducing local search after smallest-last: a fifth
    class of a few dozen sites)."""
    w = workloads.CONFIGS[cfg]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=w.S, reduce_colours=reduce_colours)
    assert all(O.colouring_is_proper(g.row_ptr[k], g.col_idx[k], g.colour[k]) for k in range(min(w.S, 2)))
    T = w.temperatures()
    ens = U.ensemble_from_levy(g, T, SEED + 1)
    graphs = U.graphs_of_levy(g)
    ens.run(1, w.sweeps_per_swap, w.or_per_sweep, 1)                   # decorrelate from the init, permute labels
    s = w.S - 1 if cfg != 3 else 10                                    # not the first sample of a launch group
    Q = int(g.n_colours[s])
    sweep = ens.get_counters()[0] + 1
    tm = dict(updates=0, near=0, bad=0, accepted=0)
    to = dict(updates=0, illcond=0, bad=0)
    ti = dict(updates=0, near=0, bad=0, illcond=0, accepted=0)
    for c in range(Q):
        st = U.lockstep_metropolis(ens, graphs, T, SEED + 1, c, sweep, samples=[s], sparse=True)
        assert st["bad"] == 0, (cfg, c, st)
        for k in tm: tm[k] += st[k]
    for c in range(Q):
        st = U.lockstep_overrelax(ens, graphs, c, samples=[s], sparse=True)
        assert st["bad"] == 0, (cfg, c, st)
        for k in to: to[k] += st[k]
    for c in range(Q):
        st = U.lockstep_metor(ens, graphs, T, SEED + 1, c, sweep + 1, samples=[s], sparse=True)
        assert st["bad"] == 0, (cfg, c, st)
        for k in ti: ti[k] += st[k]
    print(f"\n[every site, cfg {cfg}, sample {s}] metropolis {tm}  overrelax {to}  interleaved {ti}")
    n = w.N * w.R
    assert tm["updates"] == n and to["updates"] == n and ti["updates"] == n
    assert tm["near"] <= near_bound(n) and ti["near"] <= near_bound(n)
    assert to["illcond"] <= illcond_bound(n) and ti["illcond"] <= illcond_bound(n)
    if n > 2e6:          # the band accounting is not vacuous: the expected 1e-5 .. 2e-5 per update are seen
        assert tm["near"] >= 0.5e-5 * n - 10, tm
    assert 0.2 < tm["accepted"] / n < 0.95
    ens.close()


def test_full_size_graph_structure_of_all_configs():
    """integer work at full size: the builder's graphs that the bench loads are proper, symmetric, E_b = N z / 2."""
    for cfg in (1, 2, 3, 4):
        w = workloads.CONFIGS[cfg]
        g = levy.build(w.L, w.rho, w.z, w.seed, S=min(w.S, 4))
        for s in range(g.S):
            rp, ci, col = g.row_ptr[s], g.col_idx[s], g.colour[s]
            assert rp[-1] == w.N * w.z
            assert O.colouring_is_proper(rp, ci, col)
            assert np.all(np.diff(col) >= 0)
