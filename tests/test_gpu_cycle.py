"""-m gpu: the cluster path (k_cycle: one thread-block cluster per sample runs whole PT cycles in one launch, colour
classes separated by the hardware cluster barrier) must give the
SAME BITS as the per-launch path (k_phase): same Philox keying, same arithmetic, exact integer reductions.  The per-launch
path is the one held against the oracle element by element (tests/test_gpu_parity.py), so bit-identity carries that
parity over; the exact-physics equilibrium tests (ring closed form, quadrature on 3- and 4-site graphs, config 0 vs
oracle) run through the cluster path directly because the automatic choice takes it for tiny samples."""
import numpy as np
import pytest

import graphs as G
import gpu_util as U
import oracle as O
from paper_1211_3991_b200 import binding as B
from paper_1211_3991_b200 import levy, workloads

pytestmark = pytest.mark.gpu
SEED = 0xC1A57E12


def same_state(a, b, what):
    assert np.array_equal(a.get_theta(), b.get_theta()), what
    assert np.array_equal(a.get_labels(), b.get_labels()), what
    assert np.array_equal(a.read_accumulators(), b.read_accumulators()), what
    ca, cb = a.get_counters(), b.get_counters()
    assert ca[:2] == cb[:2] and np.array_equal(ca[2], cb[2]) and np.array_equal(ca[3], cb[3]), what
    assert np.array_equal(a.get_energy(), b.get_energy()), what


@pytest.mark.parametrize("L,rho,R,S", [(16, 3.5, 8, 1), (24, 2.5, 16, 5), (16, 4.5, 32, 3), (12, 3.0, 2, 2), (12, 3.0, 4, 40),
                                        (20, 3.5, 64, 2), (32, 2.5, 16, 32), (8, 3.0, 4, 320)])      # the last one: more samples than
                                        # resident clusters of any size (the clusters run in waves)
@pytest.mark.parametrize("order", [0, 1])
def test_cluster_path_is_bit_identical_to_the_launch_path(L, rho, R, S, order):
    g = levy.build(L, rho, 6, workloads.BASE_SEED, S=S, sample_base=3)
    T = O.geometric_temperatures(R, 1.0, 4.0)
    a = U.ensemble_from_levy(g, T, SEED, sample_base=3); a.set_path(1); a.set_order(order)
    b = U.ensemble_from_levy(g, T, SEED, sample_base=3); b.set_path(2); b.set_order(order)
    assert a.get_path()[0] == 1 and b.get_path()[0] == 2 and 1 <= b.get_path()[1] <= 16
    for (n, sps, orps, me) in [(3, 10, 1, 1), (2, 4, 1 if order else 2, 3), (1, 1, 1, 0), (4, 3, 1, 2)]:
        a.run(n, sps, orps, me); b.run(n, sps, orps, me)
        same_state(a, b, (n, sps, orps, me))
    a.run_sweeps(3, 5, 1); b.run_sweeps(3, 5, 1)
    same_state(a, b, "run_sweeps")
    assert a.read_accumulators()[..., 0].min() > 0 and (R < 8 or a.get_counters()[3].sum() > 0)          # measured, swaps accepted
    # mixing the paths inside one run, and checkpoint/resume across them
    a.run(2, 10, 1, 1)
    b.set_path(1); b.run(1, 10, 1, 1); b.set_path(2); b.run(1, 10, 1, 1)
    same_state(a, b, "mixed")
    a.close(); b.close()


def test_cluster_path_degenerate_graphs_and_unequal_colour_counts():
    """isolated sites, empty colour classes in some samples, a 2-site graph, more CTAs than sites"""
    N = 8
    g0 = G.colour_major(N, [(0, 1), (1, 2), (2, 0), (3, 4)])            # 3 colours, 3 isolated sites
    g1 = G.colour_major(N, [(0, 1), (2, 3), (4, 5)])                    # 2 colours
    rp = np.stack([g0["row_ptr"], g1["row_ptr"]]); col = np.stack([g0["colour"], g1["colour"]])
    ci = np.concatenate([g0["col_idx"], g1["col_idx"]])
    T = np.array([0.5, 1.0, 2.0, 4.0])
    a = B.Ensemble(rp, ci, col, T, SEED); a.set_path(1)
    b = B.Ensemble(rp, ci, col, T, SEED); b.set_path(2)
    a.run(5, 10, 1, 1); b.run(5, 10, 1, 1)
    same_state(a, b, "degenerate")
    a.close(); b.close()
    g2 = G.colour_major(2, [(0, 1)])
    a = U.ensemble_from_graph(g2, T, SEED, S=3); a.set_path(1)
    b = U.ensemble_from_graph(g2, T, SEED, S=3); b.set_path(2)
    a.run(20, 10, 1, 1); b.run(20, 10, 1, 1)
    same_state(a, b, "two sites")
    a.close(); b.close()


def test_cluster_path_selection_and_errors():
    g = levy.build(16, 3.5, 6, workloads.BASE_SEED, S=2)
    small = U.ensemble_from_levy(g, O.geometric_temperatures(16, 1.0, 4.0), SEED)
    assert small.get_path()[0] == 2                          # automatic: tiny samples take the cluster path
    assert small.get_path(or_per_sweep=0)[0] == 1            # no over-relaxation sweep to fuse the measurement into
    small.run(1, 10, 0, 1)                                   # ... and xy_run falls back by itself
    small.set_path(2)
    with pytest.raises(B.XYError):
        small.run(1, 10, 0, 1)
    small.close()
    odd = U.ensemble_from_levy(g, O.geometric_temperatures(6, 1.0, 4.0), SEED)          # any-R path: no cluster flavour
    assert odd.get_path()[0] == 1
    with pytest.raises(B.XYError):
        odd.set_path(2)
    odd.close()
    wide = U.ensemble_from_levy(g, O.geometric_temperatures(128, 1.0, 4.0), SEED)       # two column blocks
    with pytest.raises(B.XYError):
        wide.set_path(2)
    wide.close()


@pytest.mark.parametrize("cfg", [0, 1])
def test_cluster_path_full_size_configs_bit_identical_and_energy_vs_oracle(cfg):
    """BASELINE configs 0 and 1 at full size (the small configs) through the cluster path"""
    w = workloads.CONFIGS[cfg]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=w.S)
    T = w.temperatures()
    a = U.ensemble_from_levy(g, T, SEED); a.set_path(1)
    b = U.ensemble_from_levy(g, T, SEED); b.set_path(2)
    assert b.get_path()[0] == 2
    a.run(3, w.sweeps_per_swap, w.or_per_sweep, 1); b.run(3, w.sweeps_per_swap, w.or_per_sweep, 1)
    same_state(a, b, cfg)
    th, E = b.get_theta(), b.get_energy()
    for s in range(min(w.S, 3)):
        Eo, _, _ = O.measure(g.row_ptr[s], g.col_idx[s], th[s])
        assert np.all(np.abs(E[s] - Eo) <= 4e-7 * 3 * w.N)
    a.close(); b.close()
