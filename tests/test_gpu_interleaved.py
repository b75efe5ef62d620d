"""-m gpu tests of the interleaved sweep order (xy_set_order(1)): per colour class,
Metropolis and then over-relaxation of each site from ONE gather (k_phase MODE 4 / 5).  Same bars as the default
order: lockstep per colour class against the oracle (1e-5 rad, near-threshold / ill-conditioned sites counted),
protocol and bookkeeping against orc_run_order, bit-identity across tuning switches, equilibrium against exact
physics and against the oracle."""
import numpy as np
import pytest

import closed_forms as CF
import graphs as G
import gpu_util as U
import oracle as O
import stats as S
from paper_1211_3991_b200 import binding as B
from paper_1211_3991_b200 import levy, workloads

pytestmark = pytest.mark.gpu
SEED = 0x1E7E41EA


@pytest.mark.parametrize("L,rho,R,S", [(16, 3.5, 8, 1), (16, 3.5, 64, 2), (24, 2.5, 16, 3), (16, 4.5, 32, 2), (12, 3.0, 2, 2),
                                        (12, 3.0, 4, 2), (8, 3.5, 128, 1)])
def test_lockstep_interleaved(L, rho, R, S):
    g = levy.build(L, rho, 6, workloads.BASE_SEED, S=S, sample_base=2)
    T = O.geometric_temperatures(R, 1.0, 4.0)
    ens = U.ensemble_from_levy(g, T, SEED, sample_base=2)
    graphs = U.graphs_of_levy(g)
    rng = np.random.default_rng(7)
    ens.set_labels(np.stack([rng.permutation(R).astype(np.int32) for _ in range(S)]))
    tot = dict(updates=0, near=0, bad=0, illcond=0, accepted=0)
    for sweep in (1, 2, 3):
        for c in range(int(g.n_colours.max())):
            st = U.lockstep_metor(ens, graphs, T, SEED, c, sweep, sample_base=2)
            assert st["bad"] == 0, st
            for k in tot: tot[k] += st[k]
    assert tot["updates"] == 3 * L * L * R * S
    assert 0.2 < tot["accepted"] / tot["updates"] < 0.95
    assert tot["near"] <= 5 + 2e-4 * tot["updates"] and tot["illcond"] <= 5 + 5e-3 * tot["updates"]
    print(f"\n[interleaved lockstep L={L} R={R} S={S}] {tot}")
    ens.close()


def test_interleaved_needs_float2_flavour_and_one_or_sweep():
    g = levy.build(8, 3.5, 6, workloads.BASE_SEED, S=1)
    ens = U.ensemble_from_levy(g, O.geometric_temperatures(3, 1.0, 2.0), SEED)
    with pytest.raises(B.XYError) as e:
        ens.set_order(1)
    assert e.value.code == B.XY_ESTATE
    ens.close()
    ens = U.ensemble_from_levy(g, O.geometric_temperatures(4, 1.0, 2.0), SEED)
    ens.set_order(1)
    with pytest.raises(B.XYError):
        ens.run(1, 2, 2, 1)
    ens.close()


def test_interleaved_run_protocol_vs_oracle_and_tuning_invariance():
    """xy_run in interleaved order against orc_run_order(order = 1) on config 0 (counts, labels, observables), and the
    same bits for every tuning switch / schedule; differs from the default order."""
    w = workloads.CONFIGS[0]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=1)
    T = w.temperatures()
    ens = U.ensemble_from_levy(g, T, SEED); ens.set_order(1)
    ch = O.Chain(g.row_ptr[0], g.col_idx[0], g.class_ptr(0), T, SEED)
    ens.run(1, 2, 1, 1); ch.run(1, 2, 1, 1, 1)
    acc = ens.read_accumulators()[0]
    assert np.array_equal(acc[:, 0], ch.acc[:, 0])
    assert np.allclose(acc[:, 1], ch.acc[:, 1], rtol=0, atol=2e-3) and np.allclose(acc[:, 4], ch.acc[:, 4], rtol=0, atol=1e-4)
    assert np.array_equal(ens.get_labels()[0], ch.temp_of_slot)
    assert U.circ(ens.get_theta()[0], ch.theta).mean() < 1e-3
    ens.close()
    g = levy.build(16, 3.5, 6, workloads.BASE_SEED, S=4)
    T = O.geometric_temperatures(16, 1.0, 4.0)
    ref = None
    for kw, sched in ((dict(), 0), (dict(balance=0, pdl=0, l2_persist=0, fuse_measure=0, cta_shape=1), 1), (dict(cta_shape=2), 4)):
        e = U.ensemble_from_levy(g, T, SEED); e.set_order(1); e.set_tuning(**kw); e.set_schedule(sched)
        e.run(3, 4, 1, 2); e.run(2, 3, 1, 2)
        cur = (e.get_theta(), e.get_labels(), e.read_accumulators())
        if ref is None: ref = cur
        else: assert all(np.array_equal(a, b) for a, b in zip(ref, cur)), kw
        e.close()
    d = U.ensemble_from_levy(g, T, SEED); d.run(3, 4, 1, 2); d.run(2, 3, 1, 2)
    assert not np.array_equal(d.get_theta(), ref[0])
    d.close()


@pytest.mark.parametrize("name", ["K3", "paw", "K4"])
def test_interleaved_small_graph_quadrature_on_gpu(name):
    N, edges = CF.SMALL_GRAPHS[name]
    betas = np.array([2.0, 1.0, 0.5, 0.25])                       # four temperatures: a float2 flavour (R = 4)
    ens = U.ensemble_from_graph(G.colour_major(N, edges), 1 / betas, SEED, S=16)
    ens.set_order(1)
    ens.run(50, 10, 1, 1)
    prev = ens.read_accumulators(); blocks = []
    for _ in range(40):
        ens.run(50, 10, 1, 1)
        cur = ens.read_accumulators(); blocks.append((cur - prev).sum(0)); prev = cur
    blocks = np.array(blocks)
    q = [CF.quadrature(N, edges, b) for b in betas]
    for fn, key in ((lambda m: m[..., S.E_], "E"), (S.obs_var_e(), "varE"), (S.obs_absm(), "absm"), (S.obs_m4(), "m4")):
        est, sig = S.jackknife(blocks, fn)
        exact = np.array([x[key] for x in q])
        assert np.all(np.abs(est - exact) < 4.5 * sig), (name, key, est, exact, sig)
    ens.close()


def test_interleaved_equilibrium_config1_vs_oracle():
    """config 1 (all 16 temperatures, sample 0): E/N, <|m|>, U4 of the interleaved GPU run against the oracle's
    interleaved run within 3 combined jackknife sigma (R13)."""
    w = workloads.CONFIGS[1]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=w.S)
    import concurrent.futures as cf
    def oracle():
        ch = O.Chain(g.row_ptr[0], g.col_idx[0], g.class_ptr(0), w.temperatures(), SEED + 1)
        ch.run(60, 10, 1, 1, 1)
        out = []
        for _ in range(10):
            ch.reset_acc(); ch.run(8, 10, 1, 1, 1); out.append(ch.acc.copy())
        return np.array(out)
    with cf.ThreadPoolExecutor(1) as pool:
        fut = pool.submit(oracle)
        ens = U.ensemble_from_levy(g, w.temperatures(), SEED); ens.set_order(1)
        ens.run(1000, 10, 1, 1)
        prev = ens.read_accumulators(); gb = []
        for _ in range(20):
            ens.run(50, 10, 1, 1)
            cur = ens.read_accumulators(); gb.append((cur - prev)[0]); prev = cur
        ens.close()
        ob = fut.result()
    gb = np.array(gb)
    zs = []
    for fn in (S.obs_energy(w.N), S.obs_absm(), S.obs_u4()):
        eg, sg = S.jackknife(gb, fn); eo, so = S.jackknife(ob, fn)
        zs.append((eg - eo) / np.sqrt(sg ** 2 + so ** 2))
    z = np.abs(np.concatenate(zs))
    print(f"\ninterleaved config 1 vs oracle: {z.size} comparisons, max |z| {z.max():.2f}, > 3 sigma {int((z > 3).sum())}")
    assert z.max() < 4.5 and (z > 3).sum() <= 2


def test_interleaved_full_size_config4_sampled_lockstep():
    """BASELINE config 4 at full size in the launch configuration bench.py times: sampled sites of every colour class."""
    w = workloads.CONFIGS[4]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=w.S)
    T = w.temperatures()
    ens = U.ensemble_from_levy(g, T, SEED); ens.set_order(1)
    graphs = U.graphs_of_levy(g)
    rng = np.random.default_rng(4)
    ens.run(2, w.sweeps_per_swap, 1, 1)
    tot = dict(updates=0, near=0, bad=0, illcond=0, accepted=0)
    for c in range(int(g.n_colours.max())):
        st = U.lockstep_metor(ens, graphs, T, SEED, c, 21, samples=[1, 6], site_subset=96, rng=rng)
        assert st["bad"] == 0, st
        for k in tot: tot[k] += st[k]
    print(f"\n[interleaved full size cfg 4] {tot}")
    assert tot["updates"] > 40000 and tot["near"] <= 5 + 2e-4 * tot["updates"]
    E = ens.get_energy()
    th = ens.get_theta()
    Eo, _, _ = O.measure(g.row_ptr[1], g.col_idx[1], th[1])
    assert np.all(np.abs(E[1] - Eo) <= 4e-7 * 3 * w.N)
    ens.close()
