"""Equilibrium pins of the oracle's Metropolis + over-relaxation + parallel tempering against exact
results (BASELINE.json north_star): periodic ring closed form, open chain (tree)
closed form, brute-force quadrature on 3- and 4-site graphs, beta = 0 moments.  Seeds are fixed, so
the tests are deterministic; thresholds are 4.5 sigma of the block-jackknife error."""
import numpy as np
import pytest

import closed_forms as CF
import graphs as G
import oracle as O
import stats as S

SEED = 0x5EED1234
NSIG = 4.5


def run_blocks(g, T, n_blocks, cycles_per_block, burn_cycles, seed=SEED, sweeps_per_swap=10, or_per_sweep=1, order=0):
    ch = O.Chain(g["row_ptr"], g["col_idx"], g["class_ptr"], T, seed)
    ch.run(burn_cycles, sweeps_per_swap, or_per_sweep, 1, order)
    blocks = []
    for _ in range(n_blocks):
        ch.reset_acc()
        ch.run(cycles_per_block, sweeps_per_swap, or_per_sweep, 1, order)
        blocks.append(ch.acc.copy())
    return np.array(blocks), ch


def check(blocks, fn, exact, what):
    est, sig = S.jackknife(blocks, fn)
    exact = np.asarray(exact)
    z = np.abs(est - exact) / sig
    assert np.all(z < NSIG), f"{what}: est {est} exact {exact} sigma {sig} z {z}"
    assert np.all(sig < 0.05 * np.maximum(np.abs(exact), 0.02)), f"{what}: error bars too wide {sig}"


@pytest.mark.parametrize("N", [8, 16])
def test_ring_closed_form(N):
    T = np.array([0.5, 1.0, 2.0, 4.0])
    g = G.colour_major(N, G.ring_edges(N))
    blocks, ch = run_blocks(g, T, 40, 60 if N == 8 else 40, 40)
    exact = np.array([CF.ring(N, 1 / t) for t in T])
    check(blocks, S.obs_energy(N), exact[:, 0], f"ring N={N} e")
    check(blocks, S.obs_m2(), exact[:, 1], f"ring N={N} m2")
    assert np.array_equal(ch.slot_of_temp[ch.temp_of_slot], np.arange(4))
    assert ch.swap_attempts.sum() > 0 and 0.05 < ch.swap_accepts.sum() / ch.swap_attempts.sum() < 0.95


def test_ring_golden_table_matches_closed_form():
    """tests/golden/ring_chain.txt restates SURVEY.md Appendix A; check it against the live Bessel sums."""
    import os
    n = 0
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "ring_chain.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kind, N, T, e, m2 = line.split()
        f = CF.ring if kind == "ring" else CF.chain
        ee, mm = f(int(N), 1 / float(T))
        assert abs(ee - float(e)) < 2e-10 and abs(mm - float(m2)) < 2e-10
        n += 1
    assert n == 24


def test_ring_closed_form_vs_quadrature():
    for beta in (0.5, 1.0, 2.0):
        q = CF.quadrature(4, G.ring_edges(4), beta)
        e, m2 = CF.ring(4, beta)
        assert abs(q["E"] / 4 - e) < 1e-10 and abs(q["m2"] - m2) < 1e-10
        q = CF.quadrature(3, G.ring_edges(3), beta)
        e, m2 = CF.ring(3, beta)
        assert abs(q["E"] / 3 - e) < 1e-10 and abs(q["m2"] - m2) < 1e-10
        q = CF.quadrature(4, G.chain_edges(4), beta)
        e, m2 = CF.chain(4, beta)
        assert abs(q["E"] / 4 - e) < 1e-10 and abs(q["m2"] - m2) < 1e-10


def test_open_chain_tree_closed_form():
    N = 16
    T = np.array([0.5, 1.0, 2.0, 4.0])
    g = G.colour_major(N, G.chain_edges(N))
    blocks, _ = run_blocks(g, T, 40, 40, 40)
    exact = np.array([CF.chain(N, 1 / t) for t in T])
    check(blocks, S.obs_energy(N), exact[:, 0], "chain e")
    check(blocks, S.obs_m2(), exact[:, 1], "chain m2")


@pytest.mark.parametrize("name", ["P3", "K3", "star", "paw", "diamond", "K4"])
def test_small_graph_quadrature(name):
    N, edges = CF.SMALL_GRAPHS[name]
    betas = np.array([2.0, 1.0, 0.5])
    T = 1 / betas
    g = G.colour_major(N, edges)
    blocks, _ = run_blocks(g, T, 40, 100, 50)
    q = [CF.quadrature(N, edges, b) for b in betas]
    check(blocks, lambda m: m[..., S.E_], [x["E"] for x in q], f"{name} E")
    check(blocks, S.obs_var_e(), [x["varE"] for x in q], f"{name} varE")
    check(blocks, S.obs_absm(), [x["absm"] for x in q], f"{name} |m|")
    check(blocks, S.obs_m2(), [x["m2"] for x in q], f"{name} m2")
    check(blocks, S.obs_m4(), [x["m4"] for x in q], f"{name} m4")
    check(blocks, S.obs_u4(), [x["m4"] / x["m2"] ** 2 - 1 for x in q], f"{name} U4")


def test_small_graph_golden_table_matches_quadrature():
    import os
    n = 0
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "small_graphs.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, beta, E, varE, absm, m2, m4, u4 = line.split()
        N, edges = CF.SMALL_GRAPHS[name]
        q = CF.quadrature(N, edges, float(beta))
        for got, want in [(q["E"], E), (q["varE"], varE), (q["absm"], absm), (q["m2"], m2), (q["m4"], m4),
                          (q["m4"] / q["m2"] ** 2 - 1, u4)]:
            assert abs(got - float(want)) < 5e-10
        n += 1
    assert n == 24


def test_metropolis_only_and_or_only_pieces():
    """Metropolis alone (or_per_sweep = 0) must already sample the Gibbs measure; adding OR sweeps must
    not change it (OR is microcanonical): K4 at beta = 1."""
    N, edges = CF.SMALL_GRAPHS["K4"]
    g = G.colour_major(N, edges)
    q = CF.quadrature(N, edges, 1.0)
    for orps in (0, 3):
        blocks, _ = run_blocks(g, np.array([1.0]), 40, 100, 50, or_per_sweep=orps)
        check(blocks, lambda m: m[..., S.E_], [q["E"]], f"K4 or={orps} E")
        check(blocks, S.obs_m2(), [q["m2"]], f"K4 or={orps} m2")


def test_beta_zero_moments():
    """T = inf: independent uniform angles: <m^2> = 1/N, <m^4> = (2N-1)/N^3, <E> = 0, Var E = E_b/2, U4 = 1-1/N."""
    edges, _ = O.levy_edges(8, 3.5, 6, 0x12113991, 0)
    N = 64
    g = G.colour_major(N, [tuple(e) for e in edges])
    blocks, _ = run_blocks(g, np.array([np.inf, np.inf]), 40, 20, 5)
    ex = CF.beta0_moments(N, len(edges))
    est, sig = S.jackknife(blocks, S.obs_m2()); assert np.all(np.abs(est - ex["m2"]) < NSIG * sig) and np.all(sig < 0.03 * ex["m2"])
    est, sig = S.jackknife(blocks, S.obs_m4()); assert np.all(np.abs(est - ex["m4"]) < NSIG * sig)
    est, sig = S.jackknife(blocks, lambda m: m[..., S.E_]); assert np.all(np.abs(est) < NSIG * sig)
    est, sig = S.jackknife(blocks, S.obs_var_e()); assert np.all(np.abs(est - ex["varE"]) < NSIG * sig) and np.all(sig < 0.05 * ex["varE"])
    est, sig = S.jackknife(blocks, S.obs_u4()); assert np.all(np.abs(est - (1 - 1 / N)) < NSIG * sig)


def test_levy_graph_low_temperature_harmonic_limit():
    """sanity: E ~ -E_b + (N - #components) T / 2 at low T on a connected Levy sample."""
    edges, _ = O.levy_edges(8, 3.5, 6, 0x12113991, 0)
    N = 64
    g = G.colour_major(N, [tuple(e) for e in edges])
    T = np.array([0.02, 0.04])
    th0 = np.full((N, 2), 1.0, np.float32)
    ch = O.Chain(g["row_ptr"], g["col_idx"], g["class_ptr"], T, SEED, theta=th0)
    ch.run(200, 10, 1, 1); ch.reset_acc(); ch.run(300, 10, 1, 1)
    e = ch.acc[:, S.E_] / ch.acc[:, S.N_]
    # number of connected components
    import scipy.sparse as sp
    from scipy.sparse.csgraph import connected_components
    A = sp.csr_matrix((np.ones(len(g["col_idx"])), g["col_idx"], g["row_ptr"]), shape=(N, N))
    ncomp = connected_components(A)[0]
    assert np.allclose(e, -len(edges) + (N - ncomp) * T / 2, rtol=0, atol=0.06 * (N - ncomp) * T / 2 + 0.02)


def test_specific_heat_two_estimators_agree():
    """the paper's equilibration check (Eq. 13): fluctuation and derivative estimators of c coincide."""
    edges, _ = O.levy_edges(8, 3.5, 6, 0x12113991, 0)
    N = 64
    g = G.colour_major(N, [tuple(e) for e in edges])
    T = O.geometric_temperatures(12, 1.2, 3.6)
    blocks, _ = run_blocks(g, T, 30, 60, 40)
    cf, sf, cd, sd = S.specific_heat_estimators(blocks, T, N)
    z = np.abs(cf - cd) / np.sqrt(sf ** 2 + sd ** 2 + (0.01 * cf) ** 2)     # 1 %: truncation of the 3-point derivative
    assert np.all(z < NSIG), (cf, cd, sf, sd)
    assert np.all(sf < 0.08 * cf) and np.all(cf > 0.05)


@pytest.mark.parametrize("name", ["K3", "paw", "K4"])
def test_interleaved_order_samples_the_same_gibbs_measure(name):
    """per colour class Metropolis then over-relaxation (orc_run_order, order = 1) is a different
    chain with the same stationary distribution: the quadrature pins must hold for it too."""
    N, edges = CF.SMALL_GRAPHS[name]
    betas = np.array([2.0, 1.0, 0.5])
    g = G.colour_major(N, edges)
    blocks, _ = run_blocks(g, 1 / betas, 40, 100, 50, order=1)
    q = [CF.quadrature(N, edges, b) for b in betas]
    check(blocks, lambda m: m[..., S.E_], [x["E"] for x in q], f"{name} E")
    check(blocks, S.obs_var_e(), [x["varE"] for x in q], f"{name} varE")
    check(blocks, S.obs_absm(), [x["absm"] for x in q], f"{name} |m|")
    check(blocks, S.obs_m4(), [x["m4"] for x in q], f"{name} m4")


def test_interleaved_order_ring_closed_form_and_differs_from_default():
    N = 16
    T = np.array([0.5, 1.0, 2.0, 4.0])
    g = G.colour_major(N, G.ring_edges(N))
    blocks, ch = run_blocks(g, T, 40, 40, 40, order=1)
    exact = np.array([CF.ring(N, 1 / t) for t in T])
    check(blocks, S.obs_energy(N), exact[:, 0], "ring interleaved e")
    check(blocks, S.obs_m2(), exact[:, 1], "ring interleaved m2")
    a = O.Chain(g["row_ptr"], g["col_idx"], g["class_ptr"], T, SEED); a.run(1, 2, 1, 1, 0)
    b = O.Chain(g["row_ptr"], g["col_idx"], g["class_ptr"], T, SEED); b.run(1, 2, 1, 1, 1)
    assert not np.array_equal(a.theta, b.theta)                   # genuinely another order


@pytest.mark.parametrize("order", [0, 1])
def test_protocol_replay_is_bit_identical_to_orc_run_and_order_sensitive(order):
    """tests/protocol.py (the PT cycle spelled out with the single-step oracle calls, used by the GPU protocol test to
    watch the decision margins) reproduces orc_run_order bit for bit; and running ONE phase out of order (over-relaxation
    before Metropolis on the last colour) moves angles by O(1) within a cycle -- the GPU test's 1e-3 rad bar notices it."""
    import protocol as P
    from paper_1211_3991_b200 import levy, workloads
    g = levy.build(8, 3.5, 6, workloads.BASE_SEED, S=1)
    T = O.geometric_temperatures(8, 1.0, 4.0)
    rp, ci, cp = g.row_ptr[0], g.col_idx[0], g.class_ptr(0)
    h = P.run_with_margins(rp, ci, cp, T, 7, 3, 10, 1, 1, order=order)
    ch = O.Chain(rp, ci, cp, T, 7)
    ch.run(3, 10, 1, 1, order=order)
    assert np.array_equal(h[-1]["theta"], ch.theta)
    assert np.array_equal(h[-1]["temp_of_slot"], ch.temp_of_slot)
    assert np.array_equal(h[-1]["acc"], ch.acc)
    assert 0 < h[-1]["min_margin"] < 1e-2 and 0 < h[-1]["min_swap_margin"] < 1.0
    if order == 0:
        bad = P.run_with_margins(rp, ci, cp, T, 7, 1, 10, 1, 1, mutate="or_first_last_colour")
        d = np.abs(bad[0]["theta"].astype(np.float64) - h[0]["theta"])
        assert np.minimum(d, 2 * np.pi - d).max() > 1.0
