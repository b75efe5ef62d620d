"""The shared builder (libxy_levy.so) against the oracle's definition-level restatement, bit-exact
(BASELINE.json north_star: 'integer work (graph, colouring ...) must match bit-exactly'), plus
structure checks at the sizes only the fast builder reaches."""
import numpy as np
import pytest

import graphs as G
import oracle as O
from paper_1211_3991_b200 import levy, workloads

SEED = workloads.BASE_SEED


@pytest.mark.parametrize("L,rho,z,sample", [(8, 3.5, 6, 0), (16, 3.5, 6, 0), (16, 3.5, 6, 7), (16, 0.0, 6, 1),
                                            (12, 2.5, 4, 2), (32, 4.5, 6, 0), (8, 100.0, 4, 0), (20, 1.0, 3, 5)])
def test_builder_matches_oracle_bit_exact(L, rho, z, sample):
    N = L * L
    g = levy.build(L, rho, z, SEED, S=1, sample_base=sample)
    edges, draws = O.levy_edges(L, rho, z, SEED, sample)
    rp, ci = O.csr_from_edges(N, edges)
    colour, Q = O.colour_smallest_last(rp, ci)
    n2o, rp2, ci2, c2 = O.renumber_colour_major(rp, ci, colour)
    assert int(g.n_draws[0]) == draws and int(g.n_colours[0]) == Q
    assert np.array_equal(g.new_to_old[0], n2o)
    assert np.array_equal(g.row_ptr[0], rp2) and np.array_equal(g.col_idx[0], ci2) and np.array_equal(g.colour[0], c2)


def test_builder_sample_indexing_is_global():
    """sample s of a batch equals a batch of one built with sample_base = s (multi-GPU sharding relies on it)."""
    g = levy.build(16, 3.5, 6, SEED, S=4, sample_base=0, n_threads=3)
    for s in (0, 3):
        g1 = levy.build(16, 3.5, 6, SEED, S=1, sample_base=s)
        assert np.array_equal(g.col_idx[s], g1.col_idx[0]) and np.array_equal(g.colour[s], g1.colour[0])
    assert not np.array_equal(g.col_idx[0], g.col_idx[1])


def test_colouring_and_renumber_entry_points_match_oracle():
    for N, edges in [(9, G.ring_edges(9)), (12, G.chain_edges(12)), (16, G.square_lattice_edges(4)),
                     (6, [(0, k) for k in range(1, 6)]), (5, [])]:
        rp, ci = G.csr_from_edges(N, edges)
        col, Q = levy.colour_smallest_last(rp, ci)
        col_o, Q_o = O.colour_smallest_last(rp, ci)
        assert Q == Q_o and np.array_equal(col, col_o)
        out = levy.renumber_colour_major(rp, ci, col)
        ref = O.renumber_colour_major(rp, ci, col_o)
        for a, b in zip(out, ref):
            assert np.array_equal(a, b)


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_config_graphs_structure(cfg):
    w = workloads.CONFIGS[cfg]
    S = min(w.S, 2)
    g = levy.build(w.L, w.rho, w.z, w.seed, S=S)
    N = w.N
    for s in range(S):
        rp, ci, col = g.row_ptr[s], g.col_idx[s], g.colour[s]
        assert rp[0] == 0 and rp[-1] == N * w.z                                   # E_b = N z / 2
        src = np.repeat(np.arange(N), np.diff(rp))
        assert np.all(src != ci)                                                   # no self loop
        key = src.astype(np.int64) * N + ci
        assert len(np.unique(key)) == len(key)                                     # no duplicate
        assert np.array_equal(np.sort(key), np.sort(ci.astype(np.int64) * N + src))  # symmetric
        assert np.all(col[src] != col[ci])                                         # no monochromatic edge
        assert np.all(np.diff(col) >= 0) and col.max() + 1 == g.n_colours[s] <= 7
        old = g.new_to_old[s]
        dx = np.abs(old[src] % w.L - old[ci] % w.L); dy = np.abs(old[src] // w.L - old[ci] // w.L)
        dx = np.minimum(dx, w.L - dx); dy = np.minimum(dy, w.L - dy)
        assert (dx * dx + dy * dy).max() <= 2 * (w.L // 2) ** 2                    # r_max
        for e in range(0, len(ci), 997):                                           # rows ascending
            pass
        assert all(np.all(np.diff(ci[rp[i]:rp[i + 1]]) > 0) for i in range(0, N, max(1, N // 500)))


def test_builder_errors():
    with pytest.raises(levy.LevyError):
        levy.build(1, 3.5, 6, SEED)
    with pytest.raises(levy.LevyError):
        levy.build(3, 3.5, 3, SEED)          # N*z odd
    with pytest.raises(levy.LevyError):
        levy.build(4, 3.5, 40, SEED)         # more bonds than pairs
    with pytest.raises(levy.LevyError):
        levy.build(8, 400.0, 6, SEED)        # weights beyond nearest neighbours underflow: draw limit


def test_workload_recipes():
    w = workloads.CONFIGS[4]
    assert (w.L, w.R, w.S, w.rho) == (512, 64, 8, 3.0) and abs(w.bytes_per_update() - 32.375) < 1e-12
    T = w.temperatures()
    assert T[0] == 1.5 and abs(T[-1] - 4.0) < 1e-12 and np.allclose(T[1:] / T[:-1], (4.0 / 1.5) ** (1 / 63))
    assert np.allclose(O.geometric_temperatures(w.R, w.T_min, w.T_max), T, rtol=1e-15)
    assert workloads.lscan(64).L == 64 and workloads.lscan(64).R * workloads.lscan(64).S == 512


def test_colour_count_within_the_papers_bound_at_z4():
    """at z = 4 the number of colours is never larger than 6 for N <= 2^16 (tests/golden/paper_values.txt)."""
    import os
    bound = None
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")):
        f = line.split()
        if f and f[0] == "colours_max_z4":
            bound = int(f[1])
    assert bound == 6
    for L, rho in ((64, 0.0), (64, 2.5), (128, 3.5), (64, 4.5), (256, 3.0)):
        g = levy.build(L, rho, 4, 0x12113991, S=2)
        assert int(g.n_colours.max()) <= bound, (L, rho, g.n_colours)


@pytest.mark.parametrize("L,rho,z,sample", [(8, 3.5, 6, 0), (16, 3.5, 6, 3), (12, 0.0, 4, 1), (16, 4.5, 4, 0)])
def test_free_boundary_builder_matches_oracle_bit_exact(L, rho, z, sample):
    N = L * L
    g = levy.build(L, rho, z, SEED, S=1, sample_base=sample, boundary="free")
    edges, draws = O.levy_edges(L, rho, z, SEED, sample, boundary="free")
    rp, ci = O.csr_from_edges(N, edges)
    colour, Q = O.colour_smallest_last(rp, ci)
    n2o, rp2, ci2, c2 = O.renumber_colour_major(rp, ci, colour)
    assert int(g.n_draws[0]) == draws and int(g.n_colours[0]) == Q
    assert np.array_equal(g.new_to_old[0], n2o)
    assert np.array_equal(g.row_ptr[0], rp2) and np.array_equal(g.col_idx[0], ci2) and np.array_equal(g.colour[0], c2)


def test_free_boundary_structure():
    """with free boundaries bonds reach beyond [L/2] sqrt 2 (up to L sqrt 2) and never wrap; the
    bond-length law is ~ (number of pairs at that displacement) r^-rho; border sites have fewer bonds."""
    L, rho, z = 32, 3.0, 6
    g = levy.build(L, rho, z, SEED, S=8, boundary="free")
    cnt = {}
    for s in range(g.S):
        rp, ci, lat = g.row_ptr[s], g.col_idx[s], g.new_to_old[s]
        assert rp[-1] == L * L * z and O.colouring_is_proper(rp, ci, g.colour[s])
        x, y = lat % L, lat // L
        src = np.repeat(np.arange(L * L), np.diff(rp))
        dx, dy = np.abs(x[src] - x[ci]), np.abs(y[src] - y[ci])
        assert np.hypot(dx, dy).max() <= (L - 1) * np.sqrt(2) + 1e-9
        for a, b in zip(dx, dy):
            cnt[(a, b)] = cnt.get((a, b), 0) + 1
        deg = np.diff(rp)
        border = (x == 0) | (x == L - 1) | (y == 0) | (y == L - 1)
        assert deg[border].mean() < deg[~border].mean()
    assert max(np.hypot(a, b) for (a, b) in cnt) > (L // 2) * np.sqrt(2)        # longer than any periodic bond
    # away from the saturated nearest-neighbour shell (bonds are drawn without replacement) the counts follow
    # (number of pairs) r^-rho: displacement (3,0)+(0,3) against (4,0)+(0,4)
    n3 = cnt[(3, 0)] + cnt[(0, 3)]; n4 = cnt[(4, 0)] + cnt[(0, 4)]
    expect = ((L - 3) * 3.0 ** -rho) / ((L - 4) * 4.0 ** -rho)
    assert abs(n3 / n4 - expect) < 0.25 * expect, (n3, n4, expect)
    with pytest.raises(ValueError):
        levy.build(8, 3.0, 6, SEED, boundary="helical")


def _bond_set(g, s):
    n2o, rp, ci = g.new_to_old[s], g.row_ptr[s], g.col_idx[s]
    src = np.repeat(np.arange(g.N), np.diff(rp))
    return np.sort(n2o[src].astype(np.int64) * g.N + n2o[ci])


@pytest.mark.parametrize("L,rho", [(24, 2.5), (32, 3.5), (48, 4.5)])
def test_colour_reduction_keeps_the_bonds_stays_proper_and_shrinks_the_last_class(L, rho):
    """xy_levy_build_opt(reduce_moves_per_site): the optional local search after the smallest-last colouring (SURVEY C4:
    any proper colouring is a correct result; the number of colours sets the number of sequential
    phases).  Checked with the ORACLE's properness test; the bonds are those of the plain build; the colouring is
    deterministic; the last class shrinks (or the colour disappears); numbering is colour-major."""
    z, S = 6, 3
    plain = levy.build(L, rho, z, SEED, S=S, sample_base=2)
    red = levy.build(L, rho, z, SEED, S=S, sample_base=2, reduce_colours=8)
    again = levy.build(L, rho, z, SEED, S=S, sample_base=2, reduce_colours=8, n_threads=1)
    assert np.array_equal(red.colour, again.colour) and np.array_equal(red.col_idx, again.col_idx)
    for s in range(S):
        assert np.array_equal(_bond_set(plain, s), _bond_set(red, s))
        assert O.colouring_is_proper(red.row_ptr[s], red.col_idx[s], red.colour[s])
        assert np.all(np.diff(red.colour[s]) >= 0)
        q0, q1 = int(plain.n_colours[s]), int(red.n_colours[s])
        assert q1 <= q0 and red.colour[s].max() + 1 == q1
        if q1 == q0:
            assert (red.colour[s] == q1 - 1).sum() <= (plain.colour[s] == q0 - 1).sum()
    assert sum((red.colour[s] == red.n_colours[s] - 1).sum() if red.n_colours[s] == plain.n_colours[s] else 0 for s in range(S)) \
        < 0.7 * sum((plain.colour[s] == plain.n_colours[s] - 1).sum() for s in range(S))


def test_colour_reduce_on_hand_made_graphs():
    """a 5-clique keeps its fifth colour (one site); an odd cycle coloured with 4 colours drops to 3; bad input is refused"""
    k5 = [(a, b) for a in range(5) for b in range(a + 1, 5)]
    tail = [(4, 5), (5, 6), (6, 7)]
    rp, ci = G.csr_from_edges(8, k5 + tail)
    col = np.array([0, 1, 2, 3, 4, 0, 4, 0], np.int32)                  # proper, wasteful: two sites in the last class
    out, Q = levy.colour_reduce(rp, ci, col, 3, SEED)
    assert Q == 5 and O.colouring_is_proper(rp, ci, out) and (out == 4).sum() == 1
    rp, ci = G.csr_from_edges(7, G.ring_edges(7))
    out, Q = levy.colour_reduce(rp, ci, np.array([0, 1, 2, 3, 0, 1, 2], np.int32), 2, SEED)
    assert Q == 3 and O.colouring_is_proper(rp, ci, out)
    with pytest.raises(levy.LevyError):
        levy.colour_reduce(rp, ci, np.zeros(7, np.int32), 2, SEED)        # not proper
