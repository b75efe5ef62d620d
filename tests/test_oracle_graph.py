"""Pins for the oracle's definition-level Levy graph and colouring."""
import numpy as np
import pytest
from scipy.stats import chi2, poisson

import graphs as G
import oracle as O

SEED = 0x12113991


def _min_image_r2(L, i, j):
    dx = abs(i % L - j % L); dy = abs(i // L - j // L)
    dx = min(dx, L - dx); dy = min(dy, L - dy)
    return dx * dx + dy * dy


@pytest.mark.parametrize("L,rho,z", [(8, 3.5, 6), (16, 3.5, 6), (12, 0.0, 4), (16, 2.5, 6)])
def test_levy_structure(L, rho, z):
    N = L * L
    edges, draws = O.levy_edges(L, rho, z, SEED, 0)
    assert len(edges) == N * z // 2 and draws >= len(edges)            # E_b = N z / 2 exactly
    assert np.all(edges[:, 0] != edges[:, 1])                          # no self loops
    und = {(min(a, b), max(a, b)) for a, b in edges}
    assert len(und) == len(edges)                                      # no duplicates
    rmax2 = max(_min_image_r2(L, a, b) for a, b in edges)
    assert rmax2 <= 2 * (L // 2) ** 2                                  # r_max = [L/2] sqrt 2
    rp, ci = O.csr_from_edges(N, edges)
    rp2, ci2 = G.csr_from_edges(N, [tuple(e) for e in edges])
    assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)         # CSR vs independent numpy build
    assert rp[-1] == N * z                                             # nnz = N z (symmetric)


def test_levy_is_deterministic_and_sample_dependent():
    e0, _ = O.levy_edges(8, 3.5, 6, SEED, 0)
    e0b, _ = O.levy_edges(8, 3.5, 6, SEED, 0)
    e1, _ = O.levy_edges(8, 3.5, 6, SEED, 1)
    e2, _ = O.levy_edges(8, 3.5, 6, SEED + 1, 0)
    assert np.array_equal(e0, e0b) and not np.array_equal(e0, e1) and not np.array_equal(e0, e2)


def test_levy_large_rho_is_square_lattice_two_colours():
    """rho -> inf at z=4 recovers the square lattice: all degrees 4, every bond length 1, and the
    colouring finds exactly two colours."""
    L = 8
    edges, _ = O.levy_edges(L, 100.0, 4, SEED, 0)
    assert {(min(a, b), max(a, b)) for a, b in edges} == {(min(a, b), max(a, b)) for a, b in G.square_lattice_edges(L)}
    rp, ci = O.csr_from_edges(L * L, edges)
    assert np.all(np.diff(rp) == 4)
    colour, Q = O.colour_smallest_last(rp, ci)
    assert Q == 2 and O.colouring_is_proper(rp, ci, colour)
    assert np.array_equal(colour == colour[0], np.array([(i % L + i // L) % 2 == 0 for i in range(L * L)]))


def test_levy_rho0_is_erdos_renyi_poisson_degrees():
    """rho = 0: bonds uniform over all pairs; degree ~ Poisson(z)."""
    L, z = 32, 6
    deg = []
    for s in range(3):
        edges, _ = O.levy_edges(L, 0.0, z, SEED, s)
        deg.append(np.bincount(edges.reshape(-1), minlength=L * L))
    deg = np.concatenate(deg)
    assert deg.mean() == z
    kmax = 14
    obs = np.bincount(np.minimum(deg, kmax), minlength=kmax + 1).astype(float)
    p = poisson.pmf(np.arange(kmax + 1), z); p[kmax] = 1 - p[:kmax].sum()
    stat = ((obs - deg.size * p) ** 2 / (deg.size * p)).sum()
    assert stat < chi2.ppf(0.9999, kmax)       # (fixed-total-degree constraint only lowers the variance)


def test_levy_bond_length_law():
    """P(bond at squared distance r2) ~ multiplicity(r2) * r^-rho (Eq. 6) while bonds are sparse
    (z=2, rho=1.5: duplicate rejections distort the law by < 1%)."""
    L, rho, z = 24, 1.5, 2
    N = L * L
    mult = {}
    for d in range(1, N):
        r2 = _min_image_r2(L, 0, d)
        mult[r2] = mult.get(r2, 0) + 1
    keys = sorted(mult)
    w = np.array([mult[k] * k ** (-rho / 2) for k in keys]); w /= w.sum()
    counts = np.zeros(len(keys)); idx = {k: n for n, k in enumerate(keys)}
    for s in range(6):
        edges, _ = O.levy_edges(L, rho, z, SEED, s)
        for a, b in edges:
            counts[idx[_min_image_r2(L, a, b)]] += 1
    tot = counts.sum()
    big = w * tot >= 8
    o = np.append(counts[big], counts[~big].sum()); e = np.append(w[big] * tot, w[~big].sum() * tot)
    stat = ((o - e) ** 2 / e).sum()
    assert stat < chi2.ppf(0.9999, len(o) - 1)
    # nearest-neighbour fraction specifically
    assert abs(counts[0] / tot - w[0]) < 5 * np.sqrt(w[0] * (1 - w[0]) / tot)


@pytest.mark.parametrize("L,rho,z", [(8, 3.5, 6), (16, 3.5, 6), (16, 0.0, 6), (16, 2.5, 4)])
def test_colouring_proper_and_renumbering(L, rho, z):
    N = L * L
    edges, _ = O.levy_edges(L, rho, z, SEED, 1)
    rp, ci = O.csr_from_edges(N, edges)
    colour, Q = O.colour_smallest_last(rp, ci)
    assert colour.min() == 0 and colour.max() == Q - 1 and Q <= int(np.diff(rp).max()) + 1
    for a, b in edges:                                          # bit-exact properness, by hand
        assert colour[a] != colour[b]
    assert O.colouring_is_proper(rp, ci, colour)
    # smallest-last bound: Q <= 1 + max over removal order of back-degree <= 1 + degeneracy
    new_to_old, rp2, ci2, c2 = O.renumber_colour_major(rp, ci, colour)
    assert sorted(new_to_old) == list(range(N)) and np.all(np.diff(c2) >= 0)
    assert np.array_equal(c2, colour[new_to_old])
    old_to_new = np.empty(N, np.int64); old_to_new[new_to_old] = np.arange(N)
    rp3, ci3 = G.csr_from_edges(N, [(int(old_to_new[a]), int(old_to_new[b])) for a, b in edges])
    assert np.array_equal(rp2, rp3) and np.array_equal(ci2, ci3)
    assert O.colouring_is_proper(rp2, ci2, c2)
    # within a class the old (lattice) order is kept
    for c in range(Q):
        cls = new_to_old[c2 == c]
        assert np.all(np.diff(cls) > 0)


def test_colouring_detects_improper():
    g = G.colour_major(4, G.ring_edges(4))
    assert O.colouring_is_proper(g["row_ptr"], g["col_idx"], g["colour"])
    bad = g["colour"].copy(); bad[:] = 0
    assert not O.colouring_is_proper(g["row_ptr"], g["col_idx"], bad)


def test_smallest_last_on_known_graphs():
    # trees are 2-colourable by smallest-last (degeneracy 1); odd ring needs 3; K4 needs 4
    for N, edges, q in [(7, G.chain_edges(7), 2), (6, [(0, k) for k in range(1, 6)], 2), (5, G.ring_edges(5), 3),
                        (6, G.ring_edges(6), 2), (4, [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)], 4)]:
        rp, ci = G.csr_from_edges(N, edges)
        colour, Q = O.colour_smallest_last(rp, ci)
        assert Q == q and O.colouring_is_proper(rp, ci, colour)
