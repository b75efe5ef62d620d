"""Pins of the oracle's random-walk self-return histogram (SURVEY.md 8(f) item 3; PAPER.md:149-155 Eq. 11, :436-440
App. A): the exact return probability (A^t)_00 from numpy matrix powers on small graphs, the closed forms of the ring
and the square lattice, and the spectral dimension 2 of the periodic square lattice."""
import numpy as np
from scipy.special import comb

import graphs as G
import oracle as O

SEED = 0x3A1C
W = 200_000


def exact_return(row_ptr, col_idx, origin, n_steps):
    N = len(row_ptr) - 1
    P = np.zeros((N, N))
    for i in range(N):
        nb = col_idx[row_ptr[i]:row_ptr[i + 1]]
        if len(nb) == 0:
            P[i, i] = 1.0
        for j in nb:
            P[i, j] = 1.0 / len(nb)
    out, M = [1.0], np.eye(N)
    for _ in range(n_steps):
        M = M @ P
        out.append(M[origin, origin])
    return np.array(out)


def check(hist, exact, n):
    p = hist / n
    sig = np.sqrt(np.maximum(exact * (1 - exact), 1e-12) / n)
    assert np.all(np.abs(p - exact) <= 4.5 * sig + 1e-12), np.max(np.abs(p - exact) / (sig + 1e-12))


def test_small_graphs_matrix_power():
    for N, edges, origin in [(4, [(0, 1), (0, 2), (0, 3)], 0), (4, [(0, 1), (0, 2), (0, 3)], 2),
                             (4, [(0, 1), (1, 2), (0, 2), (2, 3)], 2), (5, [(0, 1), (1, 2), (2, 3), (3, 4), (4, 0), (0, 2)], 0),
                             (3, [(0, 1)], 2)]:                     # the last origin is an isolated site: it stays
        rp, ci = G.csr_from_edges(N, edges)
        h = O.random_walk(rp, ci, np.full(W, origin, np.int32), 12, SEED)
        assert h[0] == W
        check(h, exact_return(rp, ci, origin, 12), W)


def test_ring_and_square_lattice_closed_forms():
    N = 64                                                        # ring: P(2n) = C(2n, n) / 4^n while 2n < N
    rp, ci = G.csr_from_edges(N, G.ring_edges(N))
    h = O.random_walk(rp, ci, np.full(W, 5, np.int32), 20, SEED)
    ex = np.array([comb(t, t // 2) / 2.0 ** t if t % 2 == 0 else 0.0 for t in range(21)])
    assert np.all(h[1::2] == 0)                                   # bipartite: no return at odd times (exact)
    check(h, ex, W)
    L = 32                                                        # square lattice: P(2n) = [C(2n, n) / 4^n]^2 while 2n < L
    rp, ci = G.csr_from_edges(L * L, G.square_lattice_edges(L))
    h = O.random_walk(rp, ci, np.full(W, L * L // 2 + L // 2, np.int32), 24, SEED + 1)
    ex = np.array([(comb(t, t // 2) / 2.0 ** t) ** 2 if t % 2 == 0 else 0.0 for t in range(25)])
    assert np.all(h[1::2] == 0)
    check(h, ex, W)
    # Eq. 11: P ~ tau^(-dbar/2), dbar = 2 on the square lattice: log-log slope over tau = 8..24
    t = np.arange(8, 25, 2)
    slope = np.polyfit(np.log(t), np.log(h[t] / W), 1)[0]
    assert abs(-2 * slope - 2.0) < 0.15, slope


def test_walk_is_reproducible_and_sample_dependent():
    rp, ci = G.csr_from_edges(16, G.ring_edges(16))
    st = np.arange(1000, dtype=np.int32) % 16
    a = O.random_walk(rp, ci, st, 30, SEED, 3)
    assert np.array_equal(a, O.random_walk(rp, ci, st, 30, SEED, 3))
    assert not np.array_equal(a, O.random_walk(rp, ci, st, 30, SEED, 4))
    assert not np.array_equal(a, O.random_walk(rp, ci, st, 30, SEED + 1, 3))
