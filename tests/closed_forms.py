"""Exact results that pin the oracle.  numpy/scipy only: nothing
here touches oracle/ or the CUDA path.

ring   : periodic N-site ring, Z ~ sum_n I_n(beta)^N (BASELINE.json north_star "exact ring closed form")
chain  : open chain (a tree), Z = (2 pi)^N I_0(beta)^(N-1)
quad   : brute-force quadrature on 3- and 4-site graphs (theta_0 fixed by O(2) symmetry)
beta0  : independent uniform angles
"""
import itertools

import numpy as np
from scipy.special import iv

SMALL_GRAPHS = {
    "P3": (3, [(0, 1), (1, 2)]),
    "K3": (3, [(0, 1), (1, 2), (0, 2)]),
    "P4": (4, [(0, 1), (1, 2), (2, 3)]),
    "star": (4, [(0, 1), (0, 2), (0, 3)]),
    "C4": (4, [(0, 1), (1, 2), (2, 3), (3, 0)]),
    "paw": (4, [(0, 1), (1, 2), (0, 2), (2, 3)]),
    "diamond": (4, [(0, 1), (1, 2), (2, 3), (3, 0), (0, 2)]),
    "K4": (4, [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]),
}


def ring(N, beta, nmax=60):
    """energy per site e and <m^2> of the periodic ring of N sites (N >= 3)."""
    n = np.arange(-nmax, nmax + 1)
    In = iv(n, beta)
    dIn = 0.5 * (iv(n - 1, beta) + iv(n + 1, beta))
    Z = np.sum(In ** N)
    e = -np.sum(In ** (N - 1) * dIn) / Z
    Inp1 = iv(n + 1, beta)
    C = [np.sum(In ** (N - r) * Inp1 ** r) / Z for r in range(N)]
    return float(e), float(np.sum(C) / N)


def ring_structure_factor(N, beta, k_index=1, nmax=60):
    """chi(k) = sum_r C(r) cos(2 pi k_index r / N) of the periodic ring, C(r) = <cos(theta_0 - theta_r)>
    = sum_n I_n^(N-r) I_(n+1)^r / sum_n I_n^N (transfer matrix in the angular-momentum basis)."""
    n = np.arange(-nmax, nmax + 1)
    In = iv(n, beta)
    Inp1 = iv(n + 1, beta)
    Z = np.sum(In ** N)
    C = np.array([np.sum(In ** (N - r) * Inp1 ** r) / Z for r in range(N)])
    return float(np.sum(C * np.cos(2.0 * np.pi * k_index * np.arange(N) / N)))


def chain(N, beta):
    """energy per site and <m^2> of the open chain of N sites."""
    t = iv(1, beta) / iv(0, beta)
    e = -(N - 1) * t / N
    r = np.arange(1, N)
    m2 = (N + 2.0 * np.sum((N - r) * t ** r)) / N ** 2
    return float(e), float(m2)


def tree_energy(n_bonds, beta):
    return float(-n_bonds * iv(1, beta) / iv(0, beta))


def quadrature(N, edges, beta, G=64):
    """<E>, Var E, <|m|>, <m^2>, <m^4> by periodic trapezoid on theta_1..theta_{N-1}, theta_0 = 0."""
    g = 2.0 * np.pi * np.arange(G) / G
    grids = np.meshgrid(*([g] * (N - 1)), indexing="ij")
    th = [np.zeros_like(grids[0])] + list(grids)
    E = np.zeros_like(grids[0])
    for (i, j) in edges:
        E -= np.cos(th[i] - th[j])
    mx = sum(np.cos(t) for t in th) / N
    my = sum(np.sin(t) for t in th) / N
    m2 = mx * mx + my * my
    w = np.exp(-beta * (E - E.min()))
    Z = w.sum()
    avg = lambda f: float((f * w).sum() / Z)
    Em = avg(E)
    return {"E": Em, "varE": avg(E * E) - Em * Em, "absm": avg(np.sqrt(m2)), "m2": avg(m2),
            "m4": avg(m2 * m2)}


def beta0_moments(N, n_bonds):
    """independent uniform angles: <m^2>=1/N, <m^4>=(2N-1)/N^3, <E>=0, Var E = E_b/2."""
    return {"m2": 1.0 / N, "m4": (2.0 * N - 1.0) / N ** 3, "E": 0.0, "varE": n_bonds / 2.0}
