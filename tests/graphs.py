"""Small hand-made graphs for tests: edge list -> symmetric CSR, a natural-order greedy colouring
and the colour-major renumbering.  Pure numpy/python, independent of oracle/ and of the package's
builder (it is what pins both)."""
import numpy as np


def csr_from_edges(N, edges):
    nb = [[] for _ in range(N)]
    for (a, b) in edges:
        nb[a].append(b)
        nb[b].append(a)
    row_ptr = np.zeros(N + 1, np.int32)
    cols = []
    for i in range(N):
        nb[i].sort()
        cols += nb[i]
        row_ptr[i + 1] = len(cols)
    return row_ptr, np.asarray(cols, np.int32).reshape(-1)


def greedy_colour(row_ptr, col_idx):
    N = len(row_ptr) - 1
    colour = -np.ones(N, np.int32)
    for v in range(N):
        used = {int(colour[u]) for u in col_idx[row_ptr[v]:row_ptr[v + 1]]}
        c = 0
        while c in used:
            c += 1
        colour[v] = c
    return colour


def colour_major(N, edges):
    """returns dict(row_ptr, col_idx, colour, class_ptr, new_to_old, edges) in colour-major numbering."""
    rp, ci = csr_from_edges(N, edges)
    col = greedy_colour(rp, ci)
    new_to_old = np.lexsort((np.arange(N), col)).astype(np.int32)
    old_to_new = np.empty(N, np.int32)
    old_to_new[new_to_old] = np.arange(N, dtype=np.int32)
    new_edges = [(int(old_to_new[a]), int(old_to_new[b])) for (a, b) in edges]
    rp2, ci2 = csr_from_edges(N, new_edges)
    colour = col[new_to_old].astype(np.int32)
    Q = int(colour.max()) + 1
    class_ptr = np.searchsorted(colour, np.arange(Q + 1)).astype(np.int32)
    return dict(N=N, row_ptr=rp2, col_idx=ci2, colour=colour, class_ptr=class_ptr,
                new_to_old=new_to_old, edges=new_edges)


def ring_edges(N):
    return [(i, (i + 1) % N) for i in range(N)]


def chain_edges(N):
    return [(i, i + 1) for i in range(N - 1)]


def square_lattice_edges(L):
    e = []
    for y in range(L):
        for x in range(L):
            i = y * L + x
            e.append((i, y * L + (x + 1) % L))
            e.append((i, ((y + 1) % L) * L + x))
    return e


def dense_energy_magnetisation(N, edges, theta):
    """Eq. 5 / Eq. 16 straight from the definition with a dense adjacency matrix; theta [N][R] fp32."""
    J = np.zeros((N, N))
    for (a, b) in edges:
        J[a, b] = J[b, a] = 1.0
    th = theta.astype(np.float64)
    E = np.array([-0.5 * np.sum(J * np.cos(th[:, r][:, None] - th[:, r][None, :])) for r in range(th.shape[1])])
    return E, np.cos(th).sum(0), np.sin(th).sum(0)
