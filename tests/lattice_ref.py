"""Independent lattice helpers for the tests (numpy + scipy only; imports neither oracle/ nor the
CUDA package): neighbour maps of the periodic lattice and connected components of a bond mask."""
import numpy as np
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components


def plus_neighbours(dim, L):
    """nb[k][i] = index of the +e_k neighbour of site i = x + L y (+ L^2 z), periodic."""
    N = L ** dim
    idx = np.arange(N, dtype=np.int64)
    out = []
    for k in range(dim):
        c = (idx // L ** k) % L
        out.append(idx + np.where(c == L - 1, -(L - 1) * L ** k, L ** k))
    return out


def components_min_label(dim, L, bonds):
    """(label, ncomp): minimum site index of every site's component of the active-bond graph
    (bit k of bonds[i] = bond i -> i + e_k), via scipy's connected_components."""
    N = L ** dim
    nb = plus_neighbours(dim, L)
    rows, cols = [], []
    for k in range(dim):
        a = np.nonzero(bonds & (1 << k))[0]
        rows.append(a)
        cols.append(nb[k][a])
    rows, cols = np.concatenate(rows), np.concatenate(cols)
    g = coo_matrix((np.ones(len(rows), dtype=np.int8), (rows, cols)), shape=(N, N))
    ncomp, comp = connected_components(g, directed=False)
    mins = np.full(ncomp, N, dtype=np.int64)
    np.minimum.at(mins, comp, np.arange(N))
    return mins[comp], ncomp
