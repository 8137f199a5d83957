"""Exact results used to pin the oracle -- independent of oracle/ and of the CUDA path.

* brute-force enumeration of every spin state of a tiny periodic lattice (Ising Eq. 1, Potts Eq. 2
  of arXiv 1403.7560) -> exact <E>, <E^2>, <M^2>, <M^4>, <|M|>, <#equal pairs>;
* brute-force enumeration of every bond configuration of the Fortuin-Kasteleyn representation
  (weight p^|A| (1-p)^(B-|A|) q^C(A)) of a 3x3 lattice -> exact <#active bonds>, <#clusters>,
  Var(#clusters), <sum_c n_c^2>;
* Kaufman's partition function of the finite m x n torus (B. Kaufman, Phys. Rev. 76 (1949) 1232)
  -> exact <E>/N of the 2D Ising model at any L (Onsager's -sqrt(2) is its L -> infinity limit at
  T_c).  The formula itself is pinned to the enumeration at 3x3 and 4x4 in test_exact_pins.py.
"""
import itertools

import mpmath as mp
import numpy as np


def lattice_bonds(dim, L):
    """List of (i, j) for every owned bond i -> i + e_k, periodic, x fastest."""
    N = L ** dim
    idx = np.arange(N)
    coords = [(idx // L ** k) % L for k in range(dim)]
    bonds = []
    for k in range(dim):
        j = idx + np.where(coords[k] == L - 1, -(L - 1) * L ** k, L ** k)
        bonds += list(zip(idx.tolist(), j.tolist()))
    return bonds


def enumerate_spin_states(dim, L, q):
    """All q^N states as an (q^N, N) uint8 array."""
    N = L ** dim
    n = q ** N
    s = np.empty((n, N), dtype=np.int8)
    a = np.arange(n, dtype=np.int64)
    for i in range(N):
        s[:, i] = (a // q ** i) % q
    return s


def exact_ising(dim, L, T):
    """Boltzmann averages of the Ising model (Eq. 1, J = 1) by enumeration of all 2^N states."""
    N = L ** dim
    s = enumerate_spin_states(dim, L, 2).astype(np.int64) * 2 - 1
    bonds = lattice_bonds(dim, L)
    E = np.zeros(s.shape[0], dtype=np.int64)
    for (i, j) in bonds:
        E -= s[:, i] * s[:, j]
    M = s.sum(axis=1)
    w = np.exp(-(E - E.min()) / T)
    Z = w.sum()
    avg = lambda x: float((w * x).sum() / Z)
    nequal = (len(bonds) - E) / 2
    return {
        "N": N, "n_bonds": len(bonds),
        "E": avg(E), "E2": avg(E.astype(float) ** 2), "M2": avg(M.astype(float) ** 2),
        "M4": avg(M.astype(float) ** 4), "absM": avg(np.abs(M)), "n_equal": avg(nequal),
        "E_values": E, "weights": w / Z,
    }


def exact_potts(dim, L, q, T):
    """Boltzmann averages of the q-state Potts model (Eq. 2: E = #unequal pairs, J = 1)."""
    N = L ** dim
    s = enumerate_spin_states(dim, L, q)
    bonds = lattice_bonds(dim, L)
    E = np.zeros(s.shape[0], dtype=np.int64)
    for (i, j) in bonds:
        E += (s[:, i] != s[:, j])
    nk2 = np.zeros(s.shape[0], dtype=np.float64)
    for k in range(q):
        nk2 += (s == k).sum(axis=1).astype(np.float64) ** 2
    M2 = (q * nk2 - N * N) / (q - 1)          # Eq. (5)
    w = np.exp(-(E - E.min()) / T)
    Z = w.sum()
    avg = lambda x: float((w * x).sum() / Z)
    return {"N": N, "n_bonds": len(bonds), "E": avg(E), "E2": avg(E.astype(float) ** 2),
            "M2": avg(M2), "M4": avg(M2 ** 2), "n_equal": avg(len(bonds) - E)}


def exact_fk(dim, L, q, p):
    """Averages over the Fortuin-Kasteleyn bond measure by enumeration of all 2^B bond sets."""
    N = L ** dim
    bonds = lattice_bonds(dim, L)
    B = len(bonds)
    assert B <= 20, "FK enumeration is only feasible for B <= 20 bonds"
    n = 1 << B
    cfg = np.arange(n, dtype=np.int64)
    active = np.stack([(cfg >> b) & 1 for b in range(B)], axis=1).astype(bool)   # (n, B)
    lab = np.tile(np.arange(N, dtype=np.int16), (n, 1))
    for _ in range(N):                       # label propagation to the fixed point
        for b, (i, j) in enumerate(bonds):
            m = np.minimum(lab[:, i], lab[:, j])
            a = active[:, b]
            lab[a, i] = m[a]
            lab[a, j] = m[a]
    # chase to roots (labels are min over direct neighbours only until converged)
    for _ in range(N):
        lab = np.take_along_axis(lab, lab.astype(np.int64), axis=1)
    ncl = np.zeros(n, dtype=np.int64)
    snc2 = np.zeros(n, dtype=np.float64)
    for r in range(N):
        size = (lab == r).sum(axis=1)
        ncl += (size > 0)
        snc2 += size.astype(np.float64) ** 2
    nact = active.sum(axis=1)
    w = p ** nact * (1 - p) ** (B - nact) * float(q) ** ncl
    Z = w.sum()
    avg = lambda x: float((w * x).sum() / Z)
    return {"n_active": avg(nact), "n_clusters": avg(ncl),
            "var_clusters": avg(ncl.astype(float) ** 2) - avg(ncl) ** 2, "sum_nc2": avg(snc2)}


def kaufman_lnZ(m, n, K):
    """ln Z of the m x n periodic square-lattice Ising model at coupling K = J/T (mpmath)."""
    K = mp.mpf(K)
    c = mp.cosh(2 * K) * mp.coth(2 * K)

    def gamma(l):
        if l == 0:
            return 2 * K + mp.log(mp.tanh(K))
        return mp.acosh(c - mp.cos(mp.pi * l / n))

    p1 = mp.mpf(1); p2 = mp.mpf(1); p3 = mp.mpf(1); p4 = mp.mpf(1)
    for r in range(n):
        go, ge = gamma(2 * r + 1), gamma(2 * r)
        p1 *= 2 * mp.cosh(m * go / 2)
        p2 *= 2 * mp.sinh(m * go / 2)
        p3 *= 2 * mp.cosh(m * ge / 2)
        p4 *= 2 * mp.sinh(m * ge / 2)
    return mp.log(mp.mpf(1) / 2) + (mp.mpf(m * n) / 2) * mp.log(2 * mp.sinh(2 * K)) + mp.log(p1 + p2 + p3 + p4)


def kaufman_energy_per_site(L, T, dps=None):
    """<E>/N = -(1/N) d ln Z / dK for the L x L torus; C/N = K^2 (1/N) d^2 ln Z / dK^2."""
    mp.mp.dps = dps or 50
    K = mp.mpf(1) / mp.mpf(T)
    f = lambda k: kaufman_lnZ(L, L, k)
    d1 = mp.diff(f, K, 1)
    d2 = mp.diff(f, K, 2)
    N = L * L
    return float(-d1 / N), float(K * K * d2 / N)


def exact_clock(dim, L, q, T):
    """Boltzmann averages of the q-state clock model (Eq. 3 with theta = 2 pi p / q, PAPER.md:84-88,
    J = 1) by enumeration of all q^N states: <E>, <E^2>, <M^2> with M = |sum_i (cos, sin) theta_i|."""
    s = enumerate_spin_states(dim, L, q).astype(np.int64)
    bonds = lattice_bonds(dim, L)
    ang = 2.0 * np.pi / q
    E = np.zeros(s.shape[0], dtype=np.float64)
    for (i, j) in bonds:
        E -= np.cos(ang * (s[:, i] - s[:, j]))
    mx = np.cos(ang * s).sum(axis=1)
    my = np.sin(ang * s).sum(axis=1)
    w = np.exp(-(E - E.min()) / T)
    Z = w.sum()
    avg = lambda x: float((w * x).sum() / Z)
    M2 = mx * mx + my * my
    return {"N": L ** dim, "n_bonds": len(bonds), "E": avg(E), "E2": avg(E * E), "M2": avg(M2), "M4": avg(M2 * M2)}
