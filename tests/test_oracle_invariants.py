"""Structural invariants I1-I6 of the oracle's SW step,
checked with code that is independent of the oracle: neighbour maps are rebuilt here with numpy and
connected components come from scipy.sparse.csgraph (CPU only)."""
import math

import numpy as np
import pytest

from lattice_ref import components_min_label, plus_neighbours
from oracle import sw_oracle as so

CASES = [(2, 3, so.ISING, 0, 0.44), (2, 4, so.ISING, 0, 0.44), (2, 7, so.POTTS, 3, 1.0), (2, 32, so.ISING, 0, 0.4406868),
         (2, 48, so.POTTS, 4, 1.1), (3, 3, so.ISING, 0, 0.22), (3, 5, so.POTTS, 3, 0.55), (3, 16, so.ISING, 0, 0.2216544),
         (2, 20, so.XY, 0, 1.1), (3, 8, so.XY, 0, 0.45416)]


@pytest.mark.parametrize("dim,L,model,q,beta", CASES)
def test_step_invariants(dim, L, model, q, beta):
    o = so.Oracle(dim, L, model, q, beta, seed=11)
    nb = plus_neighbours(dim, L)
    N = L ** dim
    for step in range(6):
        before = o.spins().copy()
        o.step(1)
        bonds, labels, after = o.bonds(), o.labels().astype(np.int64), o.spins()
        assert bonds.max() < (1 << dim)
        # I1: bonds join only aligned spins
        if model == so.XY:
            rx, ry, c = o.xy_dir()
            a = np.float64(rx) * np.cos(before.astype(np.float64)) + np.float64(ry) * np.sin(before.astype(np.float64))
        for k in range(dim):
            act = (bonds >> k) & 1 == 1
            if model == so.XY:
                assert np.all(a[act] * a[nb[k]][act] > 0)
            else:
                assert np.all(before[act] == before[nb[k]][act])
        # I2 + I3: labels are exactly the connected components, named by their minimum index
        ref, ncomp = components_min_label(dim, L, bonds)
        assert np.array_equal(labels, ref)
        assert np.all(labels <= np.arange(N)) and np.array_equal(labels[labels], labels)
        # I4: clusters uniform after the flip; XY: reflected entirely or not at all
        if model != so.XY:
            assert np.array_equal(after, after[labels])
            for k in range(dim):
                act = (bonds >> k) & 1 == 1
                assert np.all(after[act] == after[nb[k]][act])
        else:
            changed = after != before
            assert np.array_equal(changed, changed[labels])
            a2 = np.float64(rx) * np.cos(after.astype(np.float64)) + np.float64(ry) * np.sin(after.astype(np.float64))
            assert np.allclose(np.abs(a2), np.abs(a), atol=2e-6)
            assert np.all(np.sign(a2[changed]) == -np.sign(a[changed]))
            assert after.min() >= 0.0 and after.max() <= np.float32(2 * math.pi)


def test_beta_zero_and_cold_start():
    """I5: beta = 0 -> no bonds, label[i] = i; large beta + aligned start -> one cluster, label 0."""
    for dim, L in [(2, 6), (3, 4), (2, 32)]:
        N = L ** dim
        o = so.Oracle(dim, L, so.ISING, 0, 0.0, seed=3)
        o.step(1)
        assert not o.bonds().any() and np.array_equal(o.labels(), np.arange(N))
        o = so.Oracle(dim, L, so.ISING, 0, 40.0, seed=3)
        o.set_spins(np.ones(N, dtype=np.int8), 0)
        o.step(1)
        assert np.all(o.bonds() == (1 << dim) - 1) and not o.labels().any()
        assert len(np.unique(o.spins())) == 1
        o = so.Oracle(dim, L, so.POTTS, 5, 50.0, seed=3)
        o.set_spins(np.full(N, 2, dtype=np.uint8), 0)
        o.step(1)
        assert np.all(o.bonds() == (1 << dim) - 1) and not o.labels().any()


def test_determinism_and_state_injection():
    """I6: a step is a pure function of (seed, spins, t)."""
    a = so.Oracle(2, 24, so.POTTS, 3, 1.0, seed=5)
    b = so.Oracle(2, 24, so.POTTS, 3, 1.0, seed=5)
    a.step(7)
    b.step(4)
    c = so.Oracle(2, 24, so.POTTS, 3, 1.0, seed=5)
    c.set_spins(b.spins(), b.t)
    b.step(3)
    c.step(3)
    assert np.array_equal(a.spins(), b.spins()) and np.array_equal(a.spins(), c.spins())
    assert np.array_equal(a.labels(), c.labels()) and np.array_equal(a.bonds(), c.bonds())
    d = so.Oracle(2, 24, so.POTTS, 3, 1.0, seed=6)
    d.step(7)
    assert not np.array_equal(a.spins(), d.spins())


def _ising_bits_restated(dim, i, t, seed):
    """DESIGN.md reading 6 written out again with the Philox routine as a library step: the F-bit
    bond fields and the top bit of site i's piece of PACK call i // S."""
    S, W = (4, 32) if dim == 2 else (2, 64)
    F = (W - 1) // dim
    w = so.philox4x32_10([i // S, t & 0xffffffff, t >> 32, 1], [seed & 0xffffffff, seed >> 32])
    piece = w[i % 4] if dim == 2 else (w[2 * (i % 2)] | (w[2 * (i % 2) + 1] << 32))
    return [(piece >> (F * k)) & ((1 << F) - 1) for k in range(dim)], (piece >> (W - 1)) & 1, F


@pytest.mark.parametrize("dim,L", [(2, 32), (3, 8)])
def test_ising_packed_keying_and_tie_rule(dim, L):
    """Reading 6 (packed Ising keying): every bond decision and every cluster value of the oracle
    against the rule restated here, including bonds whose field sits exactly on the threshold
    (settled by the TIE call).  A tie has probability 2^-F, so it is forced: the threshold's top
    part is set to a field value that does occur at t = 0 (beta is free)."""
    seed, N = 11, L ** dim
    F = (31 if dim == 2 else 63) // dim
    cold = np.ones(N, dtype=np.int8)
    ties = 0
    for site, k0 in [(5, 0), (N // 2 + 3, dim - 1), (N - 1, 1), (17, 0)]:
        v = _ising_bits_restated(dim, site, 0, seed)[0][k0]
        p_bond = (v + 0.5) / (1 << F)          # Ptop = v, Plow = half its range
        beta = -0.5 * math.log1p(-p_bond)
        P32 = int(math.floor(-math.expm1(-2.0 * beta) * 4294967296.0))
        Ptop, Plow = P32 >> (32 - F), P32 & ((1 << (32 - F)) - 1)
        assert Ptop == v and 0 < Plow < (1 << (32 - F))
        o = so.Oracle(dim, L, so.ISING, 0, beta, seed=seed)
        o.set_spins(cold, 0)          # every pair is aligned: the bond byte is the random decision
        o.step(1)
        bonds, labels, spins = o.bonds(), o.labels(), o.spins()
        for i in range(N):
            fields, top, _ = _ising_bits_restated(dim, i, 0, seed)
            for k in range(dim):
                if fields[k] == Ptop:
                    ties += 1
                    tw = so.philox4x32_10([i, 0, 0, 4], [seed, 0])
                    want = (tw[k] >> F) < Plow
                else:
                    want = fields[k] < Ptop
                assert bool((bonds[i] >> k) & 1) == want, (site, i, k)
        for r in np.unique(labels)[:64]:
            _, top, _ = _ising_bits_restated(dim, int(r), 0, seed)
            assert (spins[labels == r] == (1 if top else -1)).all()
    assert ties >= 4, "the tie rule was not exercised"


def test_ising_threshold_split_is_exact():
    """P(active) = Ptop / 2^F + 2^-F Plow / 2^(32-F) must equal P32 / 2^32 for every P32."""
    from fractions import Fraction
    rng = np.random.default_rng(3)
    for F in (15, 21):
        for P32 in [0, 1, 2 ** 32 - 1, 2515933809, 1537996873] + [int(x) for x in rng.integers(0, 2 ** 32, size=50)]:
            Ptop, Plow = P32 >> (32 - F), P32 & ((1 << (32 - F)) - 1)
            assert Fraction(Ptop, 2 ** F) + Fraction(1, 2 ** F) * Fraction(Plow, 2 ** (32 - F)) == Fraction(P32, 2 ** 32)


def test_thresholds_of_the_configs():
    """The integer thresholds SURVEY.md S4 prints for the BASELINE configs: the measured active-bond
    fraction among equal pairs must sit at P32 / 2^32 (binomial 4 sigma)."""
    for dim, L, model, q, T, P32 in [(2, 64, so.ISING, 0, 2.269185, 2515933809), (2, 64, so.POTTS, 3, 0.994973, 2722899936),
                                     (3, 16, so.ISING, 0, 4.5115, 1537996873)]:
        o = so.Oracle(dim, L, model, q, 1.0 / T, seed=1)
        nb = plus_neighbours(dim, L)
        n_eq = n_act = 0
        for _ in range(20):
            s = o.spins().copy()
            o.step(1)
            b = o.bonds()
            for k in range(dim):
                n_eq += int((s == s[nb[k]]).sum())
                n_act += int(((b >> k) & 1).sum())
        p = P32 / 2.0 ** 32
        assert abs(n_act - p * n_eq) < 4.0 * math.sqrt(n_eq * p * (1 - p))


def test_observables_definitions():
    """Eq. (1), (2), (4), (5) and Eq. (3) re-evaluated with numpy on the oracle's spins."""
    o = so.Oracle(3, 6, so.ISING, 0, 0.2, seed=2)
    o.step(3)
    s = o.spins().astype(np.int64)
    nb = plus_neighbours(3, 6)
    E, M, M2, M4 = o.observables()
    assert E == -sum(int((s * s[n]).sum()) for n in nb) and M == s.sum() and M2 == M * M and M4 == M2 * M2
    assert o.counts() == (int(E), [int(M)])
    o = so.Oracle(2, 9, so.POTTS, 4, 0.9, seed=2)
    o.step(3)
    s = o.spins().astype(np.int64)
    nb = plus_neighbours(2, 9)
    E, M, M2, M4 = o.observables()
    nk = np.bincount(s, minlength=4)
    assert E == sum(int((s != s[n]).sum()) for n in nb)
    assert M2 == pytest.approx((4 * (nk ** 2).sum() - 81 ** 2) / 3) and M == pytest.approx(math.sqrt(M2))
    assert o.counts() == (int(E), nk.tolist())
    o = so.Oracle(2, 10, so.XY, 0, 1.0, seed=2)
    o.step(3)
    th = o.spins().astype(np.float64)
    nb = plus_neighbours(2, 10)
    E, M, M2, M4 = o.observables()
    assert E == pytest.approx(-sum(np.cos(th - th[n]).sum() for n in nb), rel=1e-12)
    assert M2 == pytest.approx(np.cos(th).sum() ** 2 + np.sin(th).sum() ** 2, rel=1e-12)
    assert M4 == pytest.approx(M2 * M2)
