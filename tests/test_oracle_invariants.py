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


def _group_word(G, t, n, seed):
    """DESIGN.md reading 6 with the Philox routine as a library step: word n of the stream of group G."""
    return so.philox4x32_10([G, t & 0xffffffff, t >> 32, 5 + 256 * (n >> 2)], [seed & 0xffffffff, seed >> 32])[n & 3]


@pytest.mark.parametrize("dim,L,model,q", [(2, 32, so.ISING, 0), (3, 8, so.ISING, 0), (2, 12, so.POTTS, 5), (3, 5, so.POTTS, 3)])
def test_group_keying_layout(dim, L, model, q):
    """Reading 6 (GROUP domain) restated: which word and bit feed which decision.  This is a check of
    the LAYOUT (a keying convention both sides of the parity tests must share), not a pin of the
    method: what pins the method's arithmetic is the exact-enumeration, FK and independence tests."""
    seed, N, beta = 11, L ** dim, 0.37
    o = so.Oracle(dim, L, model, q, beta, seed=seed)
    cold = np.ones(N, dtype=np.int8) if model == so.ISING else np.full(N, q - 1, dtype=np.uint8)
    o.set_spins(cold, 3)          # every pair is aligned: the bond byte is the random decision
    o.step(1)
    bonds, labels, spins = o.bonds(), o.labels(), o.spins()
    P32 = int(math.floor(-math.expm1(-(2.0 if model == so.ISING else 1.0) * beta) * 4294967296.0))
    for i in range(N):
        G, b = i >> 5, i & 31
        for k in range(dim):
            u = 0
            for s_ in range(32):
                u |= ((_group_word(G, 3, 1 + s_ * dim + k, seed) >> b) & 1) << (31 - s_)
            assert bool((bonds[i] >> k) & 1) == (u < P32), (i, k)
    for r in np.unique(labels)[:64]:
        r = int(r)
        if model == so.ISING:
            want = 1 if (_group_word(r >> 5, 3, 0, seed) >> (r & 31)) & 1 else -1
        else:
            want = (_group_word(r >> 5, 3, 128 + (r & 31), seed) * q) >> 32
        assert (spins[labels == r] == want).all()


@pytest.mark.parametrize("dim,L,T", [(2, 32, 2.269185), (3, 12, 4.5115)])
def test_bond_randoms_are_unbiased_and_independent(dim, L, T):
    """Pin of the transposed random words (reading 6): on an all-aligned lattice the bond bits ARE the
    random decisions u < P32.  Their frequency must be P32 / 2^32 for every direction and every
    position b inside a group (binomial, 3 sigma over all cells jointly: chi^2), and decisions must be
    uncorrelated between directions of a site, between neighbouring sites of a group, between
    consecutive steps and with the cluster draw of the site -- a word used twice, a shifted bit index
    or digits taken in the wrong order out of a shared word would show up here as a bias or a
    correlation of order one."""
    N, steps = L ** dim, 60
    p = -math.expm1(-2.0 / T)
    o = so.Oracle(dim, L, so.ISING, 0, 1.0 / T, seed=5)
    cold = np.ones(N, dtype=np.int8)
    acts, draws = [], []
    for t in range(steps):
        o.set_spins(cold, t)
        o.step(1)
        b = o.bonds()
        acts.append(np.stack([(b >> k) & 1 for k in range(dim)]).astype(np.float64))
        # draw of every site that is its own root (label == index)
        lab, sp = o.labels(), o.spins()
        d = np.full(N, np.nan)
        roots = np.nonzero(lab == np.arange(N))[0]
        d[roots] = (sp[roots] > 0)
        draws.append(d)
    A = np.stack(acts)                       # (steps, dim, N)
    n = steps * N
    for k in range(dim):
        assert abs(A[:, k].mean() - p) <= 3.0 * math.sqrt(p * (1 - p) / n)
    # per position inside a group: chi^2 over the 32 cells and dim directions
    cells = A.reshape(steps, dim, N // 32, 32).mean(axis=(0, 2))        # (dim, 32)
    var = p * (1 - p) / (steps * N // 32)
    chi2 = ((cells - p) ** 2 / var).sum()
    dof = 32 * dim
    assert abs(chi2 - dof) <= 3.0 * math.sqrt(2 * dof)
    c = A - p
    s2 = p * (1 - p)
    def corr(x, y):
        return float((x * y).mean() / s2), 1.0 / math.sqrt(x.size)
    pairs = [(c[:, 0], c[:, 1])]
    if dim == 3:
        pairs += [(c[:, 0], c[:, 2]), (c[:, 1], c[:, 2])]
    for k in range(dim):
        pairs.append((c[:, k, :-1], c[:, k, 1:]))           # neighbouring sites (same group except 1 in 32)
        pairs.append((c[:-1, k], c[1:, k]))                 # consecutive steps
    pairs.append((c[:, 0, :-1], c[:, 1, 1:]))
    for x, y in pairs:
        r, e = corr(x, y)
        assert abs(r) <= 3.0 * e, (r, e)
    # cluster draw vs the site's own bond decisions; and the draw itself is a fair coin
    D = np.stack(draws)
    ok = ~np.isnan(D)
    assert ok.sum() > 50
    assert abs(D[ok].mean() - 0.5) <= 3.0 * 0.5 / math.sqrt(ok.sum())


def test_ising_and_potts_q2_share_bonds():
    """What is left of the former bit identity R1 (the cluster draws of the two models are keyed
    differently, reading 6): Ising at beta and Potts q = 2 at 2 beta have the same threshold P32 and
    use the same digits, so from the same configuration (s = 2 k - 1) at the same step they activate
    exactly the same bonds and find the same clusters; and their moments agree (3 sigma) on 4x4."""
    from stats import pooled
    beta = 1.0 / 2.269185
    a = so.Oracle(2, 20, so.ISING, 0, beta, seed=9)
    b = so.Oracle(2, 20, so.POTTS, 2, 2.0 * beta, seed=9)
    for t in range(5):
        k = (a.spins() > 0).astype(np.uint8)
        b.set_spins(k, a.t)
        a.step(1)
        b.step(1)
        assert np.array_equal(a.bonds(), b.bonds()) and np.array_equal(a.labels(), b.labels())
    ra, rb = [], []
    for seed in (1, 2, 3, 4):
        x = so.Oracle(2, 4, so.ISING, 0, beta, seed)
        y = so.Oracle(2, 4, so.POTTS, 2, 2.0 * beta, seed)
        x.step(500)
        y.step(500)
        ra.append(x.run_series(60000))
        rb.append(y.run_series(60000))
    for key, fa, fb in [("E", lambda r: r["E"], lambda r: 2.0 * r["E"] - 32.0),       # Eq. 1 vs Eq. 2: E_I = 2 E_P - #bonds
                        ("M2", lambda r: r["M2"], lambda r: r["M2"]),
                        ("n_clusters", lambda r: r["n_clusters"], lambda r: r["n_clusters"])]:
        ma, ea = pooled([fa(r) for r in ra])
        mb, eb = pooled([fb(r) for r in rb])
        assert abs(ma - mb) <= 3.0 * math.hypot(ea, eb), key


def test_thresholds_of_the_configs():
    """The integer thresholds SURVEY.md S4 prints for the BASELINE configs: the measured active-bond
    fraction among equal pairs must sit at P32 / 2^32 (binomial 3 sigma)."""
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
        assert abs(n_act - p * n_eq) < 3.0 * math.sqrt(n_eq * p * (1 - p))


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
