"""Pins of the oracle's q-state clock model (the model the paper's "XY" program actually runs,
PAPER.md:88, 159, 210; readings 23-25) -- CPU only, independent of the CUDA path.

* exact enumeration of 3x3 lattices (q = 3, 4, 5): <E>, <M^2> within 3 sigma;
* the 4-state clock model is two decoupled Ising models at half the coupling
  (s_i . s_j = (sigma_i sigma_j + tau_i tau_j) / 2), so its energy at temperature T is Kaufman's
  exact finite-torus Ising energy at temperature 2 T;
* structural invariants with independent code: bonds only between sites whose components along the
  mirror normal have the same sign, labels = connected components (scipy), clusters mirrored
  entirely or not at all with p -> (m - p) mod q, |component| unchanged by the mirror;
* q = 512 against the continuous XY oracle (the paper: "the discretization level is small enough").
"""
import math

import numpy as np
import pytest

import exact
from lattice_ref import components_min_label, plus_neighbours
from oracle import sw_oracle as so
from stats import binned_mean_err


@pytest.mark.parametrize("q,T", [(3, 1.0), (4, 1.1), (5, 0.8), (4, 0.6)])
def test_clock_exact_enumeration_3x3(q, T):
    ex = exact.exact_clock(2, 3, q, T)
    es, ms = [], []
    for seed in (1, 2, 3, 4):
        o = so.Oracle(2, 3, so.CLOCK, q, 1.0 / T, seed)
        o.step(500)
        s = o.run_series(150000)
        es.append(s["E"])
        ms.append(s["M2"])
    for name, series, want in (("E", es, ex["E"]), ("M2", ms, ex["M2"])):
        means, errs = zip(*[binned_mean_err(x, 64) for x in series])
        mean, err = float(np.mean(means)), float(np.sqrt(np.sum(np.square(errs))) / len(errs))
        assert abs(mean - want) <= 3.0 * err, f"q={q} {name}: {mean} +- {err}, exact {want}"
        assert err < 0.02 * abs(want) + 1e-3


@pytest.mark.parametrize("L,T_ising", [(8, 2.269185), (16, 2.269185), (12, 3.0)])
def test_clock_q4_is_two_ising_models_at_double_temperature(L, T_ising):
    e_exact, _ = exact.kaufman_energy_per_site(L, T_ising)
    T = T_ising / 2.0
    means, errs = [], []
    for seed in (1, 2, 3, 4):
        o = so.Oracle(2, L, so.CLOCK, 4, 1.0 / T, seed)
        o.step(500)
        s = o.run_series(60000)
        m, e = binned_mean_err(s["E"] / (L * L), 64)
        means.append(m)
        errs.append(e)
    mean, err = float(np.mean(means)), float(np.sqrt(np.sum(np.square(errs))) / len(errs))
    assert abs(mean - float(e_exact)) <= 3.0 * err, f"E/N = {mean} +- {err}, exact {float(e_exact)}"
    assert err < 3e-3


@pytest.mark.parametrize("dim,L,q,beta", [(2, 12, 6, 1.0), (2, 9, 5, 1.3), (3, 6, 8, 0.5), (2, 16, 512, 1.1), (3, 5, 2, 0.3)])
def test_clock_step_invariants(dim, L, q, beta):
    o = so.Oracle(dim, L, so.CLOCK, q, beta, seed=7)
    nb = plus_neighbours(dim, L)
    N = L ** dim
    seen_mirrors = set()
    for step in range(8):
        before = o.spins().astype(np.int64)
        o.step(1)
        m = o.clock_mirror()
        seen_mirrors.add(m)
        assert 0 <= m < q
        bonds, labels, after = o.bonds(), o.labels().astype(np.int64), o.spins().astype(np.int64)
        a = np.sin(math.pi * (2 * before - m) / q)          # component along the mirror normal
        a[np.abs(a) < 1e-12] = 0.0
        for k in range(dim):
            act = (bonds >> k) & 1 == 1
            assert np.all(a[act] * a[nb[k]][act] > 0)
        ref, _ = components_min_label(dim, L, bonds)
        assert np.array_equal(labels, ref)
        changed = after != before
        mirrored = (m - before) % q
        fixed = mirrored == before                              # states on the mirror axis do not move
        assert np.array_equal(after[changed], mirrored[changed])
        flipped = changed | fixed
        # a cluster is mirrored entirely or not at all
        per_cluster = {}
        for i in range(N):
            if not fixed[i]:
                per_cluster.setdefault(labels[i], set()).add(bool(changed[i]))
        assert all(len(v) == 1 for v in per_cluster.values())
        a2 = np.sin(math.pi * (2 * after - m) / q)
        assert np.allclose(np.abs(a2), np.abs(a), atol=1e-12)
        assert after.min() >= 0 and after.max() < q
        D, n = o.clock_hist()
        assert D.sum() == dim * N and n.sum() == N
        e, mm, m2, m4 = o.observables()
        th = 2 * math.pi * after / q
        e_ref = -sum(np.cos(th - th[nb[k]]).sum() for k in range(dim))
        assert e == pytest.approx(e_ref, rel=1e-12, abs=1e-9)
        assert m2 == pytest.approx(np.cos(th).sum() ** 2 + np.sin(th).sum() ** 2, rel=1e-10, abs=1e-8)
    assert len(seen_mirrors) > 1 or q == 2


def test_clock_512_matches_continuous_xy():
    """"we dealt with the 512-state clock model.  The discretization level is small
    enough": E/N and <M^2> of q = 512 against the continuous XY oracle on 6^3 at T = 2.2019."""
    T, L = 2.2019, 6
    N = L ** 3
    res = {}
    for model, q in ((so.CLOCK, 512), (so.XY, 0)):
        es, ms = [], []
        for seed in (1, 2, 3):
            o = so.Oracle(3, L, model, q, 1.0 / T, seed)
            o.step(300)
            s = o.run_series(25000)
            es.append(binned_mean_err(s["E"] / N, 50))
            ms.append(binned_mean_err(s["M2"] / N ** 2, 50))
        res[model] = (np.mean([x[0] for x in es]), np.sqrt(np.sum([x[1] ** 2 for x in es])) / 3,
                      np.mean([x[0] for x in ms]), np.sqrt(np.sum([x[1] ** 2 for x in ms])) / 3)
    c, x = res[so.CLOCK], res[so.XY]
    assert abs(c[0] - x[0]) <= 3.0 * math.hypot(c[1], x[1])
    assert abs(c[2] - x[2]) <= 3.0 * math.hypot(c[3], x[3])
