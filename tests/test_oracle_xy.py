"""Pins of the oracle's XY path (Wolff-embedded SW; Eq. 3) -- CPU only.

There is no closed form for the 3D XY model, so the continuous model is pinned by
  R2  a special case that reduces to the Ising model, whose exact values are known, and
  R3  agreement with an independent algorithm (single-spin Metropolis, written here in numpy with
      numpy's own generator; it shares nothing with the oracle), and
  F3  the cluster identity <M^2> = 2 <sum_c (sum_{i in c} a_i)^2>, which ties labels to spins.
"""
import math

import numpy as np
import pytest

import exact
from lattice_ref import plus_neighbours
from oracle import sw_oracle as so
from stats import binned_mean_err, pooled

NSIG = 3.0


def test_xy_restricted_to_two_angles_is_the_ising_model():
    """R2: all theta in {0, float(pi)}, direction forced to r = (1, 0): a_i = +-1 (to 1e-7),
    p = 1 - exp(-2 beta), the reflection c - theta with c = pi maps 0 <-> float(pi) exactly.
    The XY oracle must then reproduce the exact 4x4 Ising averages (pin P1)."""
    T = 2.269185
    ex = exact.exact_ising(2, 4, T)
    Es, M2s = [], []
    for seed in (1, 2, 3, 4):
        o = so.Oracle(2, 4, so.XY, 0, 1.0 / T, seed)
        o.force_xy_phi(True, 0.0)
        rng = np.random.default_rng(seed)
        th0 = np.where(rng.integers(0, 2, 16) == 1, np.float32(math.pi), np.float32(0.0)).astype(np.float32)
        o.set_spins(th0, 0)
        o.step(500)
        r = o.run_series(150000)
        th = o.spins()
        assert set(np.unique(th).tolist()) <= {0.0, float(np.float32(math.pi))}
        Es.append(r["E"])
        M2s.append(r["M2"])
    m, e = pooled(Es)
    assert abs(m - ex["E"]) <= NSIG * e
    m, e = pooled(M2s)
    assert abs(m - ex["M2"]) <= NSIG * e


def _metropolis_xy(dim, L, beta, nrep, nsweeps, discard, seed):
    """Checkerboard single-spin Metropolis for Eq. (3), nrep independent replicas vectorised in
    numpy.  Returns per-sweep E/N and M^2 arrays of shape (nsweeps, nrep)."""
    rng = np.random.default_rng(seed)
    N = L ** dim
    idx = np.arange(N)
    coords = [(idx // L ** k) % L for k in range(dim)]
    parity = sum(coords) % 2
    nbp = plus_neighbours(dim, L)
    nbm = [np.argsort(n) for n in nbp]                 # inverse permutation = minus neighbour
    nbrs = np.stack(nbp + nbm, axis=0)                 # (2 dim, N)
    sub = [np.nonzero(parity == c)[0] for c in (0, 1)]
    th = rng.uniform(0, 2 * math.pi, size=(nrep, N))
    E, M2 = [], []
    for sweep in range(discard + nsweeps):
        for s in sub:
            old = th[:, s]
            new = old + rng.uniform(-1.6, 1.6, size=old.shape)
            nb = th[:, nbrs[:, s]]                     # (nrep, 2 dim, |s|)
            dE = -(np.cos(new[:, None, :] - nb) - np.cos(old[:, None, :] - nb)).sum(axis=1)
            acc = rng.uniform(size=old.shape) < np.exp(-beta * dE)
            th[:, s] = np.where(acc, new, old)
        if sweep >= discard:
            e = -sum(np.cos(th - th[:, n]).sum(axis=1) for n in nbp)
            E.append(e / N)
            M2.append(np.cos(th).sum(axis=1) ** 2 + np.sin(th).sum(axis=1) ** 2)
    return np.array(E), np.array(M2)


@pytest.mark.parametrize("dim,L,T", [(3, 4, 2.2019), (2, 6, 1.0)])
def test_xy_matches_independent_metropolis(dim, L, T):
    """R3.  Replica means of the Metropolis run are independent samples (error from their spread);
    the SW run uses binned errors.  SURVEY.md S6 quotes, for 4^3 at T = 2.2019,
    E/N = -1.21348(28), <M^2> = 1222.5(5), U = 1.2116(4) (soft, 'computed here')."""
    N = L ** dim
    Em, M2m = _metropolis_xy(dim, L, 1.0 / T, nrep=192, nsweeps=2500, discard=400, seed=7)
    e_met, e_met_err = Em.mean(), Em.mean(axis=0).std(ddof=1) / math.sqrt(Em.shape[1])
    m_met, m_met_err = M2m.mean(), M2m.mean(axis=0).std(ddof=1) / math.sqrt(M2m.shape[1])
    runs = []
    for seed in (1, 2, 3, 4):
        o = so.Oracle(dim, L, so.XY, 0, 1.0 / T, seed)
        o.step(500)
        runs.append(o.run_series(60000))
    e_sw, e_sw_err = pooled([r["E"] / N for r in runs])
    m_sw, m_sw_err = pooled([r["M2"] for r in runs])
    assert abs(e_sw - e_met) <= NSIG * math.hypot(e_sw_err, e_met_err)
    assert abs(m_sw - m_met) <= NSIG * math.hypot(m_sw_err, m_met_err)
    # F3: improved estimator from the cluster projections (sum_nc2 holds sum_c (sum a_i)^2 for XY)
    c_sw, c_sw_err = pooled([2.0 * r["sum_nc2"] for r in runs])
    assert abs(c_sw - m_sw) <= NSIG * math.hypot(c_sw_err, m_sw_err)
    if (dim, L) == (3, 4):
        assert e_sw == pytest.approx(-1.21348, abs=0.002)
        assert m_sw == pytest.approx(1222.5, abs=6.0)
        u = np.mean([np.mean(r["M2"] ** 2) for r in runs]) / m_sw ** 2
        assert u == pytest.approx(1.2116, abs=0.004)


def test_xy_high_temperature_series():
    """Soft closed-form check: for small beta, <cos(theta_i - theta_j)> = I1(beta)/I0(beta) + O(beta^3)
    corrections of relative size 2(d-1) t^2; at beta = 0.1 (d = 2) the correction is 0.5 %."""
    from scipy.special import i0, i1
    beta, L = 0.1, 12
    t = i1(beta) / i0(beta)
    o = so.Oracle(2, L, so.XY, 0, beta, 5)
    o.step(200)
    r = o.run_series(20000)
    m, e = binned_mean_err(-r["E"] / (2 * L * L))
    assert abs(m - (t + 2 * t ** 3)) <= NSIG * e + 1e-4
