"""Statistical pins of the oracle's Markov chain against exact results (CPU only).

The oracle samples the Boltzmann distribution iff bond probabilities, labelling and the per-cluster
draw are all right; a dropped factor 2 in beta, a missed wrap bond, a biased draw or a correlated
random stream each shift at least one of these averages by many sigma.  Exact values come from
tests/exact.py (brute-force enumeration / Kaufman's formula, themselves pinned in
test_exact_pins.py to the numbers SURVEY.md section 8(c) S6 prints).  Fixed seeds, 4 independent
runs as in the paper; pass = |mean - exact| <= 3 sigma of the pooled binned error
(north_star's tolerance; fixed seeds, none is re-tuned).
"""
import math

import numpy as np
import pytest

import exact
from oracle import sw_oracle as so
from stats import pooled

SEEDS = (1, 2, 3, 4)
NSIG = 3.0


def _runs(dim, L, model, q, beta, nsteps, discard=1000):
    out = []
    for seed in SEEDS:
        o = so.Oracle(dim, L, model, q, beta, seed)
        o.step(discard)
        out.append(o.run_series(nsteps))
    return out


def _check(runs, key, exact_value, f=lambda x: x):
    m, e = pooled([f(r[key]) for r in runs])
    assert e > 0
    assert abs(m - exact_value) <= NSIG * e, "%s: %.6f +- %.6f vs exact %.6f" % (key, m, e, exact_value)
    return m, e


@pytest.mark.parametrize("L,T", [(4, 2.269185), (4, 2.0), (4, 3.0), (3, 2.269185)])
def test_ising_small_lattice_matches_enumeration(L, T):
    """Pins P1, P1', P3: 4x4 and 3x3 Ising, <E>, <E^2>, <M^2>, <M^4>, <|M|> and the FK identities
    F1 (<#active> = p <#equal>) and F2 (<sum_c n_c^2> = <M^2>)."""
    ex = exact.exact_ising(2, L, T)
    runs = _runs(2, L, so.ISING, 0, 1.0 / T, 250000)
    p = -math.expm1(-2.0 / T)
    _check(runs, "E", ex["E"])
    _check(runs, "E", ex["E2"], lambda x: x * x)
    _check(runs, "M2", ex["M2"])
    _check(runs, "M2", ex["M4"], lambda x: x * x)
    _check(runs, "M", ex["absM"], np.abs)
    _check(runs, "M", 0.0)                                   # signed M: symmetric draw per cluster
    _check(runs, "n_active", p * ex["n_equal"])
    _check(runs, "sum_nc2", ex["M2"])
    if L == 3:
        fk = exact.exact_fk(2, 3, 2, p)
        _check(runs, "n_clusters", fk["n_clusters"])
        _check(runs, "n_clusters", fk["var_clusters"] + fk["n_clusters"] ** 2, lambda x: x * x)


@pytest.mark.parametrize("T", [0.994973, 0.8, 1.5])
def test_potts_3x3_q3_matches_enumeration(T):
    """Pins P2, P2': 3x3 q=3 Potts (Eq. 2 energy, Eq. 5 magnetisation) and FK cluster counts."""
    ex = exact.exact_potts(2, 3, 3, T)
    p = -math.expm1(-1.0 / T)
    fk = exact.exact_fk(2, 3, 3, p)
    runs = _runs(2, 3, so.POTTS, 3, 1.0 / T, 250000)
    _check(runs, "E", ex["E"])
    _check(runs, "E", ex["E2"], lambda x: x * x)
    _check(runs, "M2", ex["M2"])
    _check(runs, "M2", ex["M4"], lambda x: x * x)
    _check(runs, "n_active", fk["n_active"])
    _check(runs, "n_clusters", fk["n_clusters"])
    _check(runs, "sum_nc2", ex["M2"])


def test_ising_3d_small_matches_enumeration():
    """3D code path (third bond direction, z wrap).  3x3x3 has 2^27 states, too many to enumerate
    in a unit test, so 3D is pinned through the FK identities, which hold on any lattice and tie
    independent parts of the oracle together: F1 <#active> = p <#equal pairs> (bonds vs spins) and
    F2 <sum_c n_c^2> = <M^2> (labels vs spins)."""
    T = 4.5115
    runs = _runs(3, 4, so.ISING, 0, 1.0 / T, 100000)
    p = -math.expm1(-2.0 / T)
    nb = 3 * 64
    # n_active(t) is drawn from the configuration BEFORE step t, E(t) is measured AFTER it; in
    # equilibrium both averages are stationary, so compare the means.
    m_act, e_act = pooled([r["n_active"] for r in runs])
    m_eq, e_eq = pooled([(nb - r["E"]) / 2.0 for r in runs])
    assert abs(m_act - p * m_eq) <= NSIG * math.hypot(e_act, p * e_eq)
    m_a, e_a = pooled([r["sum_nc2"] for r in runs])
    m_b, e_b = pooled([r["M2"] for r in runs])
    assert abs(m_a - m_b) <= NSIG * math.hypot(e_a, e_b)


def test_ising_L64_matches_kaufman():
    """Pin P5 (finite-torus form of Onsager's -sqrt 2, P6): 2D Ising L = 64 at T = 2.269185,
    <E>/N = -1.42393907865393; config 1 of BASELINE.json."""
    e_exact, c_exact = exact.kaufman_energy_per_site(64, 2.269185)
    runs = _runs(2, 64, so.ISING, 0, 1.0 / 2.269185, 6000, discard=300)
    m, e = _check(runs, "E", e_exact * 4096)
    assert e / 4096 < 0.003                                   # resolves the finite-size shift 0.0097 from -sqrt(2)
    assert abs(m / 4096 + math.sqrt(2.0)) > 2.0 * e / 4096
    # specific heat from energy fluctuations, loose: 15 %
    var = np.mean([np.var(r["E"]) for r in runs])
    assert var / 2.269185 ** 2 / 4096 == pytest.approx(c_exact, rel=0.15)


def test_potts_2d_selfdual_bond_density():
    """Pin P7: at the self-dual point of the 2D q = 3 Potts model the active-bond density tends to
    1/2 and E/N (Eq. 2) to 2 (1 - (1 + 1/sqrt 3)/2) = 0.42265 as L grows.  Soft pin: the finite-size
    shift of the energy decays only like L^(1/nu - 2) = L^-0.8 (nu = 5/6), about -0.017 at L = 48
    (the periodic lattice is more ordered), so the tolerance is 0.03; the sign is checked too."""
    T = 1.0 / math.log(1.0 + math.sqrt(3.0))
    runs = _runs(2, 48, so.POTTS, 3, 1.0 / T, 3000, discard=300)
    m, e = pooled([r["n_active"] for r in runs])
    assert m / (2 * 48 * 48) == pytest.approx(0.5, abs=0.01)
    m, e = pooled([r["E"] for r in runs])
    e_inf = 2.0 * (1.0 - (1.0 + 1.0 / math.sqrt(3.0)) / 2.0)
    assert m / (48 * 48) == pytest.approx(e_inf, abs=0.03) and m / (48 * 48) < e_inf
