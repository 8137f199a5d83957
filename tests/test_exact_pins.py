"""Pins for the exact-result module tests/exact.py itself (CPU only).

The oracle is tested against exact.py; exact.py is tested here against (a) the values SURVEY.md
section 8(c) S6 prints (tests/golden/*.txt) and (b) itself across three independent routes:
spin-state enumeration, FK bond-set enumeration, and Kaufman's closed formula.
"""
import math
import os

import pytest

import exact
from stats import golden_rows

GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.mark.parametrize("row", golden_rows(os.path.join(GOLD, "exact_small_lattices.txt")),
                         ids=lambda r: "-".join(r[:1] + r[4:6]))
def test_enumeration_matches_printed_values(row):
    name, dim, L, q, T, quantity, value = row
    dim, L, q, T, value = int(dim), int(L), int(q), float(T), float(value)
    r = exact.exact_ising(dim, L, T) if name.startswith("ising") else exact.exact_potts(dim, L, q, T)
    assert r[quantity] == pytest.approx(value, rel=1e-9)


@pytest.mark.parametrize("row", golden_rows(os.path.join(GOLD, "kaufman_energy.txt")),
                         ids=lambda r: "L%s-T%s" % (r[0], r[1]))
def test_kaufman_matches_printed_values(row):
    L, T, e, c = int(row[0]), float(row[1]), float(row[2]), float(row[3])
    e_k, c_k = exact.kaufman_energy_per_site(L, T)
    assert e_k == pytest.approx(e, rel=1e-9)
    if not math.isnan(c):
        assert c_k == pytest.approx(c, rel=1e-8)


@pytest.mark.parametrize("L,T", [(3, 2.269185), (4, 2.269185), (4, 2.0), (4, 3.0)])
def test_kaufman_equals_enumeration(L, T):
    r = exact.exact_ising(2, L, T)
    e_k, c_k = exact.kaufman_energy_per_site(L, T)
    assert e_k * L * L == pytest.approx(r["E"], rel=1e-10)
    assert c_k * L * L == pytest.approx((r["E2"] - r["E"] ** 2) / T ** 2, rel=1e-8)


def test_kaufman_tends_to_onsager():
    """Onsager: E/N = -sqrt(2) at T_c = 2/ln(1+sqrt 2) for L -> infinity; finite-L shift ~ 1/L."""
    Tc = 2.0 / math.log(1.0 + math.sqrt(2.0))
    d = [exact.kaufman_energy_per_site(L, Tc)[0] + math.sqrt(2.0) for L in (32, 64, 128)]
    assert all(x < 0 for x in d)
    assert d[0] / d[1] == pytest.approx(2.0, rel=0.02) and d[1] / d[2] == pytest.approx(2.0, rel=0.02)


def test_fk_enumeration_equals_spin_enumeration_3x3():
    """FK identities: <#active> = p <#equal>, <sum_c n_c^2> = <M^2> (Ising and Potts Eq. 5)."""
    T = 2.269185
    p = -math.expm1(-2.0 / T)
    s, fk = exact.exact_ising(2, 3, T), exact.exact_fk(2, 3, 2, p)
    assert fk["n_active"] == pytest.approx(p * s["n_equal"], rel=1e-10)
    assert fk["sum_nc2"] == pytest.approx(s["M2"], rel=1e-10)
    assert fk["n_clusters"] == pytest.approx(1.8755802082, rel=1e-9)     # SURVEY.md S6 pin P3
    T = 0.994973
    p = -math.expm1(-1.0 / T)
    s, fk = exact.exact_potts(2, 3, 3, T), exact.exact_fk(2, 3, 3, p)
    assert fk["n_active"] == pytest.approx(p * s["n_equal"], rel=1e-10)
    assert fk["sum_nc2"] == pytest.approx(s["M2"], rel=1e-10)
    assert fk["n_active"] == pytest.approx(9.94014932185, rel=1e-9)      # SURVEY.md S6 pin P2
    assert fk["n_clusters"] == pytest.approx(1.8955740954, rel=1e-9)
    assert fk["var_clusters"] == pytest.approx(1.3824481119, rel=1e-8)


def test_potts_q2_equals_ising_3x3():
    """Pin P4: Potts q=2 at T/2 has the Ising M^2 (Eq. 5 at q=2 is (n1-n2)^2)."""
    a = exact.exact_ising(2, 3, 2.269185)
    b = exact.exact_potts(2, 3, 2, 2.269185 / 2)
    assert b["M2"] == pytest.approx(a["M2"], rel=1e-12)
    assert b["n_equal"] == pytest.approx(a["n_equal"], rel=1e-12)
