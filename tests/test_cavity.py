"""the cavity free-energy barrier (Eqs. (3)-(4), L169-L208) against
the two numbers the paper prints (tests/golden/cavity_paper_values.txt) and against what the
equations fix by themselves.  Host only: no kernel is launched."""
from __future__ import annotations

import math
import os

import pytest

import paper_2102_09510_b200 as xs

GOLD = os.path.join(os.path.dirname(__file__), "golden", "cavity_paper_values.txt")


def _gold():
    d = {}
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split(None, 1)
            d[k] = v.strip()
    return d


def test_paper_values_T_sp_and_barrier_at_T_run():
    g = _gold()
    K, w1 = int(g["K"]), float(g["w1"])
    T_run = -2.0 / math.log(w1)                              # L169
    r = xs.xs_cavity_barrier(K, T_run)
    assert r["T_sp"] == pytest.approx(float(g["T_sp"]), abs=5e-7)              # six printed decimals
    assert r["barrier"] == pytest.approx(float(g["barrier_at_T_run"]), abs=5e-8)
    # "a very good approximation to the actual rate" (L208): within 6 % of the fitted exponent
    assert abs(r["barrier"] / float(g["fitted_exponent"]) - 1.0) < 0.06
    assert 0.0 < r["m_barrier"] < r["m_ferro"] < 1.0


def test_structure_fixed_by_the_equations():
    # L202: "the ferromagnetic state has always a higher free-energy than the paramagnetic state"
    for T in (0.55, 0.7, 0.9, 0.97):
        r = xs.xs_cavity_barrier(3, T)
        assert r["ferro_bdf"] > 0.0 and r["barrier"] > r["ferro_bdf"]
    # the barrier vanishes at the spinodal: barrier top and ferromagnetic state merge
    r = xs.xs_cavity_barrier(3, 0.9805)
    assert r["barrier"] - r["ferro_bdf"] < 1e-5 and r["m_ferro"] - r["m_barrier"] < 0.05
    # above T_sp there is no ferromagnetic solution
    r = xs.xs_cavity_barrier(3, 1.0)
    assert math.isnan(r["barrier"]) and r["T_sp"] == pytest.approx(0.980548, abs=5e-7)
    # L208 / Fig. 7: "in principle a purely thermal algorithm could be even faster": beta * barrier
    # decreases on cooling below T_run
    b = [xs.xs_cavity_barrier(3, T)["barrier"] for T in (0.95, 0.85, 0.75, 0.65, 0.55)]
    assert all(x > y for x, y in zip(b, b[1:]))
    # argument errors
    for bad in ((2, 0.7), (3, 0.0), (3, -1.0)):
        with pytest.raises(xs.XsError):
            xs.xs_cavity_barrier(*bad)


def test_barrier_point_is_a_stationary_point_without_field():
    """max_m Delta f is reached where the conjugate field b vanishes: h = (K-1) u (Eq. (4) with b = 0)."""
    for K, T in ((3, 0.6896), (3, 0.8), (4, 0.9)):
        r = xs.xs_cavity_barrier(K, T)
        beta, h = 1.0 / T, r["h_barrier"]
        u = math.atanh(math.tanh(beta) * math.tanh(beta * h) ** (K - 1)) / beta
        assert abs(h - (K - 1) * u) < 1e-6
        assert r["m_barrier"] == pytest.approx(math.tanh(beta * (u + h)), abs=1e-9)
