"""Pins of the oracle's general flip table w_0..w_3.

* the quasi-greedy table through the general path is the rule the other pins test;
* C oracle == independent pure-Python restatement for arbitrary tables;
* "by setting w0 = w1^3 we would have an algorithm satisfying detailed balance":
  with w_k = min(1, exp(-(6 - 4k)/T)) the sequential sweep leaves the Boltzmann law of
  H = -sum J s s s invariant, so the energy histogram of many clones after a burn-in must equal
  the exact one obtained by enumerating all 2^N states (a wrong k <-> threshold assignment, a wrong
  sign of Delta E or a biased compare all fail this).
"""
from __future__ import annotations

import math

import numpy as np

from oracle import xs_oracle_py as py
from oracle.xs_oracle import W1_THRESHOLD, Instance

TWO32 = 1 << 32


def metropolis_table(T: float):
    """thr4[k] = min(1, exp(-dE_k / T)) 2^32 with dE_k = 6 - 4k (L67: k -> energy change)."""
    return [min(TWO32, int(math.floor(min(1.0, math.exp(-(6 - 4 * k) / T)) * TWO32))) for k in range(4)]


def test_metropolis_table_satisfies_w0_equals_w1_cubed():
    T = -2.0 / math.log(0.055)                      # L101: T_run = 0.69
    t4 = metropolis_table(T)
    w = [t / TWO32 for t in t4]
    assert abs(w[1] - 0.055) < 1e-9 and abs(w[0] - w[1] ** 3) < 1e-9 and w[2] == w[3] == 1.0


def test_qg_table_through_general_path_equals_qg_rule():
    inst = Instance(40, 9)
    a = inst.init_spins(2, 4)
    b = a.copy()
    qg = [0, W1_THRESHOLD, TWO32, TWO32]
    for t in range(1, 30):
        inst.sweep(a, 4, t)
        inst.sweep(b, 4, t, thr4=qg)
    assert np.array_equal(a, b)


def test_c_oracle_equals_python_restatement_for_general_tables():
    rng = np.random.default_rng(3)
    for N, gseed, rseed in [(12, 2, 5), (17, 3, 8)]:
        inst = Instance(N, gseed)
        t4 = [int(v) for v in rng.integers(0, TWO32 + 1, 4)]
        t4[rng.integers(0, 4)] = TWO32                                  # include an "always"
        s_c = inst.init_spins(1, rseed)
        tri = [tuple(int(v) for v in t) for t in inst.tri]
        adj = py.clauses_of(N, tri)
        J = [1 - 2 * int(j) for j in inst.jbit]
        order, _ = py.update_order(N, adj)
        s_p = py.init_spins(N, 1, rseed)
        for t in range(1, 9):
            inst.sweep(s_c, rseed, t, thr4=t4)
            py.sweep_table(N, 1, adj, J, order, rseed, t, t4, s_p)
        assert np.array_equal(s_c, np.array(s_p, dtype=np.int8))


def test_detailed_balance_table_reproduces_boltzmann_energy_law():
    N, T = 10, 1.1
    inst = Instance(N, 21)
    # exact Boltzmann law by enumeration
    states = ((np.arange(1 << N)[:, None] >> np.arange(N)) & 1).astype(np.int8)
    spins = (1 - 2 * states).astype(np.int8)
    E = inst.energy(spins)
    levels = np.unique(E)
    wgt = np.exp(-E / T)
    exact = np.array([wgt[E == e].sum() for e in levels]) / wgt.sum()
    # sampled law: 128 words (the 64 clones of a word share their noise, so a word is roughly one
    # independent sample), burn-in 60 sweeps, then every 5th sweep: ~15,000 weakly correlated samples, sigma ~ 0.005;
    # a swapped threshold or a wrong sign of Delta E moves the law by 0.1 or more
    W = 128
    s = inst.init_spins(W, 77)
    t4 = metropolis_table(T)
    counts = np.zeros(len(levels))
    t = 0
    for _ in range(60):
        t += 1
        inst.sweep(s, 77, t, thr4=t4)
    for _ in range(120):
        for _ in range(5):
            t += 1
            inst.sweep(s, 77, t, thr4=t4)
        e = inst.energy(s)
        counts += np.array([(e == lv).sum() for lv in levels])
    sampled = counts / counts.sum()
    assert np.abs(sampled - exact).max() < 0.02, (sampled, exact)
    # the quasi-greedy table breaks detailed balance (L69) and gives a different law
    s2 = inst.init_spins(W, 77)
    for t in range(1, 200):
        inst.sweep(s2, 77, t)
    e2 = inst.energy(s2)
    qg = np.array([(e2 == lv).mean() for lv in levels])
    assert np.abs(qg - exact).max() > 0.05          # the test can tell the two tables apart
