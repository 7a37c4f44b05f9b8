"""Pins of the oracle's per-clone noise variant (DESIGN.md R-clone).

PAPER.md L87 uses one random number per word; the variant gives every clone its own 7-bit number
U and flips a k = 1 spin iff U < m (w1 = m / 128).  Pinned by what does not depend on the oracle:

* m = 0 and m = 128 need no randomness: they must equal the shared-noise rule with w1 = 0 and
  w1 = 1 (already pinned elsewhere) -- catches a wrong order, a wrong k, a dropped k >= 2 rule;
* C oracle == independent pure-Python restatement -- catches counter slots, word assembly, bit order;
* the accepted fraction of k = 1 moves is m / 128 within binomial error, and the decisions of two
  clones of the same word are uncorrelated (the shared-noise rule has correlation 1) -- catches a
  comparator that is off by one or that reuses bits between clones.
"""
from __future__ import annotations

import numpy as np

from oracle import xs_oracle_py as py
from oracle.xs_oracle import Instance

TWO32 = 1 << 32


def test_m0_and_m128_reduce_to_the_shared_noise_rule_without_randomness():
    inst = Instance(48, 5)
    for m, w1 in ((0, 0), (128, TWO32)):
        a = inst.init_spins(2, 9)
        b = a.copy()
        for t in range(1, 25):
            inst.sweep_clone(a, 9, t, m)
            inst.sweep(b, 9, t, thr4=[0, w1, TWO32, TWO32])
        assert np.array_equal(a, b)


def test_c_oracle_equals_python_restatement():
    for N, gseed, rseed, m in [(12, 2, 5, 7), (17, 3, 8, 40), (9, 4, 1, 1)]:
        inst = Instance(N, gseed)
        s_c = inst.init_spins(1, rseed)
        tri = [tuple(int(v) for v in t) for t in inst.tri]
        adj = py.clauses_of(N, tri)
        J = [1 - 2 * int(j) for j in inst.jbit]
        order, _ = py.update_order(N, adj)
        s_p = py.init_spins(N, 1, rseed)
        for t in range(1, 7):
            inst.sweep_clone(s_c, rseed, t, m)
            py.sweep_clone(N, 1, adj, J, order, rseed, t, m, s_p)
        assert np.array_equal(s_c, np.array(s_p, dtype=np.int8))


def _k_of(inst, s1, i):
    J = 1 - 2 * inst.jbit.astype(np.int64)
    k = 0
    for r in range(3):
        a, b = inst.nbr[i, 2 * r], inst.nbr[i, 2 * r + 1]
        k += int(J[inst.cls[i, r]] * s1[i] * s1[a] * s1[b] == -1)
    return k


def test_k1_acceptance_rate_and_independence_between_clones():
    """Decisions are read off single-spin updates: before every sweep the k of the FIRST spin of
    the order is computed for every clone (its neighbours have not moved yet in this sweep); the
    clones with k = 1 flipped that spin iff U < m."""
    N, W, m = 30, 4, 7
    inst = Instance(N, 11)
    s = inst.init_spins(W, 3)
    i0 = int(inst.order[0])
    n1 = acc = 0
    pair_both = pair_n = 0
    pair_a = pair_b = 0
    for t in range(1, 400):
        k_before = np.array([_k_of(inst, s[c], i0) for c in range(64 * W)])
        before = s[:, i0].copy()
        inst.sweep_clone(s, 3, t, m)
        # i0 is updated first; later updates of the sweep touch other spins only
        flipped = s[:, i0] != before
        sel = k_before == 1
        n1 += int(sel.sum())
        acc += int((flipped & sel).sum())
        # pairs of clones (2j, 2j+1) of the same word that both had k = 1
        both = sel[0::2] & sel[1::2]
        pair_n += int(both.sum())
        pair_a += int((flipped[0::2] & both).sum())
        pair_b += int((flipped[1::2] & both).sum())
        pair_both += int((flipped[0::2] & flipped[1::2] & both).sum())
    p = m / 128.0
    assert n1 > 10000
    assert abs(acc / n1 - p) < 5 * np.sqrt(p * (1 - p) / n1)          # 5 sigma
    # independence: P(both) = p^2 (shared noise would give P(both) = p)
    assert pair_n > 1500
    assert abs(pair_both / pair_n - p * p) < 5 * np.sqrt(p * p * (1 - p * p) / pair_n) + 1e-3
    assert pair_both / pair_n < 0.5 * p
