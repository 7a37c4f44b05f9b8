"""CPU-side checks of the product library: it loads, exports every symbol include/xs.h declares,
its host generator agrees byte for byte with the (independently written) oracle generator, its
TTS statistics match closed forms / scipy, and argument errors come back as codes.
No kernel is launched here."""
from __future__ import annotations

import ctypes as C
import math
import os
import re

import numpy as np
import pytest

import paper_2102_09510_b200 as xs
from oracle.xs_oracle import Instance

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "xs.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(xs_[a-z_0-9]+)\s*\(", hdr))
    assert {"xs_create_instance", "xs_run_sweeps", "xs_energy", "xs_tts"} <= declared
    L = xs.lib()
    for name in sorted(declared):
        assert hasattr(L, name), f"libxs_b200.so does not export {name}"
    from paper_2102_09510_b200 import _binding
    assert declared == set(_binding.EXPORTS)


@pytest.mark.parametrize("N,seed,cap,gauge", [(64, 1, 0, True), (256, 2, 0, True), (512, 100, 0, True),
                                              (512, 101, 32, True), (20, 7, 0, False), (999, 5, 3, True),
                                              (3, 1, 0, True), (4096, 9, 0, True)])
def test_generator_matches_oracle_generator(N, seed, cap, gauge):
    tri, jbit, order, ss, att = xs.xs_generate_graph(N, seed, xs.XS_FLAG_GAUGE if gauge else 0, cap)
    o = Instance(N, seed, gauge, cap)
    assert att == o.attempt
    assert np.array_equal(tri, o.tri)
    assert np.array_equal(jbit, o.jbit)
    assert np.array_equal(order, o.order)
    assert np.array_equal(ss, o.set_size)
    assert o.check_order(order, ss)


@pytest.mark.parametrize("N,seed,cap", [(256, 2, 64), (128, 100, 0), (64, 5, 16), (512, 101, 64),
                                        (20, 3, 0), (100, 4, 32), (6, 1, 0), (3, 1, 0), (192, 7, 0), (384, 8, 0),
                                        (768, 9, 0), (1024, 10, 0), (320, 11, 0)])
def test_balanced_sets_match_oracle(N, seed, cap):
    """XS_FLAG_BALANCED (DESIGN.md R-balance): the library's tabu search and the oracle's are
    written independently and must produce the same order; it is checked for validity by the
    oracle (anti-cliques, permutation)."""
    tri, jbit, order, ss, att = xs.xs_generate_graph(N, seed, xs.XS_FLAG_GAUGE | xs.XS_FLAG_BALANCED, cap)
    o = Instance(N, seed, gauge=True, set_cap=cap, balanced=True)
    assert np.array_equal(order, o.order)
    assert np.array_equal(ss, o.set_size)
    assert o.check_order(order, ss)
    # the same two properties straight from the triplets (L277): permutation, and the three spins
    # of every triplet lie in three different sets
    assert sorted(order.tolist()) == list(range(N))
    set_of = np.empty(N, dtype=np.int64)
    set_of[order] = np.repeat(np.arange(len(ss)), ss)
    st = set_of[tri.astype(np.int64)]
    assert (st[:, 0] != st[:, 1]).all() and (st[:, 1] != st[:, 2]).all() and (st[:, 0] != st[:, 2]).all()
    if o.balanced:
        S = cap
        if S == 0:                                   # default: largest power of two in 16..256 below N/4
            S = max([v for v in (16, 32, 64, 128, 256) if v <= N // 4] or [16])
        q = max(4, -(-N // S))
        assert len(ss) == q and int(ss.max()) - int(ss.min()) <= 1 and int(ss.max()) == -(-N // q)
    else:       # no proper q-colouring found (tiny N): the greedy order
        g = Instance(N, seed, gauge=True, set_cap=cap)
        assert np.array_equal(order, g.order)


@pytest.mark.parametrize("N,seed,n_slots,balanced,cap", [
    (256, 2, 64, True, 0), (128, 100, 32, True, 0), (512, 101, 128, True, 0), (512, 355, 128, True, 0),
    (192, 7, 32, True, 0), (384, 8, 64, True, 0), (768, 9, 128, True, 0), (128, 128004, 32, True, 0),
    (1024, 1024000, 128, True, 0),     # 4 sets of 256 on 128 slots: 8 rounds, barrier after every second
    (160, 3, 32, True, 0), (224, 4, 32, True, 0), (320, 5, 64, True, 0),     # 5 / 7 / 5 sets
    (256, 2, 64, False, 0), (512, 100, 128, False, 0), (128, 9, 32, False, 0),  # greedy, ragged sets
    (100, 6, 32, True, 25), (200, 11, 64, False, 0),
    (256, 2, 32, False, 32), (192, 5, 32, False, 32)])    # the paper's cap-32 sets (L279): 10+ rounds
def test_clause_placement_is_conflict_free_and_complete(N, seed, n_slots, balanced, cap):
    """Placement tables of the clause-word kernel (include/xs.h), checked straight
    from the triplets: the entries of a set's rounds are exactly the set's spins (L277: any order
    inside a set is valid), an entry's three rows are the three interactions the spin enters (L67),
    idle slots stay on their scratch line, and the two slots of a shared-memory phase touch
    opposite halves of their 128-byte lines."""
    fl = xs.XS_FLAG_GAUGE | (xs.XS_FLAG_BALANCED if balanced else 0)
    tri, jbit, order, ss, att = xs.xs_generate_graph(N, seed, fl, cap)
    task, place, bar = xs.xs_clause_placement(N, seed, n_slots, fl, cap)
    n_rounds = len(task) // n_slots
    assert 4 <= n_rounds <= 16 and n_rounds * n_slots <= 2 * N
    t = np.arange(N, dtype=np.uint32)
    assert np.array_equal(place & ~np.uint32(64), t << 7)                 # own line, lower or upper half
    clauses_of = [[] for _ in range(N)]
    for c, (i, j, k) in enumerate(tri.tolist()):
        for v in (i, j, k):
            clauses_of[v].append(c)
    IDLE = 0xFFFFFFFF
    raw = task.copy()
    last_bits = np.where(task[:, 3] != IDLE, (task[:, 3] >> 16) & 7, 0)
    task[:, 3] = np.where(task[:, 3] != IDLE, task[:, 3] & 0xFFFF, IDLE)     # bits 16-18: last-touch mask
    r0, p0, want_bar = 0, 0, 0
    for sz in ss.tolist():
        nr = -(-sz // n_slots)
        ent = task[r0 * n_slots:(r0 + nr) * n_slots]
        spins = ent[ent[:, 3] != IDLE, 3]
        assert sorted(spins.tolist()) == sorted(order[p0:p0 + sz].tolist())
        r0, p0 = r0 + nr, p0 + sz
        want_bar |= 1 << (r0 - 1)
    assert bar == want_bar
    assert (task[r0 * n_slots:, 3] == IDLE).all()                         # padding rounds are idle
    for e_i, e in enumerate(task):
        if e[3] != IDLE:
            assert sorted((e[:3] >> 7).tolist()) == sorted(clauses_of[int(e[3])])
            assert np.array_equal(e[:3], place[e[:3] >> 7])
        else:
            assert ((e[:3] >> 7) == N + (e_i % n_slots) // 2).all()       # scratch line of the slot pair
    half = (task[:, :3] >> 6) & 1
    assert ((half[0::2] ^ half[1::2]) == 1).all()
    # last-touch mask: bit k of an entry <=> no later round of the sweep touches its clause k
    round_of = {int(e[3]): i // n_slots for i, e in enumerate(task) if e[3] != IDLE}
    for i, e in enumerate(task):
        if e[3] == IDLE:
            continue
        for k in range(3):
            members = tri[int(e[k]) >> 7].tolist()
            is_last = max(round_of[m] for m in members) == i // n_slots
            assert ((int(last_bits[i]) >> k) & 1) == int(is_last)
    if balanced and cap == 0 and N % (n_slots * 4) == 0 and len(ss) * n_slots == N:
        assert (task[:, 3] != IDLE).all()                                 # full sets: no idle slot
    # deterministic
    task2, place2, bar2 = xs.xs_clause_placement(N, seed, n_slots, fl, cap)
    assert np.array_equal(raw, task2) and np.array_equal(place, place2) and bar == bar2


def test_clause_placement_rejects_orders_that_do_not_fit():
    with pytest.raises(xs.XsError):                     # sets of 64 on 8 slots: 32 rounds
        xs.xs_clause_placement(256, 2, 8)
    with pytest.raises(xs.XsError):                     # cap-32 order: 17+ sets
        xs.xs_clause_placement(512, 2, 32, xs.XS_FLAG_GAUGE, 32)
    with pytest.raises(xs.XsError):                     # odd slot count
        xs.xs_clause_placement(256, 2, 63)


def test_workspace_bytes_and_param_errors():
    p = xs.make_params(256, 1024, 1)
    n = xs.xs_workspace_bytes(p)
    assert n >= 256 * 1024 * 8 + 65536 * 4
    for bad in [xs.make_params(2, 1, 1), xs.make_params(64, 0, 1), xs.make_params(64, 1, 0)]:
        with pytest.raises(xs.XsError) as ei:
            xs.xs_workspace_bytes(bad)
        assert ei.value.code == -1
    L = xs.lib()
    assert L.xs_run_sweeps(None, 1, None) == -1
    assert b"null" in L.xs_last_error()
    assert L.xs_destroy(None) == 0


def test_tts_stats_closed_forms():
    """L113 Eq.(2), L117/L123: TTS_p = -ln(1-p/100) tau; L145 posterior = inverse-gamma(n, T_tot)."""
    scipy_stats = pytest.importorskip("scipy.stats")
    rng = np.random.default_rng(0)
    tts = rng.exponential(5000.0, 400).astype(np.uint32) + 1
    s = xs.xs_tts_stats(tts, 0)
    assert s["n_solved"] == 400 and s["t_tot"] == float(tts.sum())
    assert s["tau_hat"] == pytest.approx(tts.mean(), rel=1e-12)
    for p, key in [(0.5, "tts50_model"), (0.9, "tts90_model"), (0.99, "tts99_model")]:
        assert s[key] == pytest.approx(-math.log(1 - p) * tts.mean(), rel=1e-12)
    srt = np.sort(tts)
    assert s["tts50_emp"] == srt[199] and s["tts90_emp"] == srt[359] and s["tts99_emp"] == srt[395]
    # with a timeout: censored runs count t_max each
    t_max = 3000
    cens = np.where(tts <= t_max, tts, xs.XS_NO_HIT).astype(np.uint32)
    c = xs.xs_tts_stats(cens, t_max)
    n = int((tts <= t_max).sum())
    t_tot = float(tts[tts <= t_max].sum() + (400 - n) * t_max)
    assert c["n_solved"] == n and c["t_tot"] == t_tot
    assert c["tau_hat"] == pytest.approx(t_tot / n)
    ig = scipy_stats.invgamma(a=n, scale=t_tot)
    assert c["tau_q16"] == pytest.approx(ig.ppf(0.16), rel=1e-6)
    assert c["tau_q50"] == pytest.approx(ig.ppf(0.50), rel=1e-6)
    assert c["tau_q84"] == pytest.approx(ig.ppf(0.84), rel=1e-6)
    assert math.isinf(c["tts99_emp"])
    # the censored estimate recovers the true scale within its own error bar
    assert c["tau_q16"] < 5000.0 * 1.15 and c["tau_q84"] > 5000.0 * 0.85
    # nothing solved: only a lower bound
    z = xs.xs_tts_stats(np.full(10, xs.XS_NO_HIT, np.uint32), 1000)
    assert z["n_solved"] == 0 and math.isinf(z["tau_hat"])
    assert z["tau_q16"] == pytest.approx(10 * 1000 / math.log(20.0))
    # n = 1: inverse-gamma(1, T): median = T / ln 2
    # no cap given (t_max = 0) but a run is censored: no censoring time -> refused, not biased low
    with pytest.raises(xs.XsError) as ei:
        xs.xs_tts_stats(np.array([10, xs.XS_NO_HIT, 30], np.uint32), 0)
    assert ei.value.code == -1
    one = xs.xs_tts_stats(np.array([700], np.uint32), 0)
    assert one["tau_q50"] == pytest.approx(700 / math.log(2.0), rel=1e-9)


def test_no_cpu_fallback_without_gpu():
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        xs.Batch(64, 1, [1], [1])
