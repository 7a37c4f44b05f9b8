"""GPU parity for the general flip table w_0..w_3 (xs_set_flip_table; PAPER.md L67, L69;
SURVEY.md 8(f) NEXT-1): generic tile kernel and streaming kernel against the oracle, bit-exact,
including tables with w0 > 0 where a ground state can be left again (first hits then have to be
looked for after every sweep)."""
from __future__ import annotations

import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from _harness import OracleRun  # noqa: E402
from oracle.xs_oracle import NO_HIT  # noqa: E402

TWO32 = 1 << 32


@pytest.fixture(autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")


def metropolis(T):
    return [min(TWO32, int(math.floor(min(1.0, math.exp(-(6 - 4 * k) / T)) * TWO32))) for k in range(4)]


def _check(b, o, what):
    assert np.array_equal(b.spins_numpy()[0], o.x()), f"{what}: spins"
    assert np.array_equal(b.first_hit_numpy()[0], o.first_hit), f"{what}: first hits"
    assert np.array_equal(b.energy().cpu().numpy()[0], o.energy()), f"{what}: energies"
    r = b.tts()[0]
    assert (r.solved, r.tts_sweeps, r.clone) == o.tts() and r.sweeps_done == o.sweeps_done, what


TABLES = {
    "metropolis_T0.69": metropolis(-2.0 / math.log(0.055)),      # w0 = w1^3 (L69)
    "metropolis_T2": metropolis(2.0),
    "arbitrary": [123456789, 3000000000, TWO32, 17],
    "greedy_w1_1": [0, TWO32, TWO32, TWO32],                      # w1 = 1: not the QG form
}


@pytest.mark.parametrize("name", sorted(TABLES))
@pytest.mark.parametrize("N,W,streaming", [(40, 2, False), (90, 16, False), (60, 8, True), (33, 5, True)])
def test_flip_table_parity(name, N, W, streaming):
    import paper_2102_09510_b200 as xs
    t4 = TABLES[name]
    flags = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | (xs.XS_FLAG_STREAMING if streaming else 0)
    b = xs.Batch(N, W, [N + 1], [N + 2], flags=flags)
    b.set_flip_table(t4)
    lay = b.layout()
    assert lay.regime == int(streaming) and (streaming or lay.variant == 0)
    o = OracleRun(N, W, N + 1, N + 2, no_skip=True, thr4=t4)
    for n in (1, 9, 23):
        b.run_sweeps(n)
        o.run_sweeps(n)
        _check(b, o, f"{name} N={N} W={W} streaming={streaming}")
    b.close()


@pytest.mark.parametrize("streaming", [False, True])
def test_first_hits_with_w0_positive_small_system(streaming):
    """N = 14 at T = 1.5: clones enter and leave ground states all the time."""
    import paper_2102_09510_b200 as xs
    N, W, t4 = 14, 4, metropolis(1.5)
    flags = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | (xs.XS_FLAG_STREAMING if streaming else 0)
    b = xs.Batch(N, W, [3], [4], flags=flags, geometry=dict(batch_sweeps=7))
    b.set_flip_table(t4)
    o = OracleRun(N, W, 3, 4, no_skip=True, thr4=t4)
    for n in (5, 20, 11):
        b.run_sweeps(n)
        o.run_sweeps(n)
        _check(b, o, f"w0>0 streaming={streaming}")
    assert (o.first_hit != NO_HIT).sum() > 30
    # some clone that has a first hit is no longer in a ground state: the table is not absorbing
    assert (o.energy()[o.first_hit != NO_HIT] > -N).any()
    b.close()


def test_back_to_quasi_greedy_table_uses_fast_kernel():
    import paper_2102_09510_b200 as xs
    N, W = 64, 8
    b = xs.Batch(N, W, [5], [6], flags=xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP)
    fast = b.layout().variant
    assert fast in (1, 2)
    b.set_flip_table(metropolis(1.0))
    assert b.layout().variant == 0
    b.set_flip_table([0, 200000000, TWO32, TWO32])       # quasi-greedy form with another w1
    assert b.layout().variant == fast
    o = OracleRun(N, W, 5, 6, no_skip=True, thr=200000000)
    b.run_sweeps(30)
    o.run_sweeps(30)
    _check(b, o, "qg with another w1")
    with pytest.raises(xs.XsError):
        b.set_flip_table([0, 1, 2, TWO32 + 1])
    b.close()


@pytest.mark.parametrize("N,W,I,T", [(128, 8, 1, 0.69), (128, 16, 3, 1.2), (192, 8, 2, 0.69), (256, 8, 1, 2.0), (512, 8, 1, 0.9)])
def test_w0_family_on_the_clause_word_kernel(N, W, I, T):
    """SURVEY.md 8(f) NEXT-1 on the fast kernel: tables (w0, w1, 1, 1) with 0 < w0 <= w1 (L69: Metropolis,
    w0 = w1^3) run on the clause-word kernel when the balanced sets fill the CTA; ground states are not
    absorbing, so the kernel looks for first hits after every sweep (OR of the clause words at their last
    touch).  Clones start a few flips away from the planted state so that they enter and leave E = -N."""
    import paper_2102_09510_b200 as xs
    t4 = metropolis(T)
    assert 0 < t4[0] <= t4[1] < TWO32 and t4[2] == t4[3] == TWO32
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_BALANCED
    gs, rs = [N + 40 + i for i in range(I)], [3 * N + i for i in range(I)]
    b = xs.Batch(N, W, gs, rs, flags=fl, geometry=dict(batch_sweeps=16))
    b.set_flip_table(t4)
    lay = b.layout()
    assert (lay.regime, lay.variant, lay.tile_words) == (0, 2, 8), (lay.regime, lay.variant, lay.tile_words)
    os_ = [OracleRun(N, W, g, r, no_skip=True, thr4=t4, balanced=True) for g, r in zip(gs, rs)]
    rng = np.random.default_rng(11)
    x = np.zeros((I, N, W), np.uint64)
    for i, o in enumerate(os_):
        taubit = o.inst.taubit.astype(np.uint64)
        x[i] = (taubit * np.uint64(0xFFFFFFFFFFFFFFFF))[:, None]
        for k in range(64):
            x[i] ^= (rng.random((N, W)) < 0.02).astype(np.uint64) << np.uint64(k)
        o.s = o.inst.unpack(x[i])
        o.first_hit = o.inst.mark_initial(o.s)
    b.set_spins(torch.from_numpy(x.view(np.int64)).cuda())
    for n in (1, 2, 21, 40):
        b.run_sweeps(n)
        for o in os_:
            o.run_sweeps(n)
    xg, fh, e = b.spins_numpy(), b.first_hit_numpy(), b.energy().cpu().numpy()
    for i, o in enumerate(os_):
        assert np.array_equal(xg[i], o.x()), f"spins inst {i}"
        assert np.array_equal(fh[i], o.first_hit), f"first hits inst {i}"
        assert np.array_equal(e[i], o.energy()), f"energies inst {i}"
    if T <= 0.9 and N <= 192:
        hit = os_[0].first_hit != NO_HIT
        assert hit.sum() > 10                       # the case really sees first hits ...
    # back to the quasi-greedy table on the same batch: the plain kernel, still bit-exact
    b.set_flip_table([0, 236223201, TWO32, TWO32])
    assert b.layout().variant == 2
    b.run_sweeps(9)
    for i, o in enumerate(os_):
        o.thr4 = None
        o.run_sweeps(9)
        assert np.array_equal(b.spins_numpy()[i], o.x()) and np.array_equal(b.first_hit_numpy()[i], o.first_hit)
    b.close()
