"""GPU-vs-oracle parity through the C ABI (bit-exact: spin words, energies, first-hit sweeps).

Protocol: SURVEY.md 8(c) "GPU-vs-oracle parity protocol" -- words evolve independently given
(seed, w) because the noise is counter based, so (i) all words for a moderate number of sweeps,
(ii) sampled words for the long runs at full size.  Tolerance: none; this is integer work.
"""
from __future__ import annotations

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from _harness import OracleRun  # noqa: E402
from oracle.xs_oracle import NO_HIT, Instance  # noqa: E402


def _xs():
    import paper_2102_09510_b200 as xs
    return xs


@pytest.fixture(autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")


def _compare(b, oracles, what=""):
    """b: xs.Batch; oracles: list of OracleRun, one per instance."""
    x = b.spins_numpy()
    fh = b.first_hit_numpy()
    e = b.energy().cpu().numpy()
    recs = b.tts()
    for i, o in enumerate(oracles):
        xo = o.x()
        eo = o.energy()
        for w in o.words:
            assert np.array_equal(x[i, :, w], xo[:, w]), f"{what}: spins differ inst {i} word {w}"
            sl = slice(64 * w, 64 * w + 64)
            assert np.array_equal(fh[i, sl], o.first_hit[sl]), f"{what}: first_hit differ inst {i} word {w}"
            assert np.array_equal(e[i, sl], eo[sl]), f"{what}: energies differ inst {i} word {w}"
        if len(o.words) == o.W:
            solved, tts, clone = o.tts()
            assert (recs[i].solved, recs[i].tts_sweeps, recs[i].clone) == (solved, tts, clone), what
        assert recs[i].sweeps_done == o.sweeps_done, f"{what}: sweeps_done inst {i}"


def test_init_state_and_energy():
    xs = _xs()
    for N, W, gs, rs in [(64, 3, 1, 1), (200, 8, 11, 12)]:
        b = xs.Batch(N, W, [gs], [rs])
        o = OracleRun(N, W, gs, rs)
        _compare(b, [o], f"init N={N}")
        b.close()


@pytest.mark.parametrize("N,W,sweeps,tile", [
    (64, 1, 300, 0),      # config-1 shape: one word, CW=1 path
    (96, 4, 120, 0),
    (96, 6, 60, 0),       # W not a power of two -> T = 2
    (200, 4, 40, 4),      # T = 4: static kernel with four row copies (variant 1)
    (256, 8, 40, 8),      # config-2 tile shape (T = 8)
    (256, 16, 24, 16),
    (130, 32, 20, 32),
    (70, 64, 12, 64),
    (512, 32, 8, 32),     # config-3 tile shape
])
@pytest.mark.parametrize("variant", [0, 1])
def test_sweep_parity_all_words(N, W, sweeps, tile, variant):
    """variant 0 = generic tile kernel, 1 = static-task kernel (falls back to 0 when T < 8)."""
    xs = _xs()
    b = xs.Batch(N, W, [N + 7], [3 * N + 1], flags=xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP,
                 geometry=dict(tile_words=tile, batch_sweeps=16, variant=variant))
    if tile:
        assert b.layout().tile_words == tile and b.layout().regime == 0
        if variant == 0:
            assert b.layout().variant == 0
    o = OracleRun(N, W, N + 7, 3 * N + 1, no_skip=True)
    half = sweeps // 3
    for n in (half, sweeps - half):          # two calls: resume must be exact
        b.run_sweeps(n)
        o.run_sweeps(n)
    _compare(b, [o], f"N={N} W={W}")
    b.close()


@pytest.mark.parametrize("N,W,cap,tile,variant,streaming", [
    (256, 8, 64, 8, 1, False),     # config-2 tile: 4 full rounds of 64 spins (static kernel, MAXT = 4)
    (256, 8, 64, 8, 0, False),     # same order on the generic kernel
    (128, 16, 0, 16, 1, False),    # q = 4 sets of 32
    (200, 4, 32, 4, 1, False),     # q = 7 sets of 28/29
    (384, 8, 64, 8, 1, False),     # q = 6
    (96, 4, 16, 0, 2, True),       # streaming regime
    (20, 2, 0, 0, 2, False),       # tiny N
])
def test_balanced_sets_parity(N, W, cap, tile, variant, streaming):
    """XS_FLAG_BALANCED (DESIGN.md R-balance): the library builds the balanced order itself (the
    oracle builds its own); trajectories must agree bit for bit on every kernel."""
    xs = _xs()
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_BALANCED
    if streaming:
        fl |= xs.XS_FLAG_STREAMING
    b = xs.Batch(N, W, [N + 11], [5 * N + 1], set_cap=cap, flags=fl,
                 geometry=dict(tile_words=tile, batch_sweeps=16, variant=variant))
    o = OracleRun(N, W, N + 11, 5 * N + 1, set_cap=cap, no_skip=True, balanced=True)
    assert o.inst.balanced
    tri, jbit, order, ss = b.get_graph(0)
    assert np.array_equal(order, o.inst.order) and np.array_equal(ss, o.inst.set_size)
    if tile and not streaming:
        assert b.layout().tile_words == tile and b.layout().variant == variant
    for n in (17, 1, 30):
        b.run_sweeps(n)
        o.run_sweeps(n)
    _compare(b, [o], f"balanced N={N} W={W}")
    b.close()


@pytest.mark.parametrize("N,W,tile,threads,sweeps", [
    (256, 8, 8, 512, 37),     # config-2 tile, one uint64 word per lane, two row copies
    (100, 16, 16, 512, 23),
    (60, 32, 32, 512, 21),
    (18, 8, 8, 128, 45),      # many solved clones: replay path with a 4-sweep noise period
    (100, 4, 4, 128, 33),     # T = 4: four row copies per 128-byte line
])
def test_static_kernel_one_word_per_lane(N, W, tile, threads, sweeps):
    """Static-task kernel with CW = 1: four lanes share a Philox call over a 4-sweep period."""
    xs = _xs()
    b = xs.Batch(N, W, [N + 3], [N + 4], flags=xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP,
                 geometry=dict(tile_words=tile, batch_sweeps=10, variant=1, words_per_lane=1, threads=threads))
    lay = b.layout()
    assert (lay.variant, lay.tile_words, lay.threads) == (1, tile, threads)
    o = OracleRun(N, W, N + 3, N + 4, no_skip=True)
    for n in (1, 2, 3, sweeps - 6):
        b.run_sweeps(n)
        o.run_sweeps(n)
        _compare(b, [o], f"CW=1 N={N} W={W}")
    b.close()


def test_config1_until_solved_matches_oracle_and_survey_hint(golden):
    """BASELINE.json configs[0]: N=64, seed 1, 64 clones, until E=-N, K=100 sweeps per call."""
    xs = _xs()
    hint = dict(line.split(None, 1) for line in open(golden("config1_survey_hint.txt"))
                if line.strip() and not line.startswith("#"))
    b = xs.Batch(64, 1, [1], [1])
    assert b.layout().variant == 3            # the latency kernel (one consumer warp + noise producers)
    o = OracleRun(64, 1, 1, 1)
    for _ in range(1000):
        b.run_sweeps(100)
        o.run_sweeps(100)
        if b.tts()[0].solved:
            break
    _compare(b, [o], "config 1")
    r = b.tts()[0]
    assert r.solved == 1
    assert r.tts_sweeps == int(hint["first_hit_sweep"]) and r.clone == int(hint["first_hit_clone"])
    # skipped once solved: further calls change nothing
    x0 = b.spins_numpy().copy()
    b.run_sweeps(100)
    o.run_sweeps(100)
    assert np.array_equal(b.spins_numpy(), x0)
    _compare(b, [o], "config 1 after solve")
    b.close()


@pytest.mark.parametrize("N,W,I,cap,balanced", [
    (64, 1, 1, 0, False),      # configs[0] shape
    (64, 4, 3, 0, False),      # four consumer warps, three instances
    (18, 2, 2, 0, False),      # tiny: clones solve all the time -> replay of the 32-sweep chunk
    (128, 1, 5, 0, True),      # 4 balanced sets of 32 = 8 passes of 16
    (200, 3, 1, 0, False),     # 16 passes (second instantiation)
    (96, 2, 1, 16, False),     # capped sets
])
def test_latency_kernel_parity(N, W, I, cap, balanced):
    """k_sweep_warp (layout variant 3): few instances with W <= 4 words; lanes <-> spins of the set,
    noise produced ahead by the producer warps.  Calls of 1, 31, 33 and 70 sweeps cross the 32-sweep
    noise chunks at odd offsets; resume must be exact."""
    xs = _xs()
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | (xs.XS_FLAG_BALANCED if balanced else 0)
    gs = [N + 2 + i for i in range(I)]
    rs = [5 * N + i for i in range(I)]
    b = xs.Batch(N, W, gs, rs, set_cap=cap, flags=fl, geometry=dict(variant=3))
    lay = b.layout()
    assert (lay.regime, lay.variant, lay.tile_words, lay.ctas) == (0, 3, W, I), (lay.variant, lay.tile_words)
    os_ = [OracleRun(N, W, g, r, set_cap=cap, no_skip=True, balanced=balanced) for g, r in zip(gs, rs)]
    for n in (1, 31, 33, 70):
        b.run_sweeps(n)
        for o in os_:
            o.run_sweeps(n)
        _compare(b, os_, f"latency kernel N={N} W={W} after {n}")
    if N == 18:
        assert (os_[0].first_hit != NO_HIT).sum() > 20
    b.close()


def test_latency_kernel_stop_rule_and_geometry_requests():
    """Solved instances are skipped by the latency kernel too; malformed geometry requests are
    refused; a request the shape cannot satisfy falls back to the rule."""
    xs = _xs()
    N, W = 32, 1
    gseeds, rseeds = list(range(3, 11)), list(range(13, 21))
    b = xs.Batch(N, W, gseeds, rseeds, set_cap=16, flags=xs.XS_FLAG_GAUGE, geometry=dict(variant=3))
    assert b.layout().variant == 3
    os_ = [OracleRun(N, W, g, r, set_cap=16) for g, r in zip(gseeds, rseeds)]
    for _ in range(10):
        b.run_sweeps(20)
        for o in os_:
            o.run_sweeps(20)
        _compare(b, os_, "latency kernel stop rule")
    assert len({o.sweeps_done for o in os_}) > 1
    for bad in (dict(tile_words=3), dict(threads=100), dict(words_per_lane=3), dict(variant=9)):
        with pytest.raises(xs.XsError) as ei:
            b.set_geometry(**bad)
        assert ei.value.code == -1
    b.set_geometry(variant=2)                  # W = 1: the clause-word kernel cannot take it
    assert b.layout().variant in (0, 1)
    b.set_geometry()                           # back to the rule
    b.close()


@pytest.mark.parametrize("batch", [1, 5, 64])
@pytest.mark.parametrize("streaming", [False, True])
@pytest.mark.parametrize("W", [4, 8])
def test_first_hit_exact_many_solved_clones(batch, streaming, W):
    """Small N: clones solve all the time -> exercises the in-kernel replay at every batch.
    W = 4 runs the generic tile kernel, W = 8 the static-task kernel (T = 8, two row copies)."""
    xs = _xs()
    N = 18
    flags = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | (xs.XS_FLAG_STREAMING if streaming else 0)
    b = xs.Batch(N, W, [5], [9], flags=flags,
                 geometry=dict(batch_sweeps=batch, variant=(1 if W == 8 else 0)))
    assert b.layout().regime == (1 if streaming else 0)
    if not streaming:
        assert b.layout().variant == (1 if W == 8 else 0)
    o = OracleRun(N, W, 5, 9, no_skip=True)
    for n in (1, 7, 30, 13):
        b.run_sweeps(n)
        o.run_sweeps(n)
        _compare(b, [o], f"batch={batch} streaming={streaming}")
    assert (o.first_hit != NO_HIT).sum() > 20
    b.close()


def test_streaming_regime_matches_oracle():
    xs = _xs()
    for N, W, sweeps in [(96, 16, 12), (150, 3, 10), (64, 2, 30)]:
        b = xs.Batch(N, W, [N], [N + 1], flags=xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_STREAMING)
        assert b.layout().regime == 1
        o = OracleRun(N, W, N, N + 1, no_skip=True)
        b.run_sweeps(sweeps)
        o.run_sweeps(sweeps)
        _compare(b, [o], f"streaming N={N} W={W}")
        b.close()


@pytest.mark.parametrize("streaming", [False, True])
def test_multi_instance_stop_rule(streaming):
    """Instances that have a solved clone at call entry are skipped (L129/L293 stop rule)."""
    xs = _xs()
    N, W = 32, 1
    gseeds = list(range(3, 11))
    rseeds = list(range(13, 21))
    b = xs.Batch(N, W, gseeds, rseeds,
                 flags=xs.XS_FLAG_GAUGE | (xs.XS_FLAG_STREAMING if streaming else 0))
    assert b.layout().regime == int(streaming)
    os_ = [OracleRun(N, W, g, r) for g, r in zip(gseeds, rseeds)]
    for _ in range(10):
        b.run_sweeps(20)
        for o in os_:
            o.run_sweeps(20)
        _compare(b, os_, "stop rule")
    done = [o.sweeps_done for o in os_]
    assert len(set(done)) > 1, "test should see instances stopping at different times"
    b.close()


def test_from_arrays_cap32_and_frustrated_couplings():
    """Paper-faithful cap-32 sets (L279) and arbitrary J (no planted solution)."""
    xs = _xs()
    N, W = 160, 4
    inst = Instance(N, 77, gauge=True, set_cap=32)
    rng = np.random.default_rng(5)
    jbit = rng.integers(0, 2, N).astype(np.uint8)
    inst2 = Instance(N, 77, set_cap=32, tri=inst.tri, jbit=jbit)
    arrays = (inst2.tri[None], jbit[None], inst2.order[None], inst2.set_size[None],
              np.array([inst2.n_sets], np.uint32))
    b = xs.Batch(N, W, run_seeds=[21], arrays=arrays, flags=xs.XS_FLAG_NO_SKIP)
    o = OracleRun(N, W, 77, 21, no_skip=True, inst=inst2)
    b.run_sweeps(25)
    o.run_sweeps(25)
    _compare(b, [o], "from arrays")
    tri, jb, order, ss = b.get_graph(0)
    assert np.array_equal(tri, inst2.tri) and np.array_equal(order, inst2.order)
    assert np.array_equal(ss, inst2.set_size) and np.array_equal(jb, jbit)
    b.close()


def test_gauge_covariance_on_gpu():
    """Run A (J=+1, x0) vs run B (planted J, x0 ^ taubit): x_B(t) = x_A(t) ^ taubit (L43)."""
    xs = _xs()
    N, W = 80, 4
    a = xs.Batch(N, W, [31], [5], flags=xs.XS_FLAG_NO_SKIP)                       # ferromagnet
    g = xs.Batch(N, W, [31], [5], flags=xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_GAUGE)    # gauged
    taubit = Instance(N, 31, gauge=True).taubit.astype(np.uint64)
    mask = (taubit * np.uint64(0xFFFFFFFFFFFFFFFF))[None, :, None]
    x0 = a.spins_numpy()
    g.set_spins(torch.from_numpy((x0 ^ mask).view(np.int64)).cuda())
    a.run_sweeps(50)
    g.run_sweeps(50)
    assert np.array_equal(g.spins_numpy(), a.spins_numpy() ^ mask)
    assert np.array_equal(g.energy().cpu().numpy(), a.energy().cpu().numpy())
    assert np.array_equal(g.first_hit_numpy(), a.first_hit_numpy())
    a.close()
    g.close()


def test_set_spins_planted_state_is_ground_state():
    xs = _xs()
    N, W = 100, 2
    b = xs.Batch(N, W, [8], [8])
    taubit = Instance(N, 8, gauge=True).taubit.astype(np.uint64)
    x = np.zeros((1, N, W), np.uint64)
    x[0, :, 0] = taubit * np.uint64(1 << 5)      # clone 5 = planted state, others all +1
    b.set_spins(torch.from_numpy(x.view(np.int64)).cuda())
    e = b.energy().cpu().numpy()[0]
    assert e[5] == -N
    r = b.tts()[0]
    fh = b.first_hit_numpy()[0]
    assert fh[5] == 0 and r.solved == 1 and r.tts_sweeps == 0 and r.clone <= 5
    b.close()


def test_error_codes_on_gpu():
    xs = _xs()
    p = xs.make_params(64, 1, 1)
    ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(xs.XsError) as ei:
        xs.xs_create_instance(p, [1], [1], ws.data_ptr() // 256 * 256 + 256, 16)
    assert ei.value.code == -2


@pytest.mark.parametrize("case", range(16))
def test_random_shapes_and_flags_parity(case):
    """Seeded random (N, W, instances, order, regime) combinations through whatever geometry the
    library picks (no overrides): the geometry rule must never change results."""
    xs = _xs()
    rng = np.random.default_rng(1000 + case)
    N = int(rng.choice([12, 24, 48, 64, 100, 128, 160, 192, 256, 320, 384]))
    W = int(rng.choice([1, 2, 4, 8, 8, 16, 24]))
    I = int(rng.choice([1, 3, 40, 160])) if N <= 256 and W <= 8 else int(rng.choice([1, 2]))
    balanced = bool(rng.integers(0, 2))
    cap = int(rng.choice([0, 0, 16, 32, 64]))
    streaming = bool(rng.integers(0, 4) == 0)
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | (xs.XS_FLAG_BALANCED if balanced else 0) | \
        (xs.XS_FLAG_STREAMING if streaming else 0)
    gseeds = [5000 + 17 * case + i for i in range(I)]
    rseeds = [9000 + 31 * case + i for i in range(I)]
    b = xs.Batch(N, W, gseeds, rseeds, set_cap=cap, flags=fl)
    lay = b.layout()
    check = sorted(set([0, I - 1, I // 2]))
    oracles = {i: OracleRun(N, W, gseeds[i], rseeds[i], set_cap=cap, no_skip=True, balanced=balanced)
               for i in check}
    for n in (int(rng.integers(1, 40)), int(rng.integers(1, 80))):
        b.run_sweeps(n)
        for o in oracles.values():
            o.run_sweeps(n)
    x, fh, e = b.spins_numpy(), b.first_hit_numpy(), b.energy().cpu().numpy()
    for i, o in oracles.items():
        what = f"case {case}: N={N} W={W} I={I} bal={balanced} cap={cap} stream={streaming} " \
               f"regime={lay.regime} variant={lay.variant} T={lay.tile_words} thr={lay.threads} inst={i}"
        assert np.array_equal(x[i], o.x()), what
        assert np.array_equal(fh[i], o.first_hit), what
        assert np.array_equal(e[i], o.energy()), what
    b.close()
