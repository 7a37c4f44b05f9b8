"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (library
defaults, no geometry overrides), on sampled words the oracle can follow one by one
(SURVEY.md 8(c) protocol (ii): words evolve independently given (seed, w))."""
from __future__ import annotations

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from _harness import OracleRun  # noqa: E402
from oracle.xs_oracle import NO_HIT  # noqa: E402


@pytest.fixture(autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")


def _check_words(b, o, inst=0):
    x = b.spins_numpy()[inst]
    fh = b.first_hit_numpy()[inst]
    e = b.energy().cpu().numpy()[inst]
    xo, eo = o.x(), o.energy()
    for w in o.words:
        sl = slice(64 * w, 64 * w + 64)
        assert np.array_equal(x[:, w], xo[:, w]), f"spin words differ in word {w}"
        assert np.array_equal(fh[sl], o.first_hit[sl]), f"first hits differ in word {w}"
        assert np.array_equal(e[sl], eo[sl]), f"energies differ in word {w}"


@pytest.mark.parametrize("balanced", [True, False])
def test_config2_full_size_sampled_words(balanced):
    """configs[1]: N=256, graph seed 2, 2^16 clones; bench.py's launch configuration (balanced
    sets of 64, clause-word kernel, T=8) and the greedy-order variant (`--workload config2_greedy`:
    6 ragged sets on 64 slots, same kernel with idle slots)."""
    import paper_2102_09510_b200 as xs
    N, W = 256, 1024
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | (xs.XS_FLAG_BALANCED if balanced else 0)
    b = xs.Batch(N, W, [2], [2], set_cap=64 if balanced else 0, flags=fl)
    lay = b.layout()
    assert (lay.regime, lay.variant, lay.tile_words, lay.ctas) == (0, 2, 8, 128)
    assert lay.n_sets_max == (4 if balanced else 6)
    words = [0, 7, 8, 517, 1023]          # first/last lane of a tile, tile boundaries, last tile
    o = OracleRun(N, W, 2, 2, set_cap=64 if balanced else 0, no_skip=True, words=words,
                  balanced=balanced)
    for n in (130, 171):                  # 301 sweeps: crosses one 256-sweep detection batch at odd offsets
        b.run_sweeps(n)
        o.run_sweeps(n)
    _check_words(b, o)
    # properties that hold for every clone at any size
    e = b.energy().cpu().numpy()[0]
    assert e.min() >= -N and (e % 2 == 0).all() and abs(e.mean() / N + 0.8957) < 0.02
    r = b.tts()[0]
    assert r.sweeps_done == 301 and r.solved == int((b.first_hit_numpy() != NO_HIT).any())
    b.close()


@pytest.mark.parametrize("balanced", [True, False])
def test_config3_shape_sampled_instances_and_words(balanced):
    """configs[2] shape: N=512, W=64 per instance, 160 instances so that every SM gets a tile.
    balanced (bench.py --workload config3): 4 sets of 128 -> clause-word kernel, T=8, 512 threads;
    greedy (config3_greedy): 7 ragged sets would leave 43 % of the clause-word kernel's slots idle ->
    generic kernel, T=16 -- the geometries the 256-instance runs use."""
    import paper_2102_09510_b200 as xs
    N, W, I = 512, 64, 160
    seeds = list(range(100, 100 + I))
    b = xs.Batch(N, W, seeds, seeds, flags=xs.XS_FLAG_GAUGE | (xs.XS_FLAG_BALANCED if balanced else 0))
    lay = b.layout()
    assert (lay.regime, lay.variant, lay.tile_words, lay.threads) == ((0, 2, 8, 512) if balanced else (0, 0, 16, 512))
    checks = {0: [0, 15, 16], 77: [33, 63], 159: [48]}
    oracles = {i: OracleRun(N, W, seeds[i], seeds[i], words=ws, balanced=balanced) for i, ws in checks.items()}
    for n in (70, 563):                   # 633 sweeps: two full 256-sweep detection batches + a remainder
        b.run_sweeps(n)
    for i, o in oracles.items():
        o.run_sweeps(633)
        _check_words(b, o, inst=i)
    recs = b.tts()
    assert all(r.sweeps_done == 633 for r in recs)
    b.close()


@pytest.mark.parametrize("N,threads,tile", [(128, 128, 8), (192, 128, 8), (256, 256, 8), (384, 256, 8),
                                            (768, 512, 8), (1024, 512, 8)])
def test_config4_shapes_balanced_static_geometry(N, threads, tile):
    """configs[3] shapes that run on the static kernel in bench.py (--workload config4_N): 160
    instances of W = 8 give one tile per SM and more; sampled instances, all words."""
    import paper_2102_09510_b200 as xs
    W, I = 8, 160
    seeds = [1000 * N + i for i in range(I)]
    b = xs.Batch(N, W, seeds, seeds, flags=xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_BALANCED)
    lay = b.layout()
    # 4 or 6 sets that fill a T = 8 CTA -> clause-word kernel (variant 2); N = 1024 (T = 4): spin-word static kernel
    assert (lay.regime, lay.variant, lay.tile_words, lay.threads) == (0, 2 if tile == 8 else 1, tile, threads)
    oracles = {i: OracleRun(N, W, seeds[i], seeds[i], no_skip=True, balanced=True) for i in (0, 101, 159)}
    for n in (65, 40, 530):               # 635 sweeps: two full 256-sweep detection batches + a remainder
        b.run_sweeps(n)
    for i, o in oracles.items():
        o.run_sweeps(635)
        _check_words(b, o, inst=i)
    b.close()


def test_config2_full_sweep_count_sampled_words():
    """configs[1] exactly as bench.py runs it: ONE xs_run_sweeps call of 10^4 sweeps (39 detection
    batches of 256 + 16) on 2^16 clones; sampled words followed by the oracle for all 10^4 sweeps
    (SURVEY.md 8(c) protocol (ii))."""
    import paper_2102_09510_b200 as xs
    N, W = 256, 1024
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_BALANCED
    b = xs.Batch(N, W, [2], [2], set_cap=64, flags=fl)
    lay = b.layout()
    assert (lay.regime, lay.variant, lay.tile_words, lay.ctas, lay.batch_sweeps) == (0, 2, 8, 128, 256)
    words = [0, 7, 517, 1023]
    o = OracleRun(N, W, 2, 2, set_cap=64, no_skip=True, words=words, balanced=True)
    b.run_sweeps(10_000)
    o.run_sweeps(10_000)
    _check_words(b, o)
    assert b.tts()[0].sweeps_done == 10_000
    b.close()


@pytest.mark.parametrize("clone_noise", [False, True])
def test_config5_full_size_grid_stride_path(clone_noise):
    """configs[4] at its real size, N = 2^20, W = 16: the largest independent set has ~262 000 spins
    x 8 lane tasks, more than the 8 CTAs per SM x 256 threads the launch has, so every thread of
    k_stream_set loops over several tasks (the path N = 2^16 never reaches).  One sampled word is
    followed by the oracle (1 GiB of one-byte spins on the host); with XS_FLAG_CLONE_NOISE the
    per-clone noise variant runs on the same path."""
    import paper_2102_09510_b200 as xs
    N, W = 1 << 20, 16
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | (xs.XS_FLAG_CLONE_NOISE if clone_noise else 0)
    b = xs.Batch(N, W, [5], [5], flags=fl)
    lay = b.layout()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    assert lay.regime == 1 and lay.ctas == 8 * sms
    _, _, _, ss = b.get_graph(0)
    assert int(ss.max()) * (W // 2) > lay.ctas * lay.threads     # more than one task per thread
    o = OracleRun(N, W, 5, 5, no_skip=True, words=[9], clone_m=7 if clone_noise else None)
    b.run_sweeps(2)
    o.run_sweeps(2)
    x = b.spins_numpy()[0]
    assert np.array_equal(x[:, 9], o.x()[:, 9]), "spin words differ"
    fh = b.first_hit_numpy()[0]
    assert np.array_equal(fh[576:640], o.first_hit[576:640])
    e = b.energy().cpu().numpy()[0]
    s9 = o.s[576:640]
    assert np.array_equal(e[576:640], o.inst.energy(s9))
    assert e.min() >= -N and (e % 2 == 0).all()
    assert b.tts()[0].sweeps_done == 2
    b.close()


def test_config5_streaming_large_instance_sampled_word():
    """configs[4] regime at N = 2^16 (2^20 is exercised by bench.py --workload config5): state
    does not fit on chip -> streaming kernel, W = 16 (128-byte rows)."""
    import paper_2102_09510_b200 as xs
    N, W = 1 << 16, 16
    b = xs.Batch(N, W, [5], [5], flags=xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP)
    assert b.layout().regime == 1
    o = OracleRun(N, W, 5, 5, no_skip=True, words=[3])
    b.run_sweeps(3)
    o.run_sweeps(3)
    _check_words(b, o)
    e = b.energy().cpu().numpy()[0]
    assert e.min() >= -N and (e % 2 == 0).all()
    b.close()


def test_max_tile_and_ragged_shapes():
    """Edge shapes: N = 3 (smallest legal), N not a multiple of anything, W = 1, W = 24 (T = 8),
    one 64-column tile."""
    import paper_2102_09510_b200 as xs
    for N, W, sweeps in [(3, 1, 5), (7, 2, 9), (131, 24, 11), (67, 64, 9), (37, 5, 12)]:
        b = xs.Batch(N, W, [N], [2 * N], flags=xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP)
        o = OracleRun(N, W, N, 2 * N, no_skip=True)
        b.run_sweeps(sweeps)
        o.run_sweeps(sweeps)
        _check_words(b, o)
        b.close()
