"""GPU-vs-oracle parity of the per-clone noise variant (XS_FLAG_CLONE_NOISE):
bit-exact spin words, energies and first hits through the C ABI."""
from __future__ import annotations

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from _harness import OracleRun  # noqa: E402
from test_gpu_parity import _compare  # noqa: E402


@pytest.fixture(autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")


@pytest.mark.parametrize("N,W,sweeps", [(64, 1, 40), (96, 4, 30), (50, 6, 25), (200, 16, 12), (18, 2, 60)])
def test_clone_noise_parity_default_m7(N, W, sweeps):
    import paper_2102_09510_b200 as xs
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_CLONE_NOISE
    b = xs.Batch(N, W, [N + 1], [2 * N + 1], flags=fl)
    assert b.layout().regime == 1                       # streaming regime
    o = OracleRun(N, W, N + 1, 2 * N + 1, no_skip=True, clone_m=7)   # round(0.055 * 128) = 7
    for n in (1, sweeps // 2, sweeps - sweeps // 2 - 1):
        b.run_sweeps(n)
        o.run_sweeps(n)
        _compare(b, [o], f"clone noise N={N} W={W}")
    b.close()


@pytest.mark.parametrize("m", [0, 1, 40, 127, 128])
def test_clone_noise_other_m_through_set_flip_table(m):
    import paper_2102_09510_b200 as xs
    N, W = 40, 2
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_CLONE_NOISE
    b = xs.Batch(N, W, [3], [4], flags=fl)
    b.set_flip_table([0, m << 25, 1 << 32, 1 << 32])
    o = OracleRun(N, W, 3, 4, no_skip=True, clone_m=m)
    for n in (7, 20):
        b.run_sweeps(n)
        o.run_sweeps(n)
    _compare(b, [o], f"clone noise m={m}")
    with pytest.raises(xs.XsError):                      # only the quasi-greedy form
        b.set_flip_table([5, m << 25, 1 << 32, 1 << 32])
    b.close()


def test_clone_noise_multi_instance_stop_rule_and_first_hits():
    import paper_2102_09510_b200 as xs
    N, W, I = 16, 2, 5
    seeds = [20 + i for i in range(I)]
    b = xs.Batch(N, W, seeds, seeds, flags=xs.XS_FLAG_GAUGE | xs.XS_FLAG_CLONE_NOISE)
    oracles = [OracleRun(N, W, s, s, clone_m=7) for s in seeds]
    for n in (3, 9, 30):
        b.run_sweeps(n)
        for o in oracles:
            o.run_sweeps(n)
        _compare(b, oracles, "clone noise stop rule")
    assert any(o.solved for o in oracles)
    b.close()


@pytest.mark.parametrize("N,W,I,m", [(128, 8, 2, None), (256, 16, 1, None), (192, 8, 1, 40), (512, 8, 1, 1), (384, 8, 1, None)])
def test_clone_noise_on_the_clause_word_kernel(N, W, I, m):
    """SURVEY.md 8(f) NEXT-2 on chip: with balanced sets that fill the CTA (4 - 8 rounds) the per-clone
    noise runs on the clause-word kernel (layout regime 0, variant 2), each lane drawing the 7-bit
    numbers of its two words' 128 clones from 8 Philox calls per round."""
    import paper_2102_09510_b200 as xs
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_CLONE_NOISE | xs.XS_FLAG_BALANCED
    gs, rs = [N + 60 + i for i in range(I)], [4 * N + i for i in range(I)]
    b = xs.Batch(N, W, gs, rs, flags=fl, geometry=dict(batch_sweeps=16))
    if m is not None:
        b.set_flip_table([0, m << 25, 1 << 32, 1 << 32])
    lay = b.layout()
    assert (lay.regime, lay.variant, lay.tile_words) == (0, 2, 8), (lay.regime, lay.variant)
    os_ = [OracleRun(N, W, g, r, no_skip=True, balanced=True, clone_m=7 if m is None else m) for g, r in zip(gs, rs)]
    for n in (1, 2, 19):
        b.run_sweeps(n)
        for o in os_:
            o.run_sweeps(n)
    _compare(b, os_, f"clone noise on chip N={N} W={W}")
    b.set_geometry(variant=0)                      # no other on-chip kernel has it: the batch streams
    assert b.layout().regime == 1
    b.run_sweeps(5)
    for o in os_:
        o.run_sweeps(5)
    _compare(b, os_, "clone noise, back to streaming")
    b.close()
