"""tts_run.run_size (the TTS accounting harness) against the oracle: every
entry's TTS = sweep of the first ground-state hit over the clones, exact."""
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


@pytest.mark.parametrize("balanced", [False, True])
def test_run_size_tts_equals_oracle_first_hits(balanced):
    import paper_2102_09510_b200 as xs
    from paper_2102_09510_b200 import tts_run
    n, words, instances, runs, cap, seed0 = 24, 1, 3, 2, 3000, 300
    out = tts_run.run_size(n, words, instances, runs, cap, 50, seed0,
                           flags_extra=xs.XS_FLAG_BALANCED if balanced else 0)
    assert out["total_runs"] == instances * runs and out["clones"] == 64
    # the same entries with the oracle, advanced in the same chunks with the same stop rule
    expect = []
    for i in range(instances):
        for r in range(runs):
            o = OracleRun(n, words, seed0 + i, seed0 + i + 7919 * (r + 1), balanced=balanced)
            done = 0
            while done < cap and not o.solved:
                o.run_sweeps(50)
                done += 50
            expect.append(o.tts()[1] if o.solved else NO_HIT)
    expect = np.array(expect, dtype=np.uint64)
    solved = expect != NO_HIT
    assert out["solved_runs"] == int(solved.sum()) and solved.sum() >= 4
    per_inst = expect.reshape(instances, runs)
    taus = []
    for i in range(instances):
        v = per_inst[i]
        n_s = int((v != NO_HIT).sum())
        t_tot = float(v[v != NO_HIT].sum() + (runs - n_s) * cap)
        taus.append(t_tot / n_s if n_s else float("inf"))
    assert out["median_tau_sweeps"] == pytest.approx(float(np.median(taus)), rel=1e-12)
