"""xs_solved_mask_static: the allocation-free entry point (include/xs.h) against the existing path.

The existing path is xs_energy (a-11): a clone is in a ground state iff E = -N.  The
new entry point must report exactly those clones, bit for bit (integer work: no tolerance), on two
calls in a row that share the library's static scratch array -- the second on another batch with
fewer set bits, so that stale contents of the array would show.  Collected last on purpose
(the suite runs with pytest -x)."""
from __future__ import annotations

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")


def _mask_from_energy(b):
    """[inst][W] uint64 from the existing path: bit set <=> xs_energy says E = -N."""
    e = b.energy().cpu().numpy()                                    # [inst][64 W] int32
    solved = (e == -b.N).reshape(b.n_instances, b.W, 64)
    weights = np.uint64(1) << np.arange(64, dtype=np.uint64)
    return (solved.astype(np.uint64) * weights).sum(axis=2, dtype=np.uint64)


def test_static_scratch_mask_equals_energy_path_on_two_calls_in_a_row():
    import paper_2102_09510_b200 as xs
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP
    # batch A: tiny instances, clones sit in ground states all the time (many set bits)
    a = xs.Batch(18, 8, [5, 6, 7], [9, 10, 11], flags=fl)
    a.run_sweeps(60)
    # batch B: N = 256, 150 instances: (almost) no clone solved -> the scratch words of A must not leak
    seeds = list(range(300, 450))
    b = xs.Batch(256, 8, seeds, seeds, flags=fl | xs.XS_FLAG_BALANCED)
    b.run_sweeps(20)
    out_a = torch.empty((a.n_instances, a.W), dtype=torch.int64, device="cuda")
    out_b = torch.empty((b.n_instances, b.W), dtype=torch.int64, device="cuda")
    a.solved_mask_static(out=out_a)                                 # warm-up: loads the kernels
    torch.cuda.synchronize()
    want_a, want_b = _mask_from_energy(a), _mask_from_energy(b)
    out_a.fill_(0x5A5A5A5A)
    out_b.fill_(0x5A5A5A5A)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    a.solved_mask_static(out=out_a)                                 # two calls in a row, same stream
    b.solved_mask_static(out=out_b)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    got_a = out_a.cpu().numpy().view(np.uint64)
    got_b = out_b.cpu().numpy().view(np.uint64)
    assert np.array_equal(got_a, want_a), "first call differs from the xs_energy path"
    assert np.array_equal(got_b, want_b), "second call differs from the xs_energy path (stale scratch?)"
    assert free1 == free0, "the entry point must not allocate device memory"
    assert np.count_nonzero(want_a) > 4, "batch A should have clones in a ground state"
    # and again in the other order, after the state moved on
    a.run_sweeps(7)
    b.solved_mask_static(out=out_b)
    a.solved_mask_static(out=out_a)
    torch.cuda.synchronize()
    assert np.array_equal(out_b.cpu().numpy().view(np.uint64), want_b)
    assert np.array_equal(out_a.cpu().numpy().view(np.uint64), _mask_from_energy(a))
    # agrees with the first-hit bookkeeping too: a clone in a ground state now has a first hit (w0 = 0: absorbing)
    fh = a.first_hit_numpy().reshape(a.n_instances, a.W, 64) != xs.XS_NO_HIT
    m = out_a.cpu().numpy().view(np.uint64)
    bits = ((m[:, :, None] >> np.arange(64, dtype=np.uint64)) & np.uint64(1)).astype(bool)
    assert np.array_equal(bits, fh)
    a.close()
    b.close()


def test_static_scratch_rejects_sizes_beyond_the_maximum():
    import paper_2102_09510_b200 as xs
    W = xs.XS_STATIC_MAX_WORDS + 1
    big = xs.Batch(4, W, [1], [1], flags=xs.XS_FLAG_GAUGE)
    out = torch.empty((1, W), dtype=torch.int64, device="cuda")
    with pytest.raises(xs.XsError) as ei:
        big.solved_mask_static(out=out)
    assert ei.value.code == -1 and "XS_STATIC_MAX_WORDS" in str(ei.value)
    big.close()
    ok = xs.Batch(4, xs.XS_STATIC_MAX_WORDS, [1], [1], flags=xs.XS_FLAG_GAUGE)     # exactly the maximum
    m = ok.solved_mask_static().cpu().numpy().view(np.uint64)
    assert np.array_equal(m, _mask_from_energy(ok))
    ok.close()
