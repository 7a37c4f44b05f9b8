"""GPU-vs-oracle parity of the clause-word kernel (`k_sweep_clause`, layout variant 2): shared
memory holds c_t = x_i ^ x_j ^ x_k ^ J_t (the number of unsatisfied interactions
a spin enters is all its update needs), the spin words live in registers.  The kernel serves the
on-chip shapes with W a multiple of 8 whose update order fits 4 to 8 rounds of a CTA: balanced sets that
fill the CTA (bench.py's config 2 / 3 / 4 geometry, kernel MODE 1 and 2) and ragged orders with idle
slots (greedy sets, N = 160 / 224 / 320, MODE 0); results must equal the oracle's bit for bit, like
every other kernel's."""
import numpy as np
import pytest
import torch

from _harness import OracleRun
from oracle.xs_oracle import NO_HIT
from test_gpu_parity import _compare, _xs

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")


@pytest.mark.parametrize("N,W,threads,batch", [
    (128, 16, 128, 16),     # 4 sets of 32, two tiles
    (256, 8, 256, 16),      # the config-2 tile
    (256, 24, 256, 64),     # three tiles, default detection batch
    (512, 8, 512, 5),       # the config-3 tile, odd batch
    (192, 8, 128, 16),      # 6 sets of 32 (6 rounds per sweep)
    (384, 16, 256, 64),     # 6 sets of 64
    (768, 8, 512, 9),       # 6 sets of 128
])
def test_clause_kernel_parity_all_words(N, W, threads, batch):
    xs = _xs()
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_BALANCED
    ref = xs.Batch(N, W, [N + 3], [7 * N], flags=fl,
                 geometry=dict(tile_words=8, variant=1, batch_sweeps=batch))          # spin-word static kernel
    b = xs.Batch(N, W, [N + 3], [7 * N], flags=fl,
                 geometry=dict(tile_words=8, batch_sweeps=batch))    # few tiles: the automatic rule would take T = 4
    lay = b.layout()
    assert (lay.regime, lay.variant, lay.tile_words, lay.threads) == (0, 2, 8, threads)
    assert ref.layout().variant == 1
    o = OracleRun(N, W, N + 3, 7 * N, no_skip=True, balanced=True)
    for n in (1, 2, 40, 23):                 # odd starts of the 2-sweep noise period, resume across calls
        b.run_sweeps(n)
        ref.run_sweeps(n)
        o.run_sweeps(n)
    _compare(b, [o], f"clause kernel N={N} W={W}")
    assert np.array_equal(b.spins_numpy(), ref.spins_numpy())
    b.close()
    ref.close()


@pytest.mark.parametrize("batch", [1, 7, 64])
def test_clause_kernel_first_hit_many_solved_clones(batch):
    """Clones started a few spin flips away from the planted state reach E = -N within a few
    sweeps at different times: detection pass, replay of the batch, exact first-hit sweep (L293)."""
    xs = _xs()
    N, W = 128, 8
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_BALANCED
    b = xs.Batch(N, W, [77], [78], flags=fl,
                 geometry=dict(tile_words=8, batch_sweeps=batch))
    assert b.layout().variant == 2
    o = OracleRun(N, W, 77, 78, no_skip=True, balanced=True)
    rng = np.random.default_rng(5)
    taubit = o.inst.taubit.astype(np.uint64)
    x = np.zeros((1, N, W), np.uint64)
    x[0] = (taubit * np.uint64(0xFFFFFFFFFFFFFFFF))[:, None]
    for k in range(64):                       # flip each (spin, clone) bit with probability 0.04
        x[0] ^= (rng.random((N, W)) < 0.04).astype(np.uint64) << np.uint64(k)
    b.set_spins(torch.from_numpy(x.view(np.int64)).cuda())
    o.s = o.inst.unpack(x[0])
    o.first_hit = o.inst.mark_initial(o.s)
    for n in (3, 70, 6):
        b.run_sweeps(n)
        o.run_sweeps(n)
    _compare(b, [o], f"clause kernel first hits, batch {batch}")
    fh = b.first_hit_numpy()[0]
    hit = fh[fh != NO_HIT]
    assert hit.size > 50 and np.unique(hit).size > 3      # the case really exercises the replay
    b.close()


def test_clause_kernel_multi_instance_stop_rule_and_flip_table_switch():
    xs = _xs()
    N, W, I = 128, 8, 150
    seeds = [900 + i for i in range(I)]
    b = xs.Batch(N, W, seeds, seeds, flags=xs.XS_FLAG_GAUGE | xs.XS_FLAG_BALANCED)
    assert b.layout().variant == 2 and b.layout().ctas == I
    b.set_flip_table([0, 236223201, 1 << 31, 1 << 32])           # w2 < 1: general table, generic kernel
    assert b.layout().variant == 0
    b.set_flip_table([0, 236223201, 1 << 32, 1 << 32])           # back to quasi-greedy
    assert b.layout().variant == 2
    oracles = {i: OracleRun(N, W, seeds[i], seeds[i], balanced=True) for i in (0, 74, 149)}
    for n in (33, 64):
        b.run_sweeps(n)
    x = b.spins_numpy()
    fh = b.first_hit_numpy()
    for i, o in oracles.items():
        o.run_sweeps(33)
        o.run_sweeps(64)
        assert np.array_equal(x[i], o.x()) and np.array_equal(fh[i], o.first_hit)
    assert all(r.sweeps_done == 97 for r in b.tts())
    b.close()


@pytest.mark.parametrize("N,W,I,balanced,cap,threads,rounds_max", [
    (256, 8, 1, False, 0, 256, 8),      # greedy sets of config 2's graph family: ragged, idle slots
    (512, 16, 3, False, 0, 512, 8),     # greedy, three instances with different set structures
    (128, 8, 5, False, 0, 128, 8),
    (160, 8, 2, True, 0, 128, 5),       # PAPER.md L99 sizes: 5 sets of 32
    (224, 8, 2, True, 0, 128, 7),       # 7 sets of 32
    (320, 16, 1, True, 0, 256, 5),      # 5 sets of 64
    (1024, 8, 2, True, 0, 512, 8),      # 4 sets of 256 on 128 slots: 8 rounds, barrier every second round
    (100, 8, 1, True, 25, 128, 4),      # 4 sets of 25 on 32 slots
    (200, 8, 2, True, 50, 256, 4),      # 4 sets of 50 on 64 slots
    (96, 8, 1, False, 0, 128, 8),
    (256, 8, 2, False, 32, 128, 11),    # the paper's cap-32 sets (L279): 9 and 11 rounds -> the long-list kernels
])
def test_clause_kernel_ragged_orders_and_round_counts(N, W, I, balanced, cap, threads, rounds_max):
    """Orders that do not fill the CTA (idle slots on scratch rows), 5 / 7 / 8 rounds per sweep, sets
    of two rounds, several instances with different set structures in one launch."""
    xs = _xs()
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | (xs.XS_FLAG_BALANCED if balanced else 0)
    gs = [N + 5 + i for i in range(I)]
    rs = [3 * N + i for i in range(I)]
    b = xs.Batch(N, W, gs, rs, set_cap=cap, flags=fl, geometry=dict(batch_sweeps=16))
    lay = b.layout()
    assert (lay.regime, lay.variant, lay.tile_words, lay.threads) == (0, 2, 8, threads), \
        (lay.regime, lay.variant, lay.tile_words, lay.threads)
    os_ = [OracleRun(N, W, g, r, set_cap=cap, no_skip=True, balanced=balanced) for g, r in zip(gs, rs)]
    for n in (1, 2, 30, 21):
        b.run_sweeps(n)
        for o in os_:
            o.run_sweeps(n)
    _compare(b, os_, f"clause kernel ragged N={N} W={W} I={I}")
    b.close()


def test_clause_kernel_more_than_256_instances_and_w1_zero():
    """Run seeds travel in the kernel parameters, 256 instances per launch: 300 instances take two
    launches.  Second batch: w1 = 0 (the k = 1 move is never taken: the compare's forced carry)."""
    xs = _xs()
    N, W, I = 64, 8, 300
    seeds = [40 + i for i in range(I)]
    fl = xs.XS_FLAG_GAUGE | xs.XS_FLAG_NO_SKIP | xs.XS_FLAG_BALANCED
    b = xs.Batch(N, W, seeds, seeds, flags=fl)
    assert b.layout().variant == 2 and b.layout().ctas == I
    b.run_sweeps(37)
    x, fh = b.spins_numpy(), b.first_hit_numpy()
    for i in (0, 255, 256, 299):
        o = OracleRun(N, W, seeds[i], seeds[i], no_skip=True, balanced=True)
        o.run_sweeps(37)
        assert np.array_equal(x[i], o.x()) and np.array_equal(fh[i], o.first_hit), i
    b.close()
    for thr in (0, 1, 0xFFFFFFFF):
        b = xs.Batch(128, 8, [3], [4], flags=fl, w1_threshold=thr)
        assert b.layout().variant == 2
        o = OracleRun(128, 8, 3, 4, thr=thr, no_skip=True, balanced=True)
        b.run_sweeps(25)
        o.run_sweeps(25)
        _compare(b, [o], f"w1 threshold {thr}")
        b.close()
