"""world_size-2 gloo test (CPU) of the N > 1 host logic: replicas only, no data-path collective
(DESIGN.md section 9).  Checks rank seeds, the max-over-ranks timing and the min-merge of TTS."""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    import torch.distributed as dist
    from paper_2102_09510_b200 import replicas
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seeds = replicas.replica_run_seeds([2, 3], rank)
    ms = replicas.max_over_ranks([10.0 + 5.0 * rank, 7.0 - rank], dist)
    rate = replicas.job_rate(1e9, 4, world, ms[0])
    tts_local = [100, replicas.NO_HIT, replicas.NO_HIT] if rank == 0 else [250, 40, replicas.NO_HIT]
    merged = replicas.merge_tts(tts_local, dist)
    np.save(os.path.join(out_dir, f"r{rank}.npy"),
            np.array([seeds[0], seeds[1], ms[0], ms[1], rate, *merged], dtype=np.float64))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_world_size_2(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0 = np.load(tmp_path / "r0.npy")
    r1 = np.load(tmp_path / "r1.npy")
    assert list(r0[:2]) == [2, 3] and list(r1[:2]) == [1002, 1003]      # different noise per rank
    for r in (r0, r1):
        assert r[2] == 15.0 and r[3] == 7.0                              # max over ranks
        assert r[4] == pytest.approx(2 * 1e9 * 4 / (15.0 * 1e6))         # whole-job rate
        assert list(r[5:].astype(np.uint64)) == [100, 40, 0xFFFFFFFF]    # min over ranks, NO_HIT kept
