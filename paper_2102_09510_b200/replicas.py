"""Multi-GPU = independent replicas ("multiple GPUs ... executing the same code with
different random seeds").  The path has no exchange step, so there is no data-path collective;
the only cross-rank traffic is the timing reduction (max over ranks) and, for a run that stops at
the first solution, one min-reduce of the per-instance TTS records.  Host logic only."""
from __future__ import annotations

import numpy as np

NO_HIT = 0xFFFFFFFF


def replica_run_seeds(base_seeds, rank: int):
    """Run seeds of rank `rank`: same instances, different noise / initial states."""
    return [int(s) + 1000 * int(rank) for s in base_seeds]


def max_over_ranks(values_ms, dist=None, device=None):
    """Element-wise max over ranks of a list of per-rank device times (ms)."""
    import torch
    t = torch.tensor(list(values_ms), dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def job_rate(updates_per_rank_per_step: float, steps: int, world: int, total_ms: float) -> float:
    """Whole-job clone-spin updates per ns: all ranks' updates / slowest rank's time."""
    return world * updates_per_rank_per_step * steps / (total_ms * 1e6)


def merge_tts(tts_sweeps, dist=None, device=None):
    """Per-instance TTS of a replicated run = min over ranks of the ranks' TTS (L111 applied to
    the union of all ranks' clones); NO_HIT where no rank solved."""
    import torch
    t = torch.tensor(np.asarray(tts_sweeps, dtype=np.int64), dtype=torch.int64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return t.cpu().numpy().astype(np.uint32)
