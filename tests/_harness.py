"""Test-side helpers: run the CPU oracle in the shape of the C ABI's calls.

Only tests import this.  The oracle (oracle/xs_oracle.py) is never imported by the product.
"""
from __future__ import annotations

import numpy as np

from oracle.xs_oracle import NO_HIT, W1_THRESHOLD, Instance


class OracleRun:
    """One instance, W words, evolving under the oracle with the harness-level stop rule of
    SURVEY.md 8(c) item 9 / include/xs.h: run_sweeps(n) advances by exactly n sweeps unless the
    instance was already solved at call entry (and skipping is on)."""

    def __init__(self, N, W, graph_seed, run_seed, gauge=True, set_cap=0, thr=W1_THRESHOLD,
                 no_skip=False, inst: Instance | None = None, words=None, thr4=None, balanced=False,
                 clone_m=None):
        self.inst = inst if inst is not None else Instance(N, graph_seed, gauge, set_cap,
                                                           balanced=balanced)
        self.N, self.W, self.run_seed, self.thr, self.no_skip = N, W, run_seed, thr, no_skip
        self.thr4 = thr4                     # general flip table or None = QG
        self.clone_m = clone_m               # per-clone noise variant (NEXT-2): w1 = clone_m / 128
        # `words`: evolve only this subset of word indices (others stay at their initial value)
        self.words = list(range(W)) if words is None else sorted(words)
        self.s = self.inst.init_spins(W, run_seed)
        self.first_hit = self.inst.mark_initial(self.s)
        self.sweeps_done = 0

    @property
    def solved(self) -> bool:
        sel = self._clone_sel()
        return bool((self.first_hit[sel] != NO_HIT).any())

    def _clone_sel(self):
        return np.concatenate([np.arange(64 * w, 64 * w + 64) for w in self.words])

    def run_sweeps(self, n):
        if self.solved and not self.no_skip:
            return
        for w in self.words:
            self.inst.run(self.s, self.first_hit, self.run_seed, self.sweeps_done, n, w, w + 1,
                          thr=self.thr, thr4=self.thr4, clone_m=self.clone_m)
        self.sweeps_done += n

    def x(self) -> np.ndarray:
        return self.inst.pack(self.s)           # uint64 [N][W]

    def energy(self) -> np.ndarray:
        return self.inst.energy(self.s)

    def tts(self):
        sel = self._clone_sel()
        fh = self.first_hit[sel]
        if not (fh != NO_HIT).any():
            return 0, NO_HIT, NO_HIT
        m = fh.min()
        return 1, int(m), int(sel[np.nonzero(fh == m)[0][0]])
