"""B200-native quasi-greedy clone sweep for 3-XORSAT (arXiv 2102.09510).

The product is libxs_b200.so (include/xs.h); this package is its thin Python binding.  `Batch`
only owns the torch tensors that serve as device memory and forwards every call to the C ABI.
"""
from __future__ import annotations

import numpy as np

from ._binding import (XS_FLAG_BALANCED, XS_FLAG_CLONE_NOISE, XS_FLAG_GAUGE, XS_FLAG_NO_SKIP, XS_FLAG_STREAMING,  # noqa: F401
                       XS_NO_HIT,
                       XS_W1_THRESHOLD_DEFAULT, XsError, lib, make_params, xs_alu_peak, xs_cavity_barrier,
                       xs_create_instance, xs_kernel_launches,
                       xs_create_instance_from_arrays, xs_destroy, xs_energy, xs_get_first_hit,
                       xs_clause_placement, xs_generate_graph, xs_get_graph, xs_get_layout, xs_get_spins, xs_params, xs_run_sweeps, xs_set_flip_table, xs_set_geometry, XS_GEOM_AUTO,
                       xs_set_spins, xs_solved_mask_static, XS_STATIC_MAX_WORDS, xs_tts, xs_tts_rec, xs_tts_stats, xs_workspace_bytes)


class Batch:
    """>= 1 instances of equal N and W on one GPU (opaque xs_batch handle + its torch workspace).

    Every call runs with the batch's device current and on that device's current torch stream
    (or the stream passed), whatever device is current in the caller."""

    def __init__(self, n_spins, n_words, graph_seeds=None, run_seeds=None, *, arrays=None,
                 set_cap=0, w1_threshold=XS_W1_THRESHOLD_DEFAULT, flags=XS_FLAG_GAUGE,
                 device="cuda:0", stream=None, geometry=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2102_09510_b200 needs a CUDA device (there is no CPU path)")
        self.device = torch.device(device)
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        run_seeds = np.atleast_1d(np.asarray(run_seeds, dtype=np.uint64))
        self.n_instances = int(run_seeds.size)
        self.params = make_params(n_spins, n_words, self.n_instances, set_cap, w1_threshold, flags)
        self.N, self.W = int(n_spins), int(n_words)
        self.ws_bytes = xs_workspace_bytes(self.params)
        self.h = None
        with torch.cuda.device(self.device):
            self.ws = torch.empty(self.ws_bytes + 256, dtype=torch.uint8, device=self.device)
            base = self.ws.data_ptr()
            self._ws_ptr = (base + 255) // 256 * 256
            if arrays is None:
                graph_seeds = np.atleast_1d(np.asarray(graph_seeds, dtype=np.uint64))
                self.h = xs_create_instance(self.params, graph_seeds, run_seeds, self._ws_ptr,
                                            self.ws_bytes, stream)
            else:
                tri, jbit, order, set_size, n_sets = arrays
                self.h = xs_create_instance_from_arrays(self.params, tri, jbit, order, set_size,
                                                        n_sets, run_seeds, self._ws_ptr,
                                                        self.ws_bytes, stream)
            if geometry:
                xs_set_geometry(self.h, stream=stream, **geometry)

    def _on(self):
        import torch
        return torch.cuda.device(self.device)

    # -- calls, same names as the C ABI ------------------------------------------------------
    def run_sweeps(self, n_sweeps: int, stream=None):
        with self._on():
            xs_run_sweeps(self.h, n_sweeps, stream)

    def set_flip_table(self, thr4, stream=None):
        with self._on():
            xs_set_flip_table(self.h, thr4, stream)

    def set_geometry(self, stream=None, **geometry):
        """xs_set_geometry: variant=, tile_words=, threads=, words_per_lane=, batch_sweeps=, noise_sweeps=."""
        with self._on():
            xs_set_geometry(self.h, stream=stream, **geometry)

    def energy(self, stream=None):
        import torch
        with self._on():
            out = torch.empty((self.n_instances, 64 * self.W), dtype=torch.int32, device=self.device)
            xs_energy(self.h, out.data_ptr(), stream)
        return out

    def tts(self, stream=None):
        with self._on():
            return xs_tts(self.h, self.n_instances, stream)

    def get_spins(self, stream=None):
        import torch
        with self._on():
            out = torch.empty((self.n_instances, self.N, self.W), dtype=torch.int64, device=self.device)
            xs_get_spins(self.h, out.data_ptr(), stream)
        return out

    def set_spins(self, x, stream=None):
        assert x.is_cuda and x.is_contiguous() and x.numel() == self.n_instances * self.N * self.W
        assert x.device == self.device, "set_spins: tensor lives on another device"
        with self._on():
            xs_set_spins(self.h, x.data_ptr(), stream)

    def get_first_hit(self, stream=None):
        import torch
        with self._on():
            out = torch.empty((self.n_instances, 64 * self.W), dtype=torch.int32, device=self.device)
            xs_get_first_hit(self.h, out.data_ptr(), stream)
        return out

    def solved_mask_static(self, out=None, stream=None):
        """xs_solved_mask_static into `out` (int64 [instances][W], caller-owned; allocated here if None)."""
        import torch
        with self._on():
            if out is None:
                out = torch.empty((self.n_instances, self.W), dtype=torch.int64, device=self.device)
            assert out.is_cuda and out.is_contiguous() and out.numel() == self.n_instances * self.W
            xs_solved_mask_static(self.h, out.data_ptr(), stream)
        return out

    def get_graph(self, inst: int = 0):
        return xs_get_graph(self.h, inst, self.N)

    def layout(self):
        return xs_get_layout(self.h)

    # numpy views for tests / reports (uint64 words, uint32 first hits)
    def spins_numpy(self) -> np.ndarray:
        return self.get_spins().cpu().numpy().view(np.uint64)

    def first_hit_numpy(self) -> np.ndarray:
        return self.get_first_hit().cpu().numpy().view(np.uint32)

    def close(self):
        if getattr(self, "h", None) is not None:
            xs_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
