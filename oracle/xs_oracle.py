"""ctypes front end of the CPU oracle (oracle/xs_oracle.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this.  It holds no arithmetic of the method: every step is a call into xs_oracle.c,
which follows PAPER.md step by step (see the header of that file for the citations).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "xs_oracle.c")
_SO = os.path.join(_HERE, "libxs_oracle.so")

W1_THRESHOLD = 236223201  # floor(0.055 * 2**32), DESIGN.md R-thr (w1 = 0.055)
NO_HIT = 0xFFFFFFFF


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        u32p, u8p, i8p, u64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_uint8),
                                C.POINTER(C.c_int8), C.POINTER(C.c_uint64))
        L.xso_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.xso_gen_triplets.argtypes = [C.c_uint32, C.c_uint64, C.c_uint32, u32p]
        L.xso_gen_triplets.restype = C.c_int
        L.xso_gen_gauge.argtypes = [C.c_uint32, C.c_uint64, u8p]
        L.xso_couplings_from_gauge.argtypes = [C.c_uint32, u32p, u8p, u8p]
        L.xso_adjacency.argtypes = [C.c_uint32, u32p, u32p, u32p]
        L.xso_adjacency.restype = C.c_int
        L.xso_update_order.argtypes = [C.c_uint32, u32p, C.c_uint32, u32p, u32p]
        L.xso_update_order.restype = C.c_int
        L.xso_balanced_order.argtypes = [C.c_uint32, u32p, C.c_uint64, C.c_uint32, C.c_uint32,
                                         u32p, u32p]
        L.xso_balanced_order.restype = C.c_int
        L.xso_check_order.argtypes = [C.c_uint32, u32p, u32p, u32p, C.c_uint32]
        L.xso_check_order.restype = C.c_int
        L.xso_init_spins.argtypes = [C.c_uint32, C.c_uint32, C.c_uint64, i8p]
        L.xso_energy.argtypes = [C.c_uint32, u32p, u8p, i8p]
        L.xso_energy.restype = C.c_int32
        L.xso_sweep.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, u32p, u8p, u32p, u32p,
                                u32p, u32p, C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32,
                                C.c_int, C.c_int, i8p, u64p, u64p]
        L.xso_mark_initial.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, u32p, u8p, i8p,
                                       u32p]
        run_args = [C.c_uint32, C.c_uint32, C.c_uint32, u32p, u8p, u32p, u32p, u32p, u32p,
                    C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, i8p, u32p]
        L.xso_run.argtypes = run_args
        L.xso_run_omp.argtypes = run_args
        # general flip table w_0..w_3: thresholds in [0, 2^32] as uint64[4]
        L.xso_sweep_w.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, u32p, u8p, u32p, u32p,
                                  u32p, u32p, C.c_uint32, C.c_uint64, C.c_uint32, u64p,
                                  C.c_int, C.c_int, i8p, u64p, u64p]
        L.xso_run_w.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, u32p, u8p, u32p, u32p, u32p,
                                u32p, C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32, u64p, i8p, u32p]
        # per-clone noise variant
        L.xso_sweep_clone.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, u8p, u32p, u32p, u32p,
                                      C.c_uint64, C.c_uint32, C.c_uint32, i8p]
        L.xso_run_clone.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, u32p, u8p, u32p, u32p, u32p,
                                    C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, i8p, u32p]
        L.xso_pack.argtypes = [C.c_uint32, C.c_uint32, i8p, u64p]
        L.xso_unpack.argtypes = [C.c_uint32, C.c_uint32, u64p, i8p]
        L.xso_omp_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def philox(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    o = np.zeros(4, dtype=np.uint32)
    lib().xso_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(o, C.c_uint32))
    return o


def omp_threads() -> int:
    return int(lib().xso_omp_threads())


class Instance:
    """One problem instance: triplets, couplings, adjacency, update order (a-1 of DESIGN.md)."""

    def __init__(self, n_spins: int, graph_seed: int, gauge: bool = True, set_cap: int = 0,
                 tri=None, jbit=None, balanced: bool = False):
        L = lib()
        N = int(n_spins)
        self.N = N
        self.graph_seed = int(graph_seed)
        if tri is None:
            self.tri = np.zeros((N, 3), dtype=np.uint32)
            self.attempt = L.xso_gen_triplets(N, self.graph_seed, 100000, _p(self.tri, C.c_uint32))
            if self.attempt < 0:
                raise RuntimeError("xso_gen_triplets failed")
        else:
            self.tri = np.ascontiguousarray(tri, dtype=np.uint32).reshape(N, 3)
            self.attempt = -1
        self.taubit = np.zeros(N, dtype=np.uint8)
        if jbit is not None:
            self.jbit = np.ascontiguousarray(jbit, dtype=np.uint8)
        elif gauge:
            L.xso_gen_gauge(N, self.graph_seed, _p(self.taubit, C.c_uint8))
            self.jbit = np.zeros(N, dtype=np.uint8)
            L.xso_couplings_from_gauge(N, _p(self.tri, C.c_uint32), _p(self.taubit, C.c_uint8),
                                       _p(self.jbit, C.c_uint8))
        else:
            self.jbit = np.zeros(N, dtype=np.uint8)
        self.nbr = np.zeros((N, 6), dtype=np.uint32)
        self.cls = np.zeros((N, 3), dtype=np.uint32)
        if L.xso_adjacency(N, _p(self.tri, C.c_uint32), _p(self.nbr, C.c_uint32),
                           _p(self.cls, C.c_uint32)) != 0:
            raise RuntimeError("not a 3-regular hypergraph")
        self.order = np.zeros(N, dtype=np.uint32)
        ss = np.zeros(N, dtype=np.uint32)
        self.n_sets = 0
        if balanced and N <= 8192:
            # DESIGN.md R-balance: q = max(4, ceil(N / S)) sets, S = set_cap or, by default, the
            # largest of 16, 32, 64, 128, 256 with S <= N / 4 (16 if there is none);
            # 1000 + 200 N tabu steps; N > 8192 or a failed search: the greedy order below
            S = int(set_cap)
            if S == 0:
                S = 16
                while S < 256 and 2 * S <= N // 4:
                    S *= 2
            q = max(4, (N + S - 1) // S)
            self.n_sets = L.xso_balanced_order(N, _p(self.nbr, C.c_uint32), self.graph_seed, q,
                                               1000 + 200 * N, _p(self.order, C.c_uint32),
                                               _p(ss, C.c_uint32))
        self.balanced = self.n_sets > 0
        if not self.balanced:
            self.n_sets = L.xso_update_order(N, _p(self.nbr, C.c_uint32), int(set_cap),
                                             _p(self.order, C.c_uint32), _p(ss, C.c_uint32))
        if self.n_sets < 0:
            raise RuntimeError("xso_update_order failed")
        self.set_size = ss[: self.n_sets].copy()
        if not self.check_order():
            raise RuntimeError("update order is not a sequence of anti-cliques")

    def check_order(self, order=None, set_size=None) -> bool:
        order = self.order if order is None else np.ascontiguousarray(order, dtype=np.uint32)
        ss = self.set_size if set_size is None else np.ascontiguousarray(set_size, dtype=np.uint32)
        return bool(lib().xso_check_order(self.N, _p(self.nbr, C.c_uint32), _p(order, C.c_uint32),
                                          _p(ss, C.c_uint32), len(ss)))

    # --- clone states: int8 [64W][N] ------------------------------------------------------
    def init_spins(self, W: int, run_seed: int) -> np.ndarray:
        s = np.zeros((64 * W, self.N), dtype=np.int8)
        lib().xso_init_spins(self.N, W, int(run_seed), _p(s, C.c_int8))
        return s

    def energy(self, s: np.ndarray) -> np.ndarray:
        s = np.ascontiguousarray(s, dtype=np.int8).reshape(-1, self.N)
        L = lib()
        return np.array([L.xso_energy(self.N, _p(self.tri, C.c_uint32), _p(self.jbit, C.c_uint8),
                                      _p(s[c], C.c_int8)) for c in range(s.shape[0])],
                        dtype=np.int32)

    def sweep(self, s, run_seed, t, w_begin=0, w_end=None, thr=W1_THRESHOLD, mode=0,
              check_dE=False, order=None, set_size=None, thr4=None):
        """One sweep number t (in place).  Returns (n_flips, dE_mismatches).
        thr4: general flip table (4 thresholds in [0, 2^32]); default = quasi-greedy with `thr`."""
        assert s.dtype == np.int8 and s.flags.c_contiguous
        W = s.shape[0] // 64
        w_end = W if w_end is None else w_end
        order = self.order if order is None else np.ascontiguousarray(order, dtype=np.uint32)
        ss = self.set_size if set_size is None else np.ascontiguousarray(set_size, dtype=np.uint32)
        nf, mm = C.c_uint64(0), C.c_uint64(0)
        if thr4 is not None:
            t4 = np.ascontiguousarray(thr4, dtype=np.uint64)
            lib().xso_sweep_w(self.N, w_begin, w_end, _p(self.tri, C.c_uint32),
                              _p(self.jbit, C.c_uint8), _p(self.nbr, C.c_uint32),
                              _p(self.cls, C.c_uint32), _p(order, C.c_uint32), _p(ss, C.c_uint32),
                              len(ss), int(run_seed), int(t), _p(t4, C.c_uint64), int(mode),
                              int(bool(check_dE)), _p(s, C.c_int8), C.byref(nf), C.byref(mm))
            return nf.value, mm.value
        lib().xso_sweep(self.N, w_begin, w_end, _p(self.tri, C.c_uint32), _p(self.jbit, C.c_uint8),
                        _p(self.nbr, C.c_uint32), _p(self.cls, C.c_uint32),
                        _p(order, C.c_uint32), _p(ss, C.c_uint32), len(ss), int(run_seed),
                        int(t), int(thr), int(mode), int(bool(check_dE)), _p(s, C.c_int8),
                        C.byref(nf), C.byref(mm))
        return nf.value, mm.value

    def mark_initial(self, s, w_begin=0, w_end=None) -> np.ndarray:
        W = s.shape[0] // 64
        w_end = W if w_end is None else w_end
        fh = np.full(64 * W, NO_HIT, dtype=np.uint32)
        lib().xso_mark_initial(self.N, w_begin, w_end, _p(self.tri, C.c_uint32),
                               _p(self.jbit, C.c_uint8), _p(s, C.c_int8), _p(fh, C.c_uint32))
        return fh

    def sweep_clone(self, s, run_seed, t, m, w_begin=0, w_end=None):
        """One sweep of the per-clone noise variant (w1 = m / 128), in place."""
        assert s.dtype == np.int8 and s.flags.c_contiguous
        w_end = s.shape[0] // 64 if w_end is None else w_end
        lib().xso_sweep_clone(self.N, w_begin, w_end, _p(self.jbit, C.c_uint8),
                              _p(self.nbr, C.c_uint32), _p(self.cls, C.c_uint32),
                              _p(self.order, C.c_uint32), int(run_seed), int(t), int(m),
                              _p(s, C.c_int8))

    def run(self, s, first_hit, run_seed, t_begin, n_sweeps, w_begin=0, w_end=None,
            thr=W1_THRESHOLD, omp=False, thr4=None, clone_m=None):
        """Sweeps t_begin+1 .. t_begin+n_sweeps in place, maintaining first_hit."""
        assert s.dtype == np.int8 and s.flags.c_contiguous
        assert first_hit.dtype == np.uint32 and first_hit.flags.c_contiguous
        W = s.shape[0] // 64
        w_end = W if w_end is None else w_end
        if clone_m is not None:
            lib().xso_run_clone(self.N, w_begin, w_end, _p(self.tri, C.c_uint32),
                                _p(self.jbit, C.c_uint8), _p(self.nbr, C.c_uint32),
                                _p(self.cls, C.c_uint32), _p(self.order, C.c_uint32),
                                int(run_seed), int(t_begin), int(n_sweeps), int(clone_m),
                                _p(s, C.c_int8), _p(first_hit, C.c_uint32))
            return
        if thr4 is not None:
            t4 = np.ascontiguousarray(thr4, dtype=np.uint64)
            lib().xso_run_w(self.N, w_begin, w_end, _p(self.tri, C.c_uint32),
                            _p(self.jbit, C.c_uint8), _p(self.nbr, C.c_uint32),
                            _p(self.cls, C.c_uint32), _p(self.order, C.c_uint32),
                            _p(self.set_size, C.c_uint32), self.n_sets, int(run_seed),
                            int(t_begin), int(n_sweeps), _p(t4, C.c_uint64), _p(s, C.c_int8),
                            _p(first_hit, C.c_uint32))
            return
        fn = lib().xso_run_omp if omp else lib().xso_run
        fn(self.N, w_begin, w_end, _p(self.tri, C.c_uint32), _p(self.jbit, C.c_uint8),
           _p(self.nbr, C.c_uint32), _p(self.cls, C.c_uint32), _p(self.order, C.c_uint32),
           _p(self.set_size, C.c_uint32), self.n_sets, int(run_seed), int(t_begin),
           int(n_sweeps), int(thr), _p(s, C.c_int8), _p(first_hit, C.c_uint32))

    # --- conversion to the boundary's layout: uint64 x[N][W] ---------------------------------
    def pack(self, s) -> np.ndarray:
        W = s.shape[0] // 64
        x = np.zeros((self.N, W), dtype=np.uint64)
        lib().xso_pack(self.N, W, _p(np.ascontiguousarray(s), C.c_int8), _p(x, C.c_uint64))
        return x

    def unpack(self, x) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.uint64).reshape(self.N, -1)
        W = x.shape[1]
        s = np.zeros((64 * W, self.N), dtype=np.int8)
        lib().xso_unpack(self.N, W, _p(x, C.c_uint64), _p(s, C.c_int8))
        return s
