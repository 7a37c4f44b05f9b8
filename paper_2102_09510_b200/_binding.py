"""ctypes binding of libxs_b200.so (include/xs.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used for device memory
and streams.  There is no CPU fallback: if the shared library cannot be loaded, importing the
symbols raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

XS_OK, XS_EINVAL, XS_ENOMEM, XS_ECUDA, XS_ESTATE = 0, -1, -2, -3, -4
XS_NO_HIT = 0xFFFFFFFF
XS_FLAG_GAUGE, XS_FLAG_NO_SKIP, XS_FLAG_STREAMING, XS_FLAG_BALANCED, XS_FLAG_CLONE_NOISE = 1, 2, 4, 8, 16
XS_W1_THRESHOLD_DEFAULT = 236223201


class xs_params(C.Structure):
    _fields_ = [("n_spins", C.c_uint32), ("n_words", C.c_uint32), ("n_instances", C.c_uint32),
                ("set_cap", C.c_uint32), ("w1_threshold", C.c_uint32), ("flags", C.c_uint32)]


class xs_tts_rec(C.Structure):
    _fields_ = [("solved", C.c_uint32), ("tts_sweeps", C.c_uint32), ("clone", C.c_uint32),
                ("_pad", C.c_uint32), ("sweeps_done", C.c_uint64)]


class xs_layout(C.Structure):
    _fields_ = [("regime", C.c_uint32), ("tile_words", C.c_uint32), ("threads", C.c_uint32),
                ("ctas", C.c_uint32), ("smem_bytes", C.c_uint32), ("batch_sweeps", C.c_uint32),
                ("n_sets_max", C.c_uint32), ("variant", C.c_uint32)]


class xs_geometry(C.Structure):
    _fields_ = [("variant", C.c_uint32), ("tile_words", C.c_uint32), ("threads", C.c_uint32),
                ("words_per_lane", C.c_uint32), ("batch_sweeps", C.c_uint32), ("noise_sweeps", C.c_uint32)]


XS_GEOM_AUTO = 0xFFFFFFFF

EXPORTS = ["xs_workspace_bytes", "xs_create_instance", "xs_create_instance_from_arrays",
           "xs_run_sweeps", "xs_set_flip_table", "xs_set_geometry", "xs_energy", "xs_tts", "xs_get_spins", "xs_set_spins",
           "xs_get_first_hit", "xs_get_graph", "xs_generate_graph", "xs_clause_placement", "xs_get_layout", "xs_tts_stats",
           "xs_cavity_barrier", "xs_alu_peak", "xs_kernel_launches", "xs_solved_mask_static", "xs_destroy",
           "xs_last_error"]

_lib = None


def lib():
    """Loads (building first if the sources are newer) the C-ABI library.  Raises if unavailable."""
    global _lib
    if _lib is not None:
        return _lib
    so = _build.SO
    if _build.needs_build():
        so = _build.build()
    L = C.CDLL(so)
    vp, u32p, u64p, u8p = C.c_void_p, C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_uint8)
    pp = C.POINTER(xs_params)
    L.xs_workspace_bytes.argtypes = [pp, C.POINTER(C.c_size_t)]
    L.xs_create_instance.argtypes = [C.POINTER(vp), pp, u64p, u64p, vp, C.c_size_t, vp]
    L.xs_create_instance_from_arrays.argtypes = [C.POINTER(vp), pp, u32p, u8p, u32p, u32p, u32p,
                                                 C.c_uint32, u64p, vp, C.c_size_t, vp]
    L.xs_run_sweeps.argtypes = [vp, C.c_uint64, vp]
    L.xs_set_flip_table.argtypes = [vp, u64p, vp]
    L.xs_set_geometry.argtypes = [vp, C.POINTER(xs_geometry), vp]
    L.xs_energy.argtypes = [vp, vp, vp]
    L.xs_tts.argtypes = [vp, C.POINTER(xs_tts_rec), vp]
    L.xs_get_spins.argtypes = [vp, vp, vp]
    L.xs_set_spins.argtypes = [vp, vp, vp]
    L.xs_get_first_hit.argtypes = [vp, vp, vp]
    L.xs_get_graph.argtypes = [vp, C.c_uint32, u32p, u8p, u32p, u32p, u32p]
    L.xs_generate_graph.argtypes = [C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32, u32p, u8p, u32p,
                                    u32p, u32p, C.POINTER(C.c_int32)]
    L.xs_clause_placement.argtypes = [C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, u32p, u32p, u32p, u32p]
    L.xs_get_layout.argtypes = [vp, C.POINTER(xs_layout)]
    L.xs_tts_stats.argtypes = [u32p, C.c_uint32, C.c_uint64, C.POINTER(C.c_double)]
    L.xs_cavity_barrier.argtypes = [C.c_uint32, C.c_double, C.POINTER(C.c_double)]
    L.xs_solved_mask_static.argtypes = [vp, vp, vp]
    L.xs_destroy.argtypes = [vp]
    L.xs_alu_peak.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
    L.xs_kernel_launches.argtypes = []
    L.xs_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("xs_last_error", "xs_kernel_launches"):
            getattr(L, name).restype = C.c_int
    L.xs_kernel_launches.restype = C.c_uint64
    _lib = L
    return L


class XsError(RuntimeError):
    def __init__(self, code: int, where: str):
        msg = lib().xs_last_error()
        super().__init__(f"{where} failed with code {code}: {msg.decode() if msg else ''}")
        self.code = code


def _check(rc: int, where: str):
    if rc != XS_OK:
        raise XsError(rc, where)


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _ptr(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def _stream(stream):
    """cudaStream_t of a torch stream (None -> torch's current stream on the current device)."""
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def make_params(n_spins, n_words, n_instances=1, set_cap=0, w1_threshold=XS_W1_THRESHOLD_DEFAULT,
                flags=XS_FLAG_GAUGE) -> xs_params:
    return xs_params(int(n_spins), int(n_words), int(n_instances), int(set_cap), int(w1_threshold),
                     int(flags))


# ---- the C calls, same names ------------------------------------------------------------------
def xs_workspace_bytes(params: xs_params) -> int:
    n = C.c_size_t(0)
    _check(lib().xs_workspace_bytes(C.byref(params), C.byref(n)), "xs_workspace_bytes")
    return int(n.value)


def xs_create_instance(params: xs_params, graph_seeds, run_seeds, dev_ws_ptr: int, ws_bytes: int,
                       stream=None) -> C.c_void_p:
    gs, rs = _np(graph_seeds, np.uint64), _np(run_seeds, np.uint64)
    assert gs.size == params.n_instances and rs.size == params.n_instances
    h = C.c_void_p()
    _check(lib().xs_create_instance(C.byref(h), C.byref(params), _ptr(gs, C.c_uint64),
                                    _ptr(rs, C.c_uint64), C.c_void_p(dev_ws_ptr), ws_bytes,
                                    _stream(stream)), "xs_create_instance")
    return h


def xs_create_instance_from_arrays(params: xs_params, tri, jbit, order, set_size, n_sets, run_seeds,
                                   dev_ws_ptr: int, ws_bytes: int, stream=None) -> C.c_void_p:
    I, N = params.n_instances, params.n_spins
    tri = _np(tri, np.uint32).reshape(I, N, 3)
    jbit = _np(jbit, np.uint8).reshape(I, N)
    order = _np(order, np.uint32).reshape(I, N)
    n_sets = _np(n_sets, np.uint32).reshape(I)
    set_size = _np(set_size, np.uint32).reshape(I, -1)
    rs = _np(run_seeds, np.uint64).reshape(I)
    h = C.c_void_p()
    _check(lib().xs_create_instance_from_arrays(
        C.byref(h), C.byref(params), _ptr(tri, C.c_uint32), _ptr(jbit, C.c_uint8),
        _ptr(order, C.c_uint32), _ptr(set_size, C.c_uint32), _ptr(n_sets, C.c_uint32),
        set_size.shape[1], _ptr(rs, C.c_uint64), C.c_void_p(dev_ws_ptr), ws_bytes, _stream(stream)),
        "xs_create_instance_from_arrays")
    return h


def xs_run_sweeps(h, n_sweeps: int, stream=None):
    _check(lib().xs_run_sweeps(h, int(n_sweeps), _stream(stream)), "xs_run_sweeps")


def xs_set_flip_table(h, thr4, stream=None):
    t = _np(thr4, np.uint64)
    assert t.size == 4
    _check(lib().xs_set_flip_table(h, _ptr(t, C.c_uint64), _stream(stream)), "xs_set_flip_table")


def xs_set_geometry(h, variant=None, tile_words=0, threads=0, words_per_lane=0, batch_sweeps=0,
                    noise_sweeps=0, stream=None):
    """Explicit launch geometry (include/xs.h xs_geometry); all defaults = the library's rule."""
    g = xs_geometry(XS_GEOM_AUTO if variant is None else int(variant), int(tile_words), int(threads),
                    int(words_per_lane), int(batch_sweeps), int(noise_sweeps))
    _check(lib().xs_set_geometry(h, C.byref(g), _stream(stream)), "xs_set_geometry")


def xs_energy(h, dev_out_ptr: int, stream=None):
    _check(lib().xs_energy(h, C.c_void_p(dev_out_ptr), _stream(stream)), "xs_energy")


def xs_tts(h, n_instances: int, stream=None):
    recs = (xs_tts_rec * n_instances)()
    _check(lib().xs_tts(h, recs, _stream(stream)), "xs_tts")
    return recs


def xs_get_spins(h, dev_out_ptr: int, stream=None):
    _check(lib().xs_get_spins(h, C.c_void_p(dev_out_ptr), _stream(stream)), "xs_get_spins")


def xs_set_spins(h, dev_in_ptr: int, stream=None):
    _check(lib().xs_set_spins(h, C.c_void_p(dev_in_ptr), _stream(stream)), "xs_set_spins")


def xs_get_first_hit(h, dev_out_ptr: int, stream=None):
    _check(lib().xs_get_first_hit(h, C.c_void_p(dev_out_ptr), _stream(stream)), "xs_get_first_hit")


def xs_get_graph(h, inst: int, n_spins: int):
    tri = np.zeros((n_spins, 3), np.uint32)
    jbit = np.zeros(n_spins, np.uint8)
    order = np.zeros(n_spins, np.uint32)
    ss = np.zeros(n_spins, np.uint32)
    ns = C.c_uint32(0)
    _check(lib().xs_get_graph(h, inst, _ptr(tri, C.c_uint32), _ptr(jbit, C.c_uint8),
                              _ptr(order, C.c_uint32), _ptr(ss, C.c_uint32), C.byref(ns)),
           "xs_get_graph")
    return tri, jbit, order, ss[: ns.value].copy()


def xs_generate_graph(n_spins: int, graph_seed: int, flags: int = XS_FLAG_GAUGE, set_cap: int = 0):
    """Host only.  Returns (tri, jbit, order, set_size, attempt)."""
    tri = np.zeros((n_spins, 3), np.uint32)
    jbit = np.zeros(n_spins, np.uint8)
    order = np.zeros(n_spins, np.uint32)
    ss = np.zeros(n_spins, np.uint32)
    ns, att = C.c_uint32(0), C.c_int32(-1)
    _check(lib().xs_generate_graph(n_spins, int(graph_seed), int(flags), int(set_cap),
                                   _ptr(tri, C.c_uint32), _ptr(jbit, C.c_uint8),
                                   _ptr(order, C.c_uint32), _ptr(ss, C.c_uint32), C.byref(ns),
                                   C.byref(att)), "xs_generate_graph")
    return tri, jbit, order, ss[: ns.value].copy(), int(att.value)


def xs_clause_placement(n_spins: int, graph_seed: int, n_slots: int, flags: int = XS_FLAG_GAUGE | XS_FLAG_BALANCED,
                        set_cap: int = 0):
    """Host only.  Returns (task [rounds * n_slots][4], place [N], barrier_mask) of the clause-word
    kernel (include/xs.h)."""
    task = np.zeros((2 * n_spins, 4), np.uint32)
    place = np.zeros(n_spins, np.uint32)
    nr, bm = C.c_uint32(0), C.c_uint32(0)
    _check(lib().xs_clause_placement(n_spins, int(graph_seed), int(flags), int(set_cap), int(n_slots),
                                     _ptr(task, C.c_uint32), _ptr(place, C.c_uint32), C.byref(nr), C.byref(bm)),
           "xs_clause_placement")
    return task[: nr.value * n_slots].copy(), place, int(bm.value)


def xs_get_layout(h) -> xs_layout:
    out = xs_layout()
    _check(lib().xs_get_layout(h, C.byref(out)), "xs_get_layout")
    return out


def xs_tts_stats(tts, t_max: int) -> dict:
    t = _np(tts, np.uint32)
    out = (C.c_double * 12)()
    _check(lib().xs_tts_stats(_ptr(t, C.c_uint32), t.size, int(t_max), out), "xs_tts_stats")
    keys = ["n_solved", "t_tot", "tau_hat", "tts50_model", "tts90_model", "tts99_model",
            "tts50_emp", "tts90_emp", "tts99_emp", "tau_q16", "tau_q50", "tau_q84"]
    return dict(zip(keys, [float(v) for v in out]))


def xs_cavity_barrier(K: int, T: float) -> dict:
    """PAPER.md Eqs. (3)-(4): cavity free-energy barrier of the K-spin model at temperature T."""
    out = (C.c_double * 6)()
    _check(lib().xs_cavity_barrier(int(K), float(T), out), "xs_cavity_barrier")
    keys = ["barrier", "m_barrier", "h_barrier", "T_sp", "ferro_bdf", "m_ferro"]
    return dict(zip(keys, [float(v) for v in out]))


def xs_alu_peak(stream=None):
    """(lane-ops per ns of the whole GPU, kernel ms) from the LOP3 micro-kernel."""
    v, ms = C.c_double(0), C.c_double(0)
    _check(lib().xs_alu_peak(C.byref(v), C.byref(ms), _stream(stream)), "xs_alu_peak")
    return float(v.value), float(ms.value)


XS_STATIC_MAX_WORDS = 65536


def xs_solved_mask_static(h, dev_mask_ptr: int, stream=None):
    """Allocation-free ground-state mask (include/xs.h): static scratch inside the library."""
    _check(lib().xs_solved_mask_static(h, C.c_void_p(dev_mask_ptr), _stream(stream)), "xs_solved_mask_static")


def xs_kernel_launches() -> int:
    return int(lib().xs_kernel_launches())


def xs_destroy(h):
    _check(lib().xs_destroy(h), "xs_destroy")
