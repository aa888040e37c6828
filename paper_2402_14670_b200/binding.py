"""Thin ctypes binding over the C ABI of ``include/lf.h`` (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of ``liblf_b200.so``; PyTorch is used for device
memory and streams only.  There is no CPU fallback: if the library is missing or no CUDA device is
present the constructor raises.
"""
from __future__ import annotations

import ctypes as C
import os
from types import SimpleNamespace
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblf_b200.so")
NL = 12

LF_OK, LF_ERR_INVALID_ARG, LF_ERR_CUDA, LF_ERR_CAPACITY, LF_ERR_UNSUPPORTED = range(5)
_STATUS = {0: "LF_OK", 1: "LF_ERR_INVALID_ARG", 2: "LF_ERR_CUDA", 3: "LF_ERR_CAPACITY", 4: "LF_ERR_UNSUPPORTED"}


class LfError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status


class lf_geometry(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("z", C.c_float * NL), ("tan_alpha", C.c_float * NL),
                ("z_seed", C.c_float), ("z_mag", C.c_float), ("kick", C.c_float),
                ("z_ref", C.c_float), ("d_ratio", C.c_float),
                ("k_first", C.c_float), ("k_last", C.c_float), ("qop_poly", C.c_float * 5),
                ("x_half", C.c_float), ("y_half", C.c_float), ("z_state", C.c_float),
                ("polarity", C.c_int32), ("qop_mode", C.c_int32), ("qop_poly2d", (C.c_float * 10) * 5)]


class lf_params(C.Structure):
    _fields_ = [("T_triplet", C.c_float), ("T_x", C.c_float), ("T_uv_slope", C.c_float),
                ("T_uv_min", C.c_float), ("T_ty", C.c_float), ("T_y", C.c_float), ("T_Q", C.c_float),
                ("C_nhits", C.c_float * 4),
                ("n_window", C.c_int32), ("n_triplets", C.c_int32), ("min_hits", C.c_int32),
                ("xtol_base", C.c_float), ("xtol_inv_p", C.c_float), ("x_asym", C.c_float),
                ("uv_half_width", C.c_float),
                ("p_same_bend", C.c_float), ("mag_tol_base", C.c_float), ("mag_tol_inv_p", C.c_float),
                ("mag_tol_tx", C.c_float), ("mag_tol_max", C.c_float),
                ("hit_storage", C.c_int32),
                ("mode", C.c_int32), ("velo_p_min", C.c_float), ("velo_pt_min", C.c_float),
                ("xtol_poly", C.c_float * 8), ("x_overlap", C.c_float), ("seed_arith", C.c_int32)]


class lf_seeds(C.Structure):
    _fields_ = [("x", C.c_void_p), ("y", C.c_void_p), ("tx", C.c_void_p), ("ty", C.c_void_p),
                ("qop", C.c_void_p), ("event_offsets", C.c_void_p), ("n_seeds", C.c_size_t)]


class lf_hits(C.Structure):
    _fields_ = [("x", C.c_void_p), ("seg_offsets", C.c_void_p), ("n_hits", C.c_size_t),
                ("x16", C.c_void_p), ("origin16", C.c_void_p)]


class lf_tracks(C.Structure):
    _fields_ = [("hit_idx", C.c_void_p), ("seed_idx", C.c_void_p), ("n_hits", C.c_void_p),
                ("state", C.c_void_p), ("quality", C.c_void_p), ("event_offsets", C.c_void_p),
                ("n_tracks", C.c_void_p), ("capacity", C.c_size_t)]


class lf_debug(C.Structure):
    _fields_ = [("win_first", C.c_void_p), ("win_count", C.c_void_p), ("n_triplets", C.c_void_p),
                ("trip_hits", C.c_void_p), ("trip_set", C.c_void_p), ("trip_chi2", C.c_void_p),
                ("cand_hits", C.c_void_p), ("cand_quality", C.c_void_p)]


class lf_info(C.Structure):
    _fields_ = [("kernels_per_run", C.c_int32), ("regs", C.c_int32 * 4), ("block", C.c_int32 * 4),
                ("grid", C.c_int32 * 4), ("ctas_per_sm", C.c_int32 * 4), ("smem_bytes", C.c_int32 * 4),
                ("staged_hits_per_event", C.c_int32), ("sm_count", C.c_int32), ("workspace_bytes", C.c_size_t)]


KERNEL_NAMES = ("window", "seed", "extend", "fit")
N_COUNTERS = 8
COUNTER_NAMES = ("accepted_candidates", "events_with_equal_hits", "window_hits", "doublets_evaluated", "doublets_passing",
                 "triplets_passing", "triplets_kept", "tracks")
EVENT_KERNELS = KERNEL_NAMES[:4]


_STRUCTS = (lf_geometry, lf_params, lf_seeds, lf_hits, lf_tracks, lf_debug, lf_info)
_lib: Optional[C.CDLL] = None


def load_library() -> C.CDLL:
    """Loads liblf_b200.so (loudly) and checks the ABI version and struct sizes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.lf_abi_version.restype = C.c_uint32
    lib.lf_sizeof.restype = C.c_size_t
    lib.lf_sizeof.argtypes = [C.c_int]
    lib.lf_last_error.restype = C.c_char_p
    lib.lf_last_error.argtypes = [C.c_void_p]
    lib.lf_create.restype = C.c_int
    lib.lf_create.argtypes = [C.POINTER(lf_geometry), C.POINTER(lf_params), C.c_size_t, C.c_size_t, C.c_size_t,
                              C.POINTER(C.c_void_p)]
    for name in ("lf_run", "lf_run_host"):
        fn = getattr(lib, name)
        fn.restype = C.c_int
        fn.argtypes = [C.c_void_p, C.POINTER(lf_seeds), C.POINTER(lf_hits), C.c_size_t, C.POINTER(lf_tracks), C.c_void_p]
    lib.lf_host_submit.restype = C.c_int
    lib.lf_host_submit.argtypes = [C.c_void_p, C.POINTER(lf_seeds), C.POINTER(lf_hits), C.c_size_t, C.POINTER(lf_tracks),
                                   C.c_void_p, C.c_int]
    lib.lf_host_collect.restype = C.c_int
    lib.lf_host_collect.argtypes = [C.c_void_p, C.c_int]
    lib.lf_validate_inputs.restype = C.c_int
    lib.lf_validate_inputs.argtypes = [C.c_void_p, C.POINTER(lf_seeds), C.POINTER(lf_hits), C.c_size_t, C.c_void_p]
    lib.lf_run_debug.restype = C.c_int
    lib.lf_run_debug.argtypes = [C.c_void_p, C.POINTER(lf_seeds), C.POINTER(lf_hits), C.c_size_t, C.POINTER(lf_tracks),
                                 C.POINTER(lf_debug), C.c_void_p]
    lib.lf_destroy.restype = C.c_int
    lib.lf_destroy.argtypes = [C.c_void_p]
    lib.lf_get_info.restype = C.c_int
    lib.lf_get_info.argtypes = [C.c_void_p, C.POINTER(lf_info)]
    lib.lf_set_host_chunk_events.restype = C.c_int
    lib.lf_set_host_chunk_events.argtypes = [C.c_void_p, C.c_size_t]
    lib.lf_origin_slots.restype = C.c_size_t
    lib.lf_origin_slots.argtypes = [C.c_size_t, C.c_size_t]
    lib.lf_pack_hits.restype = C.c_int
    lib.lf_pack_hits.argtypes = [C.c_void_p, C.POINTER(lf_hits), C.c_size_t, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.lf_run_counters.restype = C.c_int
    lib.lf_run_counters.argtypes = [C.c_void_p, C.POINTER(C.c_uint64 * N_COUNTERS)]
    lib.lf_set_profiling.restype = C.c_int
    lib.lf_set_profiling.argtypes = [C.c_void_p, C.c_int]
    lib.lf_kernel_times.restype = C.c_int
    lib.lf_kernel_times.argtypes = [C.c_void_p, C.POINTER(C.c_float * len(KERNEL_NAMES))]
    lib.lf_windows_static.restype = C.c_int
    lib.lf_windows_static.argtypes = [C.POINTER(lf_geometry), C.POINTER(lf_params), C.POINTER(lf_seeds), C.POINTER(lf_hits),
                                      C.c_size_t, C.c_void_p, C.c_void_p, C.c_void_p]
    if lib.lf_abi_version() != 7:
        raise ImportError("liblf_b200.so: ABI version mismatch")
    for i, st in enumerate(_STRUCTS):
        if lib.lf_sizeof(i) != C.sizeof(st):
            raise ImportError(f"liblf_b200.so: sizeof({st.__name__}) mismatch ({lib.lf_sizeof(i)} vs {C.sizeof(st)})")
    _lib = lib
    return lib


def _fill(struct, values: Dict[str, object]):
    for name, ctype in struct._fields_:
        v = values[name]
        if isinstance(v, (list, tuple, np.ndarray)) and len(v) and isinstance(v[0], (list, tuple, np.ndarray)):
            setattr(struct, name, ctype(*[ctype._type_(*[float(t) for t in row]) for row in v]))
        elif isinstance(v, (list, tuple, np.ndarray)):
            setattr(struct, name, ctype(*[float(t) for t in v]))
        else:
            setattr(struct, name, v)
    return struct


STATIC_MAX_EVENTS, STATIC_MAX_ROWS = 4096, 16384  # LF_STATIC_MAX_EVENTS / LF_STATIC_MAX_ROWS of include/lf.h


def windows_static(geometry: Dict[str, object], params: Dict[str, object], db: "DeviceBatch", win_first, win_count,
                   stream=None) -> None:
    """``lf_windows_static``: the search windows of every seed of ``db``, written into the caller's two int32 CUDA
    tensors of shape (followed tracks, 12), with no handle and no device allocation anywhere in the call.

    This is the entry point for hosts that cannot call ``cudaMalloc`` once they are running (a framework that owns all of
    the GPU's memory, a latency-bound event loop): the kernel's scratch is a fixed array inside the library, so batches
    are limited to ``STATIC_MAX_EVENTS`` events and ``STATIC_MAX_ROWS`` followed tracks (``LfError`` with
    LF_ERR_CAPACITY beyond that), calls on one device must not overlap on the GPU, and the first call per device should
    be made during set-up.  The binding allocates nothing either: both outputs are the caller's.  Asynchronous on
    ``stream`` (default: torch's current stream)."""
    lib = load_library()
    g = _fill(lf_geometry(), geometry)
    p = _fill(lf_params(), params)
    seeds = lf_seeds(db.seed_x.data_ptr(), db.seed_y.data_ptr(), db.seed_tx.data_ptr(), db.seed_ty.data_ptr(),
                     db.seed_qop.data_ptr(), db.seed_offsets.data_ptr(), db.n_seeds)
    hits = db.c_hits()
    st = lib.lf_windows_static(C.byref(g), C.byref(p), C.byref(seeds), C.byref(hits), db.n_events,
                               win_first.data_ptr() if win_first is not None else None,
                               win_count.data_ptr() if win_count is not None else None, LookingForward._stream_ptr(stream))
    if st != LF_OK:
        raise LfError(st, lib.lf_last_error(None).decode())


class DeviceBatch:
    """A batch resident in HBM: torch CUDA tensors with the layout of ``datagen.Batch``."""

    def __init__(self, batch, device="cuda:0"):
        import torch
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)
        self.n_events = int(batch.n_events)
        self.n_seeds = int(batch.seed_x.shape[0])
        self.n_hits = int(batch.hit_x.shape[0])
        self.seed_x, self.seed_y = t(batch.seed_x), t(batch.seed_y)
        self.seed_tx, self.seed_ty, self.seed_qop = t(batch.seed_tx), t(batch.seed_ty), t(batch.seed_qop)
        self.seed_offsets = t(np.asarray(batch.seed_offsets, dtype=np.uint32).view(np.int32))
        self.hit_x = t(batch.hit_x)
        self.seg_offsets = t(np.asarray(batch.seg_offsets, dtype=np.uint32).view(np.int32))
        self.device = self.hit_x.device
        self.hit_x16 = None     # optional fp16 copy (LookingForward.pack_hits); with drop_fp32() the only copy
        self.origin16 = None

    def drop_fp32(self):
        """Keeps only the packed fp16 copy of the hits (hit_storage = 1 with every stage reading fp16)."""
        assert self.hit_x16 is not None, "pack the hits first"
        self.hit_x = None

    def c_hits(self) -> "lf_hits":
        p = lambda t: t.data_ptr() if t is not None else None
        return lf_hits(p(self.hit_x), self.seg_offsets.data_ptr(), self.n_hits, p(self.hit_x16), p(self.origin16))


class TrackBuffers:
    """Output arrays (torch tensors on ``device``) for ``capacity`` tracks and ``n_events`` events."""

    def __init__(self, capacity: int, n_events: int, device):
        import torch
        cap = max(int(capacity), 1)
        self.capacity = int(capacity)
        self.hit_idx = torch.empty((cap, NL), dtype=torch.int32, device=device)
        self.seed_idx = torch.empty(cap, dtype=torch.int32, device=device)
        self.n_hits = torch.empty(cap, dtype=torch.int32, device=device)
        self.state = torch.empty((cap, 5), dtype=torch.float32, device=device)
        self.quality = torch.empty(cap, dtype=torch.float32, device=device)
        self.event_offsets = torch.empty(n_events + 1, dtype=torch.int32, device=device)
        self.n_tracks = torch.zeros(1, dtype=torch.int32, device=device)

    def c_struct(self) -> lf_tracks:
        return lf_tracks(self.hit_idx.data_ptr(), self.seed_idx.data_ptr(), self.n_hits.data_ptr(),
                         self.state.data_ptr(), self.quality.data_ptr(), self.event_offsets.data_ptr(),
                         self.n_tracks.data_ptr(), self.capacity)

    def to_numpy(self) -> SimpleNamespace:
        """Synchronising read-back of the dense track list."""
        n = int(self.n_tracks.cpu()[0])
        g = lambda t: t[:n].cpu().numpy()
        return SimpleNamespace(n_tracks=n, hit_idx=g(self.hit_idx), seed_idx=g(self.seed_idx), n_hits=g(self.n_hits),
                               state=g(self.state), quality=g(self.quality),
                               event_offsets=self.event_offsets.cpu().numpy().view(np.uint32), debug=None)


class LookingForward:
    """``lf_create`` / ``lf_run`` / ``lf_destroy`` with the same names and semantics as include/lf.h."""

    def __init__(self, geometry: Dict[str, object], params: Dict[str, object], max_events: int, max_seeds: int,
                 max_hits: int):
        self._lib = load_library()
        self._h = C.c_void_p()
        self.params = dict(params)
        g = _fill(lf_geometry(), geometry)
        p = _fill(lf_params(), params)
        st = self._lib.lf_create(C.byref(g), C.byref(p), max_events, max_seeds, max_hits, C.byref(self._h))
        if st != LF_OK:
            msg = self._lib.lf_last_error(None).decode()
            self._h = C.c_void_p()
            raise LfError(st, msg)

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, st: int):
        if st != LF_OK:
            raise LfError(st, self._lib.lf_last_error(self._h).decode())

    @staticmethod
    def _stream_ptr(stream) -> Optional[int]:
        if stream is None:
            import torch
            stream = torch.cuda.current_stream()
        return C.c_void_p(stream.cuda_stream)

    def info(self) -> SimpleNamespace:
        inf = lf_info()
        self._check(self._lib.lf_get_info(self._h, C.byref(inf)))
        conv = lambda v: list(v) if hasattr(v, "__len__") else v
        return SimpleNamespace(**{n: conv(getattr(inf, n)) for n, _ in lf_info._fields_})

    def set_profiling(self, enabled: bool):
        self._check(self._lib.lf_set_profiling(self._h, 1 if enabled else 0))

    def kernel_times(self):
        """Mean (window, seed, extend, fit) milliseconds of the profiled runs; the stream must be synchronised."""
        ms = (C.c_float * len(KERNEL_NAMES))()
        self._check(self._lib.lf_kernel_times(self._h, C.byref(ms)))
        return tuple(float(v) for v in ms)

    # -- device path -----------------------------------------------------------------------------
    def run(self, db: DeviceBatch, out: Optional[TrackBuffers] = None, stream=None, debug: bool = False):
        """Enqueue the hot path for a device-resident batch; asynchronous on ``stream``."""
        if out is None:
            out = TrackBuffers(db.n_seeds, db.n_events, db.device)
        seeds = lf_seeds(db.seed_x.data_ptr(), db.seed_y.data_ptr(), db.seed_tx.data_ptr(), db.seed_ty.data_ptr(),
                         db.seed_qop.data_ptr(), db.seed_offsets.data_ptr(), db.n_seeds)
        hits = db.c_hits()
        tr = out.c_struct()
        sp = self._stream_ptr(stream)
        if not debug:
            self._check(self._lib.lf_run(self._h, C.byref(seeds), C.byref(hits), db.n_events, C.byref(tr), sp))
            return out
        import torch
        # one row per followed track: per seed, or per (seed, window side) in the no-UT mode (include/lf.h, lf_debug)
        sides = 2 if int(self.params.get("mode", 0)) == 1 else 1
        nt, ns, dev = int(self.params["n_triplets"]), max(db.n_seeds, 1) * sides, db.device
        i32 = lambda *shape: torch.full(shape, -1, dtype=torch.int32, device=dev)
        f32 = lambda *shape: torch.full(shape, -1.0, dtype=torch.float32, device=dev)
        d = SimpleNamespace(win_first=i32(ns, NL), win_count=i32(ns, NL), n_triplets=i32(ns), trip_hits=i32(ns, nt, 3),
                            trip_set=i32(ns, nt), trip_chi2=f32(ns, nt), cand_hits=i32(ns, nt, NL), cand_quality=f32(ns, nt))
        dbg = lf_debug(d.win_first.data_ptr(), d.win_count.data_ptr(), d.n_triplets.data_ptr(), d.trip_hits.data_ptr(),
                       d.trip_set.data_ptr(), d.trip_chi2.data_ptr(), d.cand_hits.data_ptr(), d.cand_quality.data_ptr())
        self._check(self._lib.lf_run_debug(self._h, C.byref(seeds), C.byref(hits), db.n_events, C.byref(tr), C.byref(dbg), sp))
        out.debug_tensors = d
        return out

    def validate_inputs(self, db: DeviceBatch, stream=None) -> None:
        """``lf_validate_inputs`` (synchronous): raises LfError naming the violated precondition."""
        seeds = lf_seeds(db.seed_x.data_ptr(), db.seed_y.data_ptr(), db.seed_tx.data_ptr(), db.seed_ty.data_ptr(),
                         db.seed_qop.data_ptr(), db.seed_offsets.data_ptr(), db.n_seeds)
        hits = db.c_hits()
        self._check(self._lib.lf_validate_inputs(self._h, C.byref(seeds), C.byref(hits), db.n_events, self._stream_ptr(stream)))

    def pack_hits(self, db: DeviceBatch, stream=None) -> DeviceBatch:
        """``lf_pack_hits``: writes the fp16 block-offset copy of ``db``'s hits into ``db.hit_x16`` / ``db.origin16``."""
        import torch
        slots = int(self._lib.lf_origin_slots(db.n_events, db.n_hits))
        db.hit_x16 = torch.empty(max(db.n_hits, 1), dtype=torch.float16, device=db.device)
        db.origin16 = torch.zeros(slots, dtype=torch.float32, device=db.device)
        hits = lf_hits(db.hit_x.data_ptr(), db.seg_offsets.data_ptr(), db.n_hits, None, None)
        self._check(self._lib.lf_pack_hits(self._h, C.byref(hits), db.n_events, db.hit_x16.data_ptr(), db.origin16.data_ptr(),
                                           self._stream_ptr(stream)))
        return db

    # -- host path (end to end) ------------------------------------------------------------------
    @staticmethod
    def _host_structs(hb: "HostBatch", out: "HostTracks"):
        seeds = lf_seeds(hb.seed_x.data_ptr(), hb.seed_y.data_ptr(), hb.seed_tx.data_ptr(), hb.seed_ty.data_ptr(),
                         hb.seed_qop.data_ptr(), hb.seed_offsets.data_ptr(), hb.n_seeds)
        p = lambda t: t.data_ptr() if t is not None else None
        hits = lf_hits(p(hb.hit_x), hb.seg_offsets.data_ptr(), hb.n_hits, p(hb.hit_x16), p(hb.origin16))
        tr = lf_tracks(out.hit_idx.data_ptr(), out.seed_idx.data_ptr(), out.n_hits.data_ptr(), out.state.data_ptr(),
                       out.quality.data_ptr(), out.event_offsets.data_ptr(), out.n_tracks.data_ptr(), out.capacity)
        return seeds, hits, tr

    def run_host(self, hb: "HostBatch", out: "HostTracks", stream=None) -> int:
        """``lf_run_host``: host buffers in, host buffers out; returns the number of tracks."""
        seeds, hits, tr = self._host_structs(hb, out)
        self._check(self._lib.lf_run_host(self._h, C.byref(seeds), C.byref(hits), hb.n_events, C.byref(tr),
                                          self._stream_ptr(stream)))
        return int(out.n_tracks[0])

    def host_submit(self, hb: "HostBatch", out: "HostTracks", slot: int, stream=None):
        """``lf_host_submit``: enqueue a host batch in ``slot`` (0 or 1) and return at once; ``hb`` and ``out`` must stay
        alive and untouched until :meth:`host_collect` of that slot."""
        seeds, hits, tr = self._host_structs(hb, out)
        self._check(self._lib.lf_host_submit(self._h, C.byref(seeds), C.byref(hits), hb.n_events, C.byref(tr),
                                             self._stream_ptr(stream), int(slot)))

    def host_collect(self, slot: int):
        """``lf_host_collect``: wait until the batch submitted to ``slot`` is complete in its host arrays."""
        self._check(self._lib.lf_host_collect(self._h, int(slot)))

    def run_counters(self):
        """``lf_run_counters`` (synchronous): the work counters of the last run as a dict (include/lf.h); entries 2..6 are
        counted by debug launches only (:meth:`run` with ``debug=True`` or :meth:`run_counting`)."""
        c = (C.c_uint64 * N_COUNTERS)()
        self._check(self._lib.lf_run_counters(self._h, C.byref(c)))
        return {n: int(v) for n, v in zip(COUNTER_NAMES, c)}

    def run_counting(self, db: "DeviceBatch", out: "TrackBuffers", stream=None):
        """``lf_run_debug`` with no stage-boundary table requested: the debug build of the kernels, which also counts
        the work items of every stage (:meth:`run_counters`)."""
        seeds = lf_seeds(db.seed_x.data_ptr(), db.seed_y.data_ptr(), db.seed_tx.data_ptr(), db.seed_ty.data_ptr(),
                         db.seed_qop.data_ptr(), db.seed_offsets.data_ptr(), db.n_seeds)
        hits = db.c_hits()
        tr = out.c_struct()
        dbg = lf_debug()
        self._check(self._lib.lf_run_debug(self._h, C.byref(seeds), C.byref(hits), db.n_events, C.byref(tr), C.byref(dbg),
                                           self._stream_ptr(stream)))
        return out

    def set_host_chunk_events(self, min_events_per_chunk: int):
        """``lf_set_host_chunk_events``: pipeline granularity of :meth:`run_host`."""
        self._check(self._lib.lf_set_host_chunk_events(self._h, int(min_events_per_chunk)))

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.lf_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class HostBatch:
    """A batch in pinned host memory (inputs of ``lf_run_host``)."""

    def __init__(self, batch, pin: bool = True):
        import torch

        def t(a):
            x = torch.from_numpy(np.ascontiguousarray(a))
            return x.pin_memory() if pin else x
        self.n_events = int(batch.n_events)
        self.n_seeds = int(batch.seed_x.shape[0])
        self.n_hits = int(batch.hit_x.shape[0])
        self.seed_x, self.seed_y = t(batch.seed_x), t(batch.seed_y)
        self.seed_tx, self.seed_ty, self.seed_qop = t(batch.seed_tx), t(batch.seed_ty), t(batch.seed_qop)
        self.seed_offsets = t(np.asarray(batch.seed_offsets, dtype=np.uint32).view(np.int32))
        self.hit_x = t(batch.hit_x)
        self.seg_offsets = t(np.asarray(batch.seg_offsets, dtype=np.uint32).view(np.int32))
        self.hit_x16 = None
        self.origin16 = None
        self._pin = pin

    def use_packed(self, db: DeviceBatch, keep_fp32: bool = False):
        """Takes the packed fp16 copy of a device batch (LookingForward.pack_hits) as the host input; unless
        ``keep_fp32`` the fp32 hits are dropped, so that the host path moves 2 bytes per hit plus the origins."""
        pin = (lambda x: x.pin_memory()) if self._pin else (lambda x: x)
        self.hit_x16 = pin(db.hit_x16.cpu())
        self.origin16 = pin(db.origin16.cpu())
        if not keep_fp32:
            self.hit_x = None
        return self

    def h2d_bytes(self) -> int:
        ts = (self.seed_x, self.seed_y, self.seed_tx, self.seed_ty, self.seed_qop, self.seed_offsets, self.hit_x,
              self.seg_offsets, self.hit_x16, self.origin16)
        return int(sum(x.numel() * x.element_size() for x in ts if x is not None))


class HostTracks:
    """Pinned host output arrays for ``lf_run_host``."""

    def __init__(self, capacity: int, n_events: int, pin: bool = True):
        import torch
        cap = max(int(capacity), 1)
        mk = lambda shape, dt: (torch.empty(shape, dtype=dt).pin_memory() if pin else torch.empty(shape, dtype=dt))
        self.capacity = int(capacity)
        self.hit_idx = mk((cap, NL), torch.int32)
        self.seed_idx = mk((cap,), torch.int32)
        self.n_hits = mk((cap,), torch.int32)
        self.state = mk((cap, 5), torch.float32)
        self.quality = mk((cap,), torch.float32)
        self.event_offsets = mk((n_events + 1,), torch.int32)
        self.n_tracks = torch.zeros(1, dtype=torch.int32)

    def d2h_bytes(self, n_tracks: int) -> int:
        return int(n_tracks * (NL + 1 + 1 + 5 + 1) * 4 + self.event_offsets.numel() * 4 + 4)

    def to_numpy(self) -> SimpleNamespace:
        n = int(self.n_tracks[0])
        g = lambda t: t[:n].numpy().copy()
        return SimpleNamespace(n_tracks=n, hit_idx=g(self.hit_idx), seed_idx=g(self.seed_idx), n_hits=g(self.n_hits),
                               state=g(self.state), quality=g(self.quality),
                               event_offsets=self.event_offsets.numpy().view(np.uint32).copy(), debug=None)
