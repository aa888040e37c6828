"""ctypes wrapper + build step for the CPU oracle (TEST INFRASTRUCTURE ONLY).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this.  It imports nothing from the CUDA package: callers
pass plain numpy arrays (any object with ``seed_x .. seed_qop, seed_offsets, hit_x, seg_offsets,
n_events`` attributes) and plain dicts for geometry / parameters.

The oracle proper is single-threaded.  ``threads > 1`` is a *harness* feature: events are
independent, so the batch is cut into contiguous event ranges, each range runs the
unchanged oracle in its own thread, and the outputs are concatenated with indices rebased.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from types import SimpleNamespace
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lf_oracle.cpp")
_LIBS = {"f32": os.path.join(_HERE, "liblf_oracle.so"), "f64": os.path.join(_HERE, "liblf_oracle_f64.so")}
_CXXFLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra", "-shared", "-fPIC"]
NL = 12


def build(force: bool = False) -> None:
    """Compile the oracle (fp32 reference build and fp64 pin build) with g++."""
    deps = [_SRC, os.path.join(_HERE, "lf_oracle.h")]
    newest = max(os.path.getmtime(d) for d in deps)
    for kind, lib in _LIBS.items():
        if not force and os.path.exists(lib) and os.path.getmtime(lib) >= newest:
            continue
        cmd = ["g++"] + _CXXFLAGS + (["-DLF_ORACLE_REAL=double"] if kind == "f64" else []) + [_SRC, "-o", lib]
        subprocess.run(cmd, check=True)


class _Geometry(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("z", C.c_float * NL), ("tan_alpha", C.c_float * NL),
                ("z_seed", C.c_float), ("z_mag", C.c_float), ("kick", C.c_float),
                ("z_ref", C.c_float), ("d_ratio", C.c_float),
                ("k_first", C.c_float), ("k_last", C.c_float), ("qop_poly", C.c_float * 5),
                ("x_half", C.c_float), ("y_half", C.c_float), ("z_state", C.c_float),
                ("polarity", C.c_int32), ("qop_mode", C.c_int32), ("qop_poly2d", (C.c_float * 10) * 5)]


class _Params(C.Structure):
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
                ("xtol_poly", C.c_float * 8), ("x_overlap", C.c_float)]


_FP = C.POINTER(C.c_float)
_IP = C.POINTER(C.c_int32)
_UP = C.POINTER(C.c_uint32)


class _Seeds(C.Structure):
    _fields_ = [("x", _FP), ("y", _FP), ("tx", _FP), ("ty", _FP), ("qop", _FP), ("event_offsets", _UP)]


class _Hits(C.Structure):
    _fields_ = [("x", _FP), ("seg_offsets", _UP)]


class _Tracks(C.Structure):
    _fields_ = [("hit_idx", _IP), ("seed_idx", _IP), ("n_hits", _IP), ("state", _FP), ("quality", _FP),
                ("event_offsets", _UP), ("n_tracks", _UP), ("capacity", C.c_size_t)]


class _Debug(C.Structure):
    _fields_ = [("win_first", _IP), ("win_count", _IP), ("n_triplets", _IP), ("trip_hits", _IP),
                ("trip_set", _IP), ("trip_chi2", _FP), ("cand_hits", _IP), ("cand_quality", _FP)]


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


_loaded: Dict[str, C.CDLL] = {}


def _lib(real: str) -> C.CDLL:
    if real not in _loaded:
        build()
        lib = C.CDLL(_LIBS[real])
        lib.lf_oracle_run.restype = C.c_int
        lib.lf_oracle_run.argtypes = [C.POINTER(_Geometry), C.POINTER(_Params), C.POINTER(_Seeds),
                                      C.POINTER(_Hits), C.c_size_t, C.POINTER(_Tracks), C.POINTER(_Debug)]
        lib.lf_oracle_real_bytes.restype = C.c_int
        assert lib.lf_oracle_real_bytes() == (4 if real == "f32" else 8)
        _loaded[real] = lib
    return _loaded[real]


def _p(a: np.ndarray, t):
    return a.ctypes.data_as(t)


def _run_one(lib, geo, par, b, n_triplets: int, debug: bool):
    n_sides = 2 if int(par.mode) == 1 else 1  # rows of the debug tables per seed (lf_oracle.h)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    u32 = lambda a: np.ascontiguousarray(a, dtype=np.uint32)
    sx, sy, stx, sty, sq = f32(b.seed_x), f32(b.seed_y), f32(b.seed_tx), f32(b.seed_ty), f32(b.seed_qop)
    so, hx, go = u32(b.seed_offsets), f32(b.hit_x), u32(b.seg_offsets)
    n_ev, n_seeds = int(b.n_events), int(sx.shape[0])
    assert so.shape[0] == n_ev + 1 and go.shape[0] == n_ev * 2 * NL + 1
    seeds = _Seeds(_p(sx, _FP), _p(sy, _FP), _p(stx, _FP), _p(sty, _FP), _p(sq, _FP), _p(so, _UP))
    hits = _Hits(_p(hx, _FP), _p(go, _UP))
    cap = max(n_seeds, 1)
    out = SimpleNamespace(
        hit_idx=np.full((cap, NL), -1, np.int32), seed_idx=np.zeros(cap, np.int32),
        n_hits=np.zeros(cap, np.int32), state=np.zeros((cap, 5), np.float32),
        quality=np.zeros(cap, np.float32), event_offsets=np.zeros(n_ev + 1, np.uint32),
        n_tracks=np.zeros(1, np.uint32))
    tr = _Tracks(_p(out.hit_idx, _IP), _p(out.seed_idx, _IP), _p(out.n_hits, _IP), _p(out.state, _FP),
                 _p(out.quality, _FP), _p(out.event_offsets, _UP), _p(out.n_tracks, _UP), cap)
    dbg_ptr = None
    dbg = None
    if debug:
        nt, rows = n_triplets, cap * n_sides
        dbg = SimpleNamespace(
            win_first=np.zeros((rows, NL), np.int32), win_count=np.zeros((rows, NL), np.int32),
            n_triplets=np.zeros(rows, np.int32), trip_hits=np.full((rows, nt, 3), -1, np.int32),
            trip_set=np.full((rows, nt), -1, np.int32), trip_chi2=np.full((rows, nt), -1, np.float32),
            cand_hits=np.full((rows, nt, NL), -1, np.int32), cand_quality=np.full((rows, nt), -1, np.float32))
        d = _Debug(_p(dbg.win_first, _IP), _p(dbg.win_count, _IP), _p(dbg.n_triplets, _IP),
                   _p(dbg.trip_hits, _IP), _p(dbg.trip_set, _IP), _p(dbg.trip_chi2, _FP),
                   _p(dbg.cand_hits, _IP), _p(dbg.cand_quality, _FP))
        dbg_ptr = C.byref(d)
    rc = lib.lf_oracle_run(C.byref(geo), C.byref(par), C.byref(seeds), C.byref(hits), n_ev, C.byref(tr), dbg_ptr)
    if rc != 0:
        raise RuntimeError(f"lf_oracle_run failed with status {rc}")
    n = int(out.n_tracks[0])
    res = SimpleNamespace(n_tracks=n, hit_idx=out.hit_idx[:n], seed_idx=out.seed_idx[:n], n_hits=out.n_hits[:n],
                          state=out.state[:n], quality=out.quality[:n], event_offsets=out.event_offsets,
                          debug=None)
    if dbg is not None:
        for k, v in vars(dbg).items():
            setattr(dbg, k, v[:n_seeds * n_sides])
        res.debug = dbg
    return res


def _slice(b, e0: int, e1: int):
    so, go = np.asarray(b.seed_offsets), np.asarray(b.seg_offsets)
    s0, s1 = int(so[e0]), int(so[e1])
    h0, h1 = int(go[e0 * 2 * NL]), int(go[e1 * 2 * NL])
    return SimpleNamespace(
        n_events=e1 - e0, seed_x=b.seed_x[s0:s1], seed_y=b.seed_y[s0:s1], seed_tx=b.seed_tx[s0:s1],
        seed_ty=b.seed_ty[s0:s1], seed_qop=b.seed_qop[s0:s1],
        seed_offsets=(so[e0:e1 + 1].astype(np.int64) - s0).astype(np.uint32),
        hit_x=b.hit_x[h0:h1],
        seg_offsets=(go[e0 * 2 * NL:e1 * 2 * NL + 1].astype(np.int64) - h0).astype(np.uint32)), s0, h0


def run(geometry: Dict[str, object], params: Dict[str, object], batch, debug: bool = False,
        real: str = "f32", threads: int = 1):
    """Run the oracle on ``batch``.  Returns a namespace of numpy arrays (tracks in (event, seed) order)."""
    lib = _lib(real)
    geo = _fill(_Geometry(), geometry)
    par = _fill(_Params(), params)
    nt = int(params["n_triplets"])
    n_ev = int(batch.n_events)
    threads = max(1, min(int(threads), n_ev))
    if threads == 1:
        return _run_one(lib, geo, par, batch, nt, debug)
    # harness-level sharding by contiguous event ranges of roughly equal seed count
    so = np.asarray(batch.seed_offsets).astype(np.int64)
    targets = (np.arange(1, threads) * so[-1]) // threads
    cuts = [0] + [int(np.searchsorted(so, t)) for t in targets] + [n_ev]
    cuts = sorted(set(min(max(c, 0), n_ev) for c in cuts))
    parts = [_slice(batch, cuts[i], cuts[i + 1]) for i in range(len(cuts) - 1)]
    with ThreadPoolExecutor(max_workers=threads) as pool:
        results = list(pool.map(lambda a: _run_one(lib, geo, par, a[0], nt, debug), parts))
    hit_idx, seed_idx, ev_off = [], [], [np.zeros(1, np.uint32)]
    base = 0
    for (sub, s0, h0), r in zip(parts, results):
        hit_idx.append(np.where(r.hit_idx >= 0, r.hit_idx + h0, -1).astype(np.int32))
        seed_idx.append((r.seed_idx + s0).astype(np.int32))
        ev_off.append((r.event_offsets[1:].astype(np.int64) + base).astype(np.uint32))
        base += r.n_tracks
    res = SimpleNamespace(
        n_tracks=base, hit_idx=np.concatenate(hit_idx), seed_idx=np.concatenate(seed_idx),
        n_hits=np.concatenate([r.n_hits for r in results]), state=np.concatenate([r.state for r in results]),
        quality=np.concatenate([r.quality for r in results]), event_offsets=np.concatenate(ev_off), debug=None)
    if debug:
        dbg = SimpleNamespace()
        for k in ("win_count", "n_triplets", "trip_set", "trip_chi2", "cand_quality"):
            setattr(dbg, k, np.concatenate([getattr(r.debug, k) for r in results]))
        for k in ("win_first", "trip_hits", "cand_hits"):
            arrs = []
            for (sub, s0, h0), r in zip(parts, results):
                a = getattr(r.debug, k)
                arrs.append(np.where(a >= 0, a + h0, -1).astype(np.int32) if k != "win_first" else (a + h0).astype(np.int32))
            setattr(dbg, k, np.concatenate(arrs))
        res.debug = dbg
    return res
