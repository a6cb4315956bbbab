"""ctypes loader for the CPU oracle (oracle/emu_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
imports nothing from paper_1311_5334_b200 and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "emu_oracle.cpp")
_LIB = os.path.join(_HERE, "libemu_oracle.so")

TRACK_DTYPE = np.dtype([("view", "<i4"), ("seed_a", "<i4"), ("seed_b", "<i4"), ("n_tube", "<i4"),
                        ("n_members", "<i4"), ("member_off", "<i4"), ("seed_d2", "<i4"), ("pad", "<i4")])
FIT_DTYPE = np.dtype([("axis", "<i4"), ("n", "<i4"), ("u_min", "<i4"), ("u_max", "<i4"),
                      ("slope", "<f8", (2,)), ("icpt", "<f8", (2,))])
assert TRACK_DTYPE.itemsize == 32 and FIT_DTYPE.itemsize == 48


class _Params(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("view_size_q", C.c_int32 * 3), ("cell_size_q", C.c_int32 * 3),
                ("sep_min_q", C.c_int32), ("sep_max_q", C.c_int32), ("tube_r2_q", C.c_int32),
                ("tube_ext_q", C.c_int32), ("min_grains", C.c_int32), ("max_tracks_per_view", C.c_int32),
                ("reserved", C.c_int32 * 4), ("angle_min_grains", C.c_int32 * 8)]


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (-fopenmp).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.emo_track_views.restype = C.c_void_p
        L.emo_track_views.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32]
        for f in (L.emo_n_tracks, L.emo_n_members, L.emo_n_seed_dump):
            f.restype = C.c_int64; f.argtypes = [C.c_void_p]
        L.emo_n_cells.restype = C.c_int64; L.emo_n_cells.argtypes = [C.c_void_p]
        L.emo_grid_dims.restype = None; L.emo_grid_dims.argtypes = [C.c_void_p, C.c_void_p]
        L.emo_get.restype = None; L.emo_get.argtypes = [C.c_void_p] * 6
        L.emo_get_seed_dump.restype = None; L.emo_get_seed_dump.argtypes = [C.c_void_p, C.c_void_p]
        L.emo_free.restype = None; L.emo_free.argtypes = [C.c_void_p]
        L.emo_bin.restype = C.c_int; L.emo_bin.argtypes = [C.c_void_p] * 3 + [C.c_int32] + [C.c_void_p] * 2
        L.emo_fit_tracks.restype = C.c_int; L.emo_fit_tracks.argtypes = [C.c_void_p] * 3 + [C.c_int32, C.c_void_p]
        L.emo_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _params(p: dict) -> _Params:
    s = _Params()
    s.struct_size = C.sizeof(_Params)
    s.view_size_q[:] = p["view_size_q"]; s.cell_size_q[:] = p["cell_size_q"]
    s.sep_min_q = p["sep_min_q"]; s.sep_max_q = p["sep_max_q"]; s.tube_r2_q = p["tube_r2_q"]
    s.tube_ext_q = p.get("tube_ext_q", -1); s.min_grains = p["min_grains"]
    s.max_tracks_per_view = p.get("max_tracks_per_view", 4096)
    s.angle_min_grains[:] = [int(x) for x in p.get("angle_min_grains", (0,) * 8)]
    return s


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def grid_dims(params: dict):
    out = np.zeros(3, np.int64)
    sp = _params(params)
    lib().emo_grid_dims(C.byref(sp), out.ctypes.data)
    return tuple(int(x) for x in out)


def bin_grains(params: dict, grains, view_off):
    """O1.  Returns (sorted int32 [N,4], cell_start int32 [n_views*n_cells+1])."""
    grains = _i32(grains); view_off = _i32(view_off)
    sp = _params(params)
    nc = lib().emo_n_cells(C.byref(sp))
    if nc < 0:
        raise ValueError("bad params")
    n_views = len(view_off) - 1
    srt = np.zeros_like(grains)
    cs = np.zeros(n_views * nc + 1, np.int32)
    rc = lib().emo_bin(C.byref(sp), grains.ctypes.data, view_off.ctypes.data, n_views, srt.ctypes.data, cs.ctypes.data)
    if rc:
        raise ValueError("emo_bin failed")
    return srt, cs


@dataclass
class OracleResult:
    tracks: np.ndarray      # TRACK_DTYPE [T]
    track_off: np.ndarray   # int32 [n_views+1]
    members: np.ndarray     # int32 [M] rows of the input array
    fits: np.ndarray        # FIT_DTYPE [T]
    counters: dict
    seed_dump: np.ndarray | None = None   # int32 [S,4]: view, row_a, row_b, n_tube


def track_views(params: dict, grains, view_off, mode: str = "cells", n_threads: int = 0,
                seed_dump: bool = False) -> OracleResult:
    """O2..O7 on a batch of views.  mode = "brute" (no cells) or "cells"."""
    grains = _i32(grains); view_off = _i32(view_off)
    sp = _params(params)
    h = lib().emo_track_views(C.byref(sp), grains.ctypes.data, view_off.ctypes.data, len(view_off) - 1,
                              {"brute": 0, "cells": 1}[mode], n_threads, int(seed_dump))
    if not h:
        raise ValueError("bad params")
    try:
        nt, nm, ns = lib().emo_n_tracks(h), lib().emo_n_members(h), lib().emo_n_seed_dump(h)
        tracks = np.zeros(nt, TRACK_DTYPE); fits = np.zeros(nt, FIT_DTYPE)
        members = np.zeros(nm, np.int32); toff = np.zeros(len(view_off), np.int32); cnt = np.zeros(8, np.int64)
        lib().emo_get(h, tracks.ctypes.data, toff.ctypes.data, members.ctypes.data, fits.ctypes.data, cnt.ctypes.data)
        dump = None
        if seed_dump:
            dump = np.zeros((ns, 4), np.int32)
            lib().emo_get_seed_dump(h, dump.ctypes.data)
    finally:
        lib().emo_free(h)
    if cnt[5] != 0:
        raise ValueError("oracle: input outside the asserted ranges (|coord| < 2^17, members < 2^13)")
    counters = dict(seeds=int(cnt[0]), tube_tests=int(cnt[1]), candidates=int(cnt[2]), tracks=int(cnt[3]),
                    members=int(cnt[4]), pair_tests=int(cnt[6]))
    return OracleResult(tracks, toff, members, fits, counters, dump)


def fit_tracks(grains, members, member_off) -> np.ndarray:
    """O6 alone on caller-given member lists."""
    grains = _i32(grains); members = _i32(members); member_off = _i32(member_off)
    fits = np.zeros(len(member_off) - 1, FIT_DTYPE)
    rc = lib().emo_fit_tracks(grains.ctypes.data, members.ctypes.data, member_off.ctypes.data,
                              len(member_off) - 1, fits.ctypes.data)
    if rc:
        raise ValueError("emo_fit_tracks failed")
    return fits


def max_threads() -> int:
    return int(lib().emo_max_threads())
