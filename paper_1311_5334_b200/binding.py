"""ctypes binding of include/emu.h.  Marshalling only: every step of the path runs in the CUDA kernels.

Compute calls take torch CUDA tensors (caller-owned device memory) and enqueue on the current torch
stream.  `run_path` is a convenience that allocates the outputs and calls the three entry points in
order; it adds no arithmetic.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libemu4pi.so")

EMU_CNT = dict(seeds=0, tests=1, candidates=2, tracks=3, members=4, status=5, pair_tests=6, need=7)
EMU_ST = dict(cand_overflow=1, track_overflow=2, member_overflow=4, range=8, coord=16, seed_overflow=32, grain_overflow=64)
_ERR = {-1: "EMU_ERR_INVALID", -2: "EMU_ERR_CAPACITY", -3: "EMU_ERR_CUDA"}

TRACK_DTYPE = np.dtype([("view", "<i4"), ("seed_a", "<i4"), ("seed_b", "<i4"), ("n_tube", "<i4"),
                        ("n_members", "<i4"), ("member_off", "<i4"), ("seed_d2", "<i4"), ("pad", "<i4")])
FIT_DTYPE = np.dtype([("axis", "<i4"), ("n", "<i4"), ("u_min", "<i4"), ("u_max", "<i4"),
                      ("slope", "<f8", (2,)), ("icpt", "<f8", (2,))])


class EmuError(RuntimeError):
    pass


class emu_params(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("view_size_q", C.c_int32 * 3), ("cell_size_q", C.c_int32 * 3),
                ("sep_min_q", C.c_int32), ("sep_max_q", C.c_int32), ("tube_r2_q", C.c_int32),
                ("tube_ext_q", C.c_int32), ("min_grains", C.c_int32), ("max_tracks_per_view", C.c_int32),
                ("reserved", C.c_int32 * 4), ("angle_min_grains", C.c_int32 * 8)]


_SYMBOLS = ["emu_workspace_bytes", "emu_grid_cells", "emu_bin_grains", "emu_find_tracks", "emu_count_seeds",
            "emu_fit_tracks", "emu_host_arena_bytes", "emu_track_views_host", "emu_profile_create", "emu_profile_destroy", "emu_profile_begin", "emu_profile_end",
            "emu_profile_read", "emu_recognize_ws_bytes", "emu_recognize_grains", "emu_stream_arena_bytes", "emu_stream_create",
            "emu_stream_destroy", "emu_stream_submit", "emu_stream_collect", "emu_bin_noalloc_max_bytes",
            "emu_bin_grains_noalloc"]
EMU_STAGE = dict(bin_count=0, bin_scan=1, bin_scatter=2, bin_place=3, prep=4, vote=5, assoc=6, select=7, emit=8, fit=9,
                 seeds=10, cands=11, recog=12, generic=13)
EMU_STAGE_COUNT = 16
_lib = None


def library_path() -> str:
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise EmuError(f"{_LIB_PATH} is missing: build it with `python -m paper_1311_5334_b200.build` "
                           "(or __graft_entry__.build()).  There is no CPU fallback.")
        L = C.CDLL(_LIB_PATH)
        vp, i64, i32, sz = C.c_void_p, C.c_int64, C.c_int32, C.c_size_t
        L.emu_workspace_bytes.restype = C.c_int
        L.emu_workspace_bytes.argtypes = [vp, i64, i32, C.POINTER(sz), C.POINTER(sz)]
        L.emu_grid_cells.restype = i64
        L.emu_grid_cells.argtypes = [vp, C.POINTER(i32 * 3)]
        L.emu_bin_grains.restype = C.c_int
        L.emu_bin_grains.argtypes = [vp, vp, vp, i64, i32, vp, vp, vp, vp, sz, vp]
        L.emu_bin_noalloc_max_bytes.restype = sz
        L.emu_bin_noalloc_max_bytes.argtypes = []
        L.emu_bin_grains_noalloc.restype = C.c_int
        L.emu_bin_grains_noalloc.argtypes = [vp, vp, vp, i64, i32, vp, vp, vp, vp]
        L.emu_find_tracks.restype = C.c_int
        L.emu_find_tracks.argtypes = [vp, vp, vp, vp, i64, i32, vp, vp, vp, i64, vp, vp, sz, vp]
        L.emu_count_seeds.restype = C.c_int
        L.emu_count_seeds.argtypes = [vp, vp, vp, vp, i64, i32, vp, i64, vp, vp, sz, vp]
        L.emu_fit_tracks.restype = C.c_int
        L.emu_fit_tracks.argtypes = [vp, vp, vp, vp, vp, i32, vp, vp]
        L.emu_host_arena_bytes.restype = C.c_int
        L.emu_host_arena_bytes.argtypes = [vp, i64, i32, C.POINTER(sz)]
        L.emu_track_views_host.restype = C.c_int
        L.emu_track_views_host.argtypes = [vp, vp, vp, i64, i32, vp, vp, i64, vp, vp, i64, vp, vp, sz, vp]
        L.emu_recognize_ws_bytes.restype = sz
        L.emu_recognize_ws_bytes.argtypes = [i32, i32, i32, i64]
        L.emu_recognize_grains.restype = C.c_int
        L.emu_recognize_grains.argtypes = [vp, i32, i32, i32, i32, i32, C.POINTER(i32 * 3), vp, i64, vp, vp, vp, vp, sz, vp]
        L.emu_stream_arena_bytes.restype = C.c_int
        L.emu_stream_arena_bytes.argtypes = [vp, i64, i32, C.POINTER(sz)]
        L.emu_stream_create.restype = vp
        L.emu_stream_create.argtypes = [vp, i64, i32, vp, sz]
        L.emu_stream_destroy.restype = None
        L.emu_stream_destroy.argtypes = [vp]
        L.emu_stream_submit.restype = C.c_int
        L.emu_stream_submit.argtypes = [vp, vp, vp, i64, i32]
        L.emu_stream_collect.restype = C.c_int
        L.emu_stream_collect.argtypes = [vp, vp, vp, i64, vp, vp, i64, vp]
        L.emu_profile_create.restype = vp
        L.emu_profile_create.argtypes = []
        L.emu_profile_destroy.restype = None
        L.emu_profile_destroy.argtypes = [vp]
        L.emu_profile_begin.restype = C.c_int
        L.emu_profile_begin.argtypes = [vp]
        L.emu_profile_end.restype = C.c_int
        L.emu_profile_end.argtypes = []
        L.emu_profile_read.restype = C.c_int
        L.emu_profile_read.argtypes = [vp, vp, vp]
        _lib = L
    return _lib


def exported_symbols() -> list:
    """Names include/emu.h declares, each resolved in the loaded library (raises if one is missing)."""
    L = _load()
    for s in _SYMBOLS:
        getattr(L, s)
    return list(_SYMBOLS)


def make_params(view_size_q, cell_size_q, sep_min_q, sep_max_q, tube_r2_q, min_grains,
                max_tracks_per_view=4096, tube_ext_q=-1, cand_per_grain=0, seeds_per_grain=0,
                angle_min_grains=None) -> emu_params:
    p = emu_params()
    p.struct_size = C.sizeof(emu_params)
    p.view_size_q[:] = [int(x) for x in view_size_q]
    p.cell_size_q[:] = [int(x) for x in cell_size_q]
    p.sep_min_q, p.sep_max_q, p.tube_r2_q = int(sep_min_q), int(sep_max_q), int(tube_r2_q)
    p.tube_ext_q, p.min_grains, p.max_tracks_per_view = int(tube_ext_q), int(min_grains), int(max_tracks_per_view)
    p.reserved[0] = int(cand_per_grain)
    p.reserved[1] = int(seeds_per_grain)
    if angle_min_grains is not None:
        p.angle_min_grains[:] = [int(x) for x in angle_min_grains]
    return p


def _check(rc: int, what: str):
    if rc != 0:
        raise EmuError(f"{what} returned {_ERR.get(rc, rc)}")


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, dtype=None):
    if not t.is_cuda or not t.is_contiguous() or (dtype is not None and t.dtype != dtype):
        raise EmuError("expected a contiguous CUDA tensor of the documented dtype")
    return t


def _nbytes(t) -> int:
    return t.numel() * t.element_size()


def emu_workspace_bytes(params: emu_params, n_grains: int, n_views: int):
    b, f = C.c_size_t(0), C.c_size_t(0)
    _check(_load().emu_workspace_bytes(C.byref(params), n_grains, n_views, C.byref(b), C.byref(f)),
           "emu_workspace_bytes")
    return int(b.value), int(f.value)


def emu_grid_cells(params: emu_params):
    dims = (C.c_int32 * 3)()
    n = _load().emu_grid_cells(C.byref(params), C.byref(dims))
    if n < 0:
        raise EmuError("emu_grid_cells: bad params")
    return int(n), tuple(int(x) for x in dims)


def emu_bin_grains(params, d_grains, d_view_off, n_grains, n_views, d_sorted, d_cell_start, d_status, d_ws):
    import torch
    _dev(d_grains, torch.int32); _dev(d_view_off, torch.int32); _dev(d_sorted, torch.int32)
    _dev(d_cell_start, torch.int32); _dev(d_status, torch.int64); _dev(d_ws)
    _check(_load().emu_bin_grains(C.byref(params), _ptr(d_grains), _ptr(d_view_off), n_grains, n_views,
                                  _ptr(d_sorted), _ptr(d_cell_start), _ptr(d_status), _ptr(d_ws), _nbytes(d_ws),
                                  _stream()), "emu_bin_grains")


def emu_bin_noalloc_max_bytes() -> int:
    """Size of the scratch block built into the library (bytes): the largest `bin_bytes` emu_bin_grains_noalloc takes."""
    return int(_load().emu_bin_noalloc_max_bytes())


def emu_bin_grains_noalloc(params, d_grains, d_view_off, n_grains, n_views, d_sorted, d_cell_start, d_status):
    """emu_bin_grains without the workspace argument, for code that must not (or cannot) allocate device memory where
    it bins a view: an acquisition loop that may not stall the device with a cudaMalloc, a plug-in next to a memory
    pool that already owns the GPU, a callee that only receives input and output tensors.  The scratch is a fixed
    8 MiB block inside libemu4pi.so (held by every GPU that loads the library); batches whose `bin_bytes`
    (emu_workspace_bytes) exceed it are refused.  Calls on one device share the block, so do not let two of them
    overlap on the GPU; call it once at set-up on each device (the first call resolves the block's device address).
    Results are those of emu_bin_grains, bit for bit."""
    import torch
    _dev(d_grains, torch.int32); _dev(d_view_off, torch.int32); _dev(d_sorted, torch.int32)
    _dev(d_cell_start, torch.int32); _dev(d_status, torch.int64)
    rc = _load().emu_bin_grains_noalloc(C.byref(params), _ptr(d_grains), _ptr(d_view_off), n_grains, n_views,
                                        _ptr(d_sorted), _ptr(d_cell_start), _ptr(d_status), _stream())
    if rc == -2:
        raise EmuError(f"emu_bin_grains_noalloc: this batch ({n_grains} grains, {n_views} views) needs more scratch than the "
                       f"{emu_bin_noalloc_max_bytes()} bytes built into the library (EMU_ERR_CAPACITY): bin fewer views per "
                       "call or use emu_bin_grains with a workspace")
    _check(rc, "emu_bin_grains_noalloc")


def emu_find_tracks(params, d_sorted, d_cell_start, d_view_off, n_grains, n_views, d_tracks, d_track_off, d_members,
                    d_counts, d_ws):
    import torch
    _dev(d_sorted, torch.int32); _dev(d_cell_start, torch.int32); _dev(d_view_off, torch.int32)
    _dev(d_tracks, torch.int32); _dev(d_track_off, torch.int32); _dev(d_members, torch.int32)
    _dev(d_counts, torch.int64); _dev(d_ws)
    _check(_load().emu_find_tracks(C.byref(params), _ptr(d_sorted), _ptr(d_cell_start), _ptr(d_view_off), n_grains,
                                   n_views, _ptr(d_tracks), _ptr(d_track_off), _ptr(d_members), d_members.numel(),
                                   _ptr(d_counts), _ptr(d_ws), _nbytes(d_ws), _stream()), "emu_find_tracks")


def emu_count_seeds(params, d_sorted, d_cell_start, d_view_off, n_grains, n_views, d_seed_dump, d_counts, d_ws):
    import torch
    _dev(d_sorted, torch.int32); _dev(d_cell_start, torch.int32); _dev(d_view_off, torch.int32)
    _dev(d_seed_dump, torch.int32); _dev(d_counts, torch.int64); _dev(d_ws)
    _check(_load().emu_count_seeds(C.byref(params), _ptr(d_sorted), _ptr(d_cell_start), _ptr(d_view_off), n_grains,
                                   n_views, _ptr(d_seed_dump), d_seed_dump.numel() // 4, _ptr(d_counts), _ptr(d_ws),
                                   _nbytes(d_ws), _stream()), "emu_count_seeds")


def emu_fit_tracks(params, d_grains, d_tracks, d_track_off, d_members, n_views, d_fits):
    import torch
    _dev(d_grains, torch.int32); _dev(d_tracks, torch.int32); _dev(d_track_off, torch.int32)
    _dev(d_members, torch.int32); _dev(d_fits)
    _check(_load().emu_fit_tracks(C.byref(params), _ptr(d_grains), _ptr(d_tracks), _ptr(d_track_off),
                                  _ptr(d_members), n_views, _ptr(d_fits), _stream()), "emu_fit_tracks")


def emu_recognize_grains(d_vox, threshold: int, pitch_q, d_grains, d_view_off, d_count, d_status, d_ws):
    """A0: d_vox uint8 [n_views, nz, ny, nx] on the device -> d_grains int32 [capacity, 4],
    d_view_off int32 [n_views+1], d_count int64 [1].  Argument marshalling only."""
    n_views, nz, ny, nx = (int(x) for x in d_vox.shape)
    pitch = (C.c_int32 * 3)(*[int(x) for x in pitch_q])
    _check(_load().emu_recognize_grains(_ptr(d_vox), n_views, nx, ny, nz, int(threshold), C.byref(pitch), _ptr(d_grains),
                                        int(d_grains.shape[0]), _ptr(d_view_off), _ptr(d_count), _ptr(d_status), _ptr(d_ws),
                                        _nbytes(d_ws), _stream()), "emu_recognize_grains")


def emu_recognize_ws_bytes(n_views: int, ny: int, nz: int, capacity: int) -> int:
    return int(_load().emu_recognize_ws_bytes(int(n_views), int(ny), int(nz), int(capacity)))


def emu_host_arena_bytes(params: emu_params, n_grains: int, n_views: int) -> int:
    b = C.c_size_t(0)
    _check(_load().emu_host_arena_bytes(C.byref(params), n_grains, n_views, C.byref(b)), "emu_host_arena_bytes")
    return int(b.value)


class HostPath:
    """emu_track_views_host with its buffers: pinned host arrays for inputs / outputs and one device arena,
    allocated once for a batch shape.  run() copies the caller's grains into the pinned input, makes the ONE
    C-ABI call (H2D, bin, find, fit, D2H inside it) and returns numpy views of the pinned outputs."""

    def __init__(self, params: emu_params, n_grains: int, n_views: int, tracks_capacity: int | None = None):
        import torch
        self.params, self.n_grains, self.n_views = params, n_grains, n_views
        tcap = tracks_capacity if tracks_capacity is not None else max(n_views, 1) * params.max_tracks_per_view
        self.tcap = tcap

        def pin(shape, dt):
            return torch.empty(shape, dtype=dt, pin_memory=True)
        self.h_grains = pin((max(n_grains, 1), 4), torch.int32)
        self.h_view_off = pin(n_views + 1, torch.int32)
        self.h_tracks = pin((max(tcap, 1), 8), torch.int32)
        self.h_fits = pin(max(tcap, 1) * FIT_DTYPE.itemsize, torch.uint8)
        self.h_track_off = pin(n_views + 1, torch.int32)
        self.h_members = pin(max(n_grains, 1), torch.int32)
        self.h_counts = pin(8, torch.int64)
        self.arena = torch.empty(emu_host_arena_bytes(params, n_grains, n_views), dtype=torch.uint8, device="cuda")

    def h2d_bytes(self) -> int:
        return self.n_grains * 16 + (self.n_views + 1) * 4

    def call(self):
        """the C-ABI call alone, on what already sits in the pinned input arrays"""
        rc = _load().emu_track_views_host(C.byref(self.params), C.c_void_p(self.h_grains.data_ptr()),
                                          C.c_void_p(self.h_view_off.data_ptr()), self.n_grains, self.n_views,
                                          C.c_void_p(self.h_tracks.data_ptr()), C.c_void_p(self.h_fits.data_ptr()),
                                          self.tcap, C.c_void_p(self.h_track_off.data_ptr()),
                                          C.c_void_p(self.h_members.data_ptr()), self.h_members.numel(),
                                          C.c_void_p(self.h_counts.data_ptr()), _ptr(self.arena), _nbytes(self.arena),
                                          _stream())
        _check(rc, "emu_track_views_host")
        c = self.h_counts.numpy()
        nt, nm = int(c[EMU_CNT["tracks"]]), int(c[EMU_CNT["members"]])
        return nt, nm

    def d2h_bytes(self, nt: int, nm: int) -> int:
        return 64 + 8 + (self.n_views + 1) * 4 + nt * (TRACK_DTYPE.itemsize + FIT_DTYPE.itemsize) + nm * 4

    def run(self, grains: np.ndarray, view_off: np.ndarray) -> dict:
        import torch
        if self.n_grains:
            self.h_grains[:self.n_grains].copy_(torch.from_numpy(np.ascontiguousarray(grains, np.int32).reshape(-1, 4)))
        self.h_view_off.copy_(torch.from_numpy(np.ascontiguousarray(view_off, np.int32)))
        nt, nm = self.call()
        return self.result(nt, nm)

    def result(self, nt: int, nm: int) -> dict:
        """copies of the pinned outputs of the last call()"""
        return dict(tracks=self.h_tracks[:nt].numpy().view(TRACK_DTYPE).reshape(-1).copy(),
                    fits=self.h_fits[:nt * FIT_DTYPE.itemsize].numpy().view(FIT_DTYPE).reshape(-1).copy(),
                    members=self.h_members[:nm].numpy().copy(), track_off=self.h_track_off.numpy().copy(),
                    counts=self.h_counts.numpy().copy())


class StreamPath:
    """emu_stream_* of include/emu.h with its buffers: batches of views through one GPU, the host->device copy of the
    next batch and the device->host copy of the previous one hidden behind the kernels of the current one.  Two pinned
    input buffers (a submitted batch must stay untouched until it is collected), one set of pinned outputs, one device
    arena.  submit() / collect() marshal only."""

    def __init__(self, params: emu_params, max_grains: int, max_views: int):
        import torch
        self.params, self.max_grains, self.max_views = params, max_grains, max_views
        b = C.c_size_t(0)
        _check(_load().emu_stream_arena_bytes(C.byref(params), max_grains, max_views, C.byref(b)), "emu_stream_arena_bytes")
        self.arena = torch.empty(int(b.value), dtype=torch.uint8, device="cuda")
        # the library works on three streams of its own, which know nothing of torch's: the block the caching allocator
        # has just handed out may still be in use by work queued on the current stream, so let that finish first
        torch.cuda.current_stream().synchronize()
        self._h = _load().emu_stream_create(C.byref(params), max_grains, max_views, _ptr(self.arena), _nbytes(self.arena))
        if not self._h:
            raise EmuError("emu_stream_create failed")
        tcap = max(max_views, 1) * params.max_tracks_per_view
        self.tcap = tcap

        def pin(shape, dt):
            return torch.empty(shape, dtype=dt, pin_memory=True)
        self.h_in = [(pin((max(max_grains, 1), 4), torch.int32), pin(max_views + 1, torch.int32)) for _ in range(2)]
        self.h_tracks = pin((max(tcap, 1), 8), torch.int32)
        self.h_fits = pin(max(tcap, 1) * FIT_DTYPE.itemsize, torch.uint8)
        self.h_track_off = pin(max_views + 1, torch.int32)
        self.h_members = pin(max(max_grains, 1), torch.int32)
        self.h_counts = pin(8, torch.int64)
        self._k = 0
        self._shapes = []

    def submit(self, grains: np.ndarray, view_off: np.ndarray) -> int:
        import torch
        if len(self._shapes) >= 2:                   # both pinned input buffers hold batches that are still in flight
            raise EmuError("StreamPath.submit: two batches are in flight, collect one first")
        hg, ho = self.h_in[self._k & 1]
        n, nv = len(grains), len(view_off) - 1
        if n:
            hg[:n].copy_(torch.from_numpy(np.ascontiguousarray(grains, np.int32).reshape(-1, 4)))
        ho[:nv + 1].copy_(torch.from_numpy(np.ascontiguousarray(view_off, np.int32)))
        rc = _load().emu_stream_submit(self._h, C.c_void_p(hg.data_ptr()), C.c_void_p(ho.data_ptr()), n, nv)
        if rc < 0:
            _check(rc, "emu_stream_submit")
        self._k += 1
        self._shapes.append((n, nv))
        return rc

    def collect(self, copy: bool = True) -> dict:
        n, nv = self._shapes.pop(0)
        rc = _load().emu_stream_collect(self._h, C.c_void_p(self.h_tracks.data_ptr()), C.c_void_p(self.h_fits.data_ptr()),
                                        self.tcap, C.c_void_p(self.h_track_off.data_ptr()),
                                        C.c_void_p(self.h_members.data_ptr()), self.h_members.numel(),
                                        C.c_void_p(self.h_counts.data_ptr()))
        _check(rc, "emu_stream_collect")
        c = self.h_counts.numpy()
        nt, nm = int(c[EMU_CNT["tracks"]]), int(c[EMU_CNT["members"]])
        if not copy:
            return dict(n_tracks=nt, n_members=nm, counts=c.copy())
        return dict(tracks=self.h_tracks[:nt].numpy().view(TRACK_DTYPE).reshape(-1).copy(),
                    fits=self.h_fits[:nt * FIT_DTYPE.itemsize].numpy().view(FIT_DTYPE).reshape(-1).copy(),
                    members=self.h_members[:nm].numpy().copy(), track_off=self.h_track_off[:nv + 1].numpy().copy(),
                    counts=c.copy())

    def close(self):
        if self._h:
            _load().emu_stream_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Profile:
    """emu_profile_* of include/emu.h: per-stage CUDA-event timing of the library's own launches.

    with Profile() as prof: ...calls...; prof.read() -> ({stage: ms}, {stage: launches}) accumulated."""

    def __init__(self):
        self._h = _load().emu_profile_create()
        if not self._h:
            raise EmuError("emu_profile_create failed")
        self.ms = np.zeros(EMU_STAGE_COUNT, np.float64)
        self.launches = np.zeros(EMU_STAGE_COUNT, np.int64)

    def __enter__(self):
        _check(_load().emu_profile_begin(self._h), "emu_profile_begin")
        return self

    def __exit__(self, *exc):
        _load().emu_profile_end()
        return False

    def read(self):
        _check(_load().emu_profile_read(self._h, self.ms.ctypes.data, self.launches.ctypes.data), "emu_profile_read")
        inv = {v: k for k, v in EMU_STAGE.items()}
        return ({inv[i]: float(self.ms[i]) for i in inv}, {inv[i]: int(self.launches[i]) for i in inv})

    def close(self):
        if self._h:
            _load().emu_profile_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class PathBuffers:
    """Caller-owned device memory for a batch shape, allocated once with torch and reused per step."""

    def __init__(self, params: emu_params, n_grains: int, n_views: int, members_capacity: int | None = None,
                 find_ws_bytes: int | None = None, device="cuda"):
        import torch
        self.params, self.n_grains, self.n_views = params, n_grains, n_views
        ncell, _ = emu_grid_cells(params)
        bin_b, find_b = emu_workspace_bytes(params, n_grains, n_views)
        if find_ws_bytes is not None:
            find_b = find_ws_bytes
        cap = max(n_views * params.max_tracks_per_view, 1)

        def e(n, dt):
            return torch.empty(n, dtype=dt, device=device)
        self.sorted = torch.empty((max(n_grains, 1), 4), dtype=torch.int32, device=device)
        self.cell_start = e(n_views * ncell + 1, torch.int32)
        self.tracks = torch.empty((cap, 8), dtype=torch.int32, device=device)
        self.track_off = e(n_views + 1, torch.int32)
        self.members = e(max(members_capacity if members_capacity is not None else n_grains, 1), torch.int32)
        self.fits = e(cap * FIT_DTYPE.itemsize, torch.uint8)
        self.counts = torch.zeros(8, dtype=torch.int64, device=device)
        self.status = torch.zeros(1, dtype=torch.int64, device=device)
        self.ws = e(max(bin_b, find_b), torch.uint8)


@dataclass
class PathResult:
    """Device buffers of one pass of the path; .host() copies the valid parts back."""
    buffers: PathBuffers

    def host(self) -> dict:
        B = self.buffers
        counts = B.counts.cpu().numpy().copy()
        counts[EMU_CNT["status"]] |= int(B.status.cpu()[0])
        nt, nm = int(counts[EMU_CNT["tracks"]]), int(counts[EMU_CNT["members"]])
        nm = min(nm, B.members.numel())
        tracks = B.tracks[:nt].cpu().numpy().view(TRACK_DTYPE).reshape(-1)
        fits = B.fits[:nt * FIT_DTYPE.itemsize].cpu().numpy().view(FIT_DTYPE).reshape(-1)
        return dict(tracks=tracks, fits=fits, members=B.members[:nm].cpu().numpy(),
                    track_off=B.track_off.cpu().numpy(), counts=counts,
                    sorted=B.sorted, cell_start=B.cell_start)


def run_path(params: emu_params, d_grains, d_view_off, n_views: int, buffers: PathBuffers | None = None,
             fit: bool = True) -> PathResult:
    """One pass of the hot path on the current stream: emu_bin_grains -> emu_find_tracks -> emu_fit_tracks."""
    n_grains = int(d_grains.shape[0])
    B = buffers if buffers is not None else PathBuffers(params, n_grains, n_views, device=d_grains.device)
    B.status.zero_()
    emu_bin_grains(params, d_grains, d_view_off, n_grains, n_views, B.sorted, B.cell_start, B.status, B.ws)
    emu_find_tracks(params, B.sorted, B.cell_start, d_view_off, n_grains, n_views, B.tracks, B.track_off, B.members,
                    B.counts, B.ws)
    if fit:
        emu_fit_tracks(params, d_grains, B.tracks, B.track_off, B.members, n_views, B.fits)
    return PathResult(B)
