"""Seeded synthetic grain clouds shaped like BASELINE.json's five configs.

Stand-in for the paper's scanned emulsion views (PAPER.md:116, :138 - not in
this container).  Recipe = SURVEY.md 8(d), restated in DESIGN.md:

* box [0,X]x[0,Y]x[0,Z] um; fog = exactly round(rho*X*Y*Z) grains, uniform;
* isotropic directions: cos(theta) ~ U[-1,1], phi ~ U[0,2pi);
* "through" tracks (cfg 0/1/4): anchor uniform in the box, track = the full chord
  of the box through it; grains = Poisson process (exponential gaps) along it;
* "short" tracks (cfg 2): start uniform, L ~ U[5,20] um, redrawn until the end
  point is inside; "stars" (cfg 3): vertices uniform, 3..8 prongs each,
  L ~ U[10,200] um clipped at the box, grains start at the vertex;
* smear N(0,0.1 um) in x,y and N(0,0.5 um) in z; quantise floor(64 v + 0.5) to
  int32 units of q = 1/64 um; clamp into [0, size_q-1]; seeded shuffle.

The random numbers come from a counter-based splitmix64 stream written out
here (numpy uint64 arithmetic only), so the bytes depend on nothing but the
key (config, view).  No track-finding arithmetic lives in this file.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

Q_PER_UM = 64  # BASELINE.json north_star: int32 fixed point at 1/64 um

_M64 = (1 << 64) - 1
_GOLD = 0x9E3779B97F4A7C15


def _mix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 output function on a uint64 array (wrap-around arithmetic)."""
    x = x.copy()
    x ^= x >> np.uint64(30)
    x *= np.uint64(0xBF58476D1CE4E5B9)
    x ^= x >> np.uint64(27)
    x *= np.uint64(0x94D049BB133111EB)
    x ^= x >> np.uint64(31)
    return x


def _mix64_int(x: int) -> int:
    x &= _M64
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & _M64
    return x ^ (x >> 31)


class Stream:
    """Counter-based stream: value i = mix64(key + (i+1)*GOLD)."""

    def __init__(self, *key: int):
        s = 0x243F6A8885A308D3
        for k in key:
            s = _mix64_int(s ^ _mix64_int((int(k) + _GOLD) & _M64))
        self.key = s
        self.ctr = 0

    def u64(self, n: int) -> np.ndarray:
        idx = np.arange(self.ctr + 1, self.ctr + n + 1, dtype=np.uint64)
        self.ctr += n
        with np.errstate(over="ignore"):
            return _mix64(np.uint64(self.key) + idx * np.uint64(_GOLD))

    def uniform(self, n: int) -> np.ndarray:
        """U[0,1) doubles with 53 random bits."""
        return (self.u64(n) >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))

    def normal(self, n: int) -> np.ndarray:
        """Standard normals by Box-Muller (two uniforms per value)."""
        u1 = 1.0 - self.uniform(n)          # (0,1]
        u2 = self.uniform(n)
        return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)

    def expo(self, n: int) -> np.ndarray:
        return -np.log(1.0 - self.uniform(n))

    def integers(self, lo: int, hi: int, n: int) -> np.ndarray:
        """Uniform integers in [lo, hi] (inclusive)."""
        return lo + np.floor(self.uniform(n) * (hi - lo + 1)).astype(np.int64)

    def permutation(self, n: int) -> np.ndarray:
        return np.argsort(self.u64(n), kind="stable")


@dataclass(frozen=True)
class ViewConfig:
    name: str
    size_um: tuple          # (X, Y, Z)
    fog_per_1000um3: float
    kind: str               # "through" | "short" | "stars"
    n_tracks: int           # tracks, or vertices for "stars"
    spacing_um: float       # mean grain spacing along a track
    n_views: int = 1
    len_um: tuple = (0.0, 0.0)      # (Lmin, Lmax) for short / stars
    prongs: tuple = (0, 0)          # (min, max) prongs per vertex for stars
    sigma_um: tuple = (0.1, 0.1, 0.5)


# BASELINE.json configs[0..4]
CONFIGS = (
    ViewConfig("tiny", (100.0, 100.0, 50.0), 3.0, "through", 10, 3.0),
    ViewConfig("microscope_view", (350.0, 300.0, 50.0), 3.0, "through", 200, 3.0),
    ViewConfig("neutron_dosimetry", (350.0, 300.0, 50.0), 3.0, "short", 1000, 1.5,
               len_um=(5.0, 20.0)),
    ViewConfig("annihilation_stars", (350.0, 300.0, 50.0), 5.0, "stars", 20, 3.0,
               len_um=(10.0, 200.0), prongs=(3, 8)),
    ViewConfig("throughput_batch", (350.0, 300.0, 50.0), 10.0, "through", 300, 3.0,
               n_views=1024),
)


def default_params(cfg: ViewConfig | int, cell_um=(8.0, 8.0, 8.0),
                   max_tracks_per_view: int = 4096) -> dict:
    """Tracking parameters BASELINE.json fixes for every config (plain values):
    tube radius 0.8 um -> tube_r2_q = floor(0.64*4096) = 2621, pair separation
    4..20 um -> 256..1280 q, min 8 grains, whole-line tube (tube_ext_q = -1)."""
    if isinstance(cfg, int):
        cfg = CONFIGS[cfg]
    return dict(
        view_size_q=tuple(int(round(s * Q_PER_UM)) for s in cfg.size_um),
        cell_size_q=tuple(int(round(c * Q_PER_UM)) for c in cell_um),
        sep_min_q=256, sep_max_q=1280, tube_r2_q=2621, tube_ext_q=-1,
        min_grains=8, max_tracks_per_view=max_tracks_per_view,
    )


@dataclass
class ViewBatch:
    grains: np.ndarray          # int32 [N,4]: x,y,z (q units), w = caller payload
    view_off: np.ndarray        # int32 [n_views+1]
    truth: np.ndarray           # int32 [N]: true track id within the view, -1 = fog
    lines: list = field(default_factory=list)   # per view: float64 [T,7] = p0(3), dir(3), length (um)
    config: ViewConfig | None = None

    @property
    def n_views(self) -> int:
        return len(self.view_off) - 1

    @property
    def n_grains(self) -> int:
        return int(self.view_off[-1])

    def view(self, v: int) -> np.ndarray:
        return self.grains[self.view_off[v]:self.view_off[v + 1]]


def _iso_dirs(st: Stream, n: int) -> np.ndarray:
    c = 2.0 * st.uniform(n) - 1.0
    phi = 2.0 * np.pi * st.uniform(n)
    s = np.sqrt(np.maximum(0.0, 1.0 - c * c))
    return np.stack([s * np.cos(phi), s * np.sin(phi), c], axis=1)


def _chord(p: np.ndarray, u: np.ndarray, size: np.ndarray):
    """Parameter range [t0,t1] of p + t*u inside the box [0,size] (slab method)."""
    with np.errstate(divide="ignore", invalid="ignore"):
        ta = (0.0 - p) / u
        tb = (size - p) / u
    lo = np.where(u != 0.0, np.minimum(ta, tb), -np.inf)
    hi = np.where(u != 0.0, np.maximum(ta, tb), np.inf)
    return lo.max(axis=1), hi.min(axis=1)


def _poisson_process(st: Stream, start: np.ndarray, dirs: np.ndarray,
                     length: np.ndarray, spacing: float):
    """Points of a rate-1/spacing Poisson process on [0,length) of each segment."""
    n_seg = len(length)
    if n_seg == 0:
        return np.zeros((0, 3)), np.zeros(0, np.int64)
    m = int(float(length.max()) / spacing * 2.0 + 40.0)
    gaps = st.expo(n_seg * m).reshape(n_seg, m) * spacing
    pos = np.cumsum(gaps, axis=1)
    assert np.all(pos[:, -1] >= length), "gap budget too small"
    keep = pos < length[:, None]
    seg = np.repeat(np.arange(n_seg), m).reshape(n_seg, m)[keep]
    s = pos[keep]
    return start[seg] + s[:, None] * dirs[seg], seg


def make_view(cfg: ViewConfig, *key: int):
    """One view: (grains int32 [N,4], truth int32 [N], lines float64 [T,7])."""
    st = Stream(*key)
    size = np.asarray(cfg.size_um, dtype=np.float64)
    n_fog = int(round(cfg.fog_per_1000um3 * 1e-3 * float(np.prod(size))))
    fog = st.uniform(3 * n_fog).reshape(n_fog, 3) * size

    if cfg.kind == "through":
        anchor = st.uniform(3 * cfg.n_tracks).reshape(cfg.n_tracks, 3) * size
        dirs = _iso_dirs(st, cfg.n_tracks)
        t0, t1 = _chord(anchor, dirs, size)
        start = anchor + t0[:, None] * dirs
        length = t1 - t0
    elif cfg.kind == "short":
        n = cfg.n_tracks
        start = np.zeros((n, 3)); dirs = np.zeros((n, 3)); length = np.zeros(n)
        todo = np.arange(n)
        while len(todo):
            s = st.uniform(3 * len(todo)).reshape(-1, 3) * size
            d = _iso_dirs(st, len(todo))
            ln = cfg.len_um[0] + (cfg.len_um[1] - cfg.len_um[0]) * st.uniform(len(todo))
            end = s + ln[:, None] * d
            ok = np.all((end >= 0.0) & (end <= size), axis=1)
            start[todo[ok]] = s[ok]; dirs[todo[ok]] = d[ok]; length[todo[ok]] = ln[ok]
            todo = todo[~ok]
    elif cfg.kind == "stars":
        vtx = st.uniform(3 * cfg.n_tracks).reshape(cfg.n_tracks, 3) * size
        n_pr = st.integers(cfg.prongs[0], cfg.prongs[1], cfg.n_tracks)
        start = np.repeat(vtx, n_pr, axis=0)
        n = len(start)
        dirs = _iso_dirs(st, n)
        ln = cfg.len_um[0] + (cfg.len_um[1] - cfg.len_um[0]) * st.uniform(n)
        _, t1 = _chord(start, dirs, size)
        length = np.minimum(ln, t1)
    else:
        raise ValueError(cfg.kind)

    pts, seg = _poisson_process(st, start, dirs, length, cfg.spacing_um)
    xyz = np.concatenate([fog, pts], axis=0)
    truth = np.concatenate([np.full(n_fog, -1, np.int64), seg])
    sig = np.asarray(cfg.sigma_um, dtype=np.float64)
    xyz = xyz + st.normal(3 * len(xyz)).reshape(-1, 3) * sig
    q = np.floor(xyz * Q_PER_UM + 0.5).astype(np.int64)
    size_q = np.round(size * Q_PER_UM).astype(np.int64)
    q = np.clip(q, 0, size_q - 1)
    perm = st.permutation(len(q))
    grains = np.zeros((len(q), 4), dtype=np.int32)
    grains[:, :3] = q[perm]
    lines = np.concatenate([start, dirs, length[:, None]], axis=1)
    return grains, truth[perm].astype(np.int32), lines


def make_batch(cfg: ViewConfig, config_index: int, n_views: int | None = None,
               first_view: int = 0) -> ViewBatch:
    """Views first_view .. first_view+n_views-1 of a config; view v uses key (config_index, v)."""
    n_views = cfg.n_views if n_views is None else n_views
    gs, ts, ls, off = [], [], [], [0]
    for v in range(first_view, first_view + n_views):
        g, t, l = make_view(cfg, config_index, v)
        gs.append(g); ts.append(t); ls.append(l); off.append(off[-1] + len(g))
    return ViewBatch(np.concatenate(gs), np.asarray(off, np.int32), np.concatenate(ts), ls, cfg)


def make_config(config_index: int, n_views: int | None = None, first_view: int = 0) -> ViewBatch:
    return make_batch(CONFIGS[config_index], config_index, n_views, first_view)


def noiseless_track_view(size_q, tracks, n_fog: int = 0, key=(99, 0)) -> ViewBatch:
    """Hand-built view for the exact-recovery checks: every track is a list of
    integer points given by the caller (already on the q lattice, no smear);
    optional uniform integer fog.  No arithmetic of the method is involved."""
    st = Stream(*key)
    pts, truth = [], []
    for i, tr in enumerate(tracks):
        tr = np.asarray(tr, dtype=np.int64).reshape(-1, 3)
        pts.append(tr); truth.append(np.full(len(tr), i, np.int64))
    if n_fog:
        f = np.floor(st.uniform(3 * n_fog).reshape(n_fog, 3) * np.asarray(size_q)).astype(np.int64)
        pts.append(f); truth.append(np.full(n_fog, -1, np.int64))
    xyz = np.concatenate(pts) if pts else np.zeros((0, 3), np.int64)
    tr = np.concatenate(truth) if truth else np.zeros(0, np.int64)
    grains = np.zeros((len(xyz), 4), np.int32)
    grains[:, :3] = xyz
    return ViewBatch(grains, np.asarray([0, len(xyz)], np.int32), tr.astype(np.int32), [], None)
