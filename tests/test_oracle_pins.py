"""Pins for the CPU oracle (CPU only, -m "not gpu").

Each test ties oracle/ to something other than itself: the hand-derived example E1
(tests/golden), an exact-rational brute force over all grain triples written the other
way round (tests/exact_bruteforce.py), constructions whose answer is known (noiseless
tracks, crossing tracks, the tube-boundary witness), invariances (grain permutation,
x<->y swap, cell size), numpy.polyfit for the fit, and Poisson closed forms.
"""
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from emu_synth import CONFIGS, default_params, make_batch, make_config, noiseless_track_view
from emu_synth.views import Stream
from exact_bruteforce import fit_exact, track_view_exact

HERE = os.path.dirname(os.path.abspath(__file__))
BJ = dict(sep_min_q=256, sep_max_q=1280, tube_r2_q=2621, tube_ext_q=-1, min_grains=8, max_tracks_per_view=256)


def _params(size_q, cell_q=(512, 512, 512), **kw):
    p = dict(BJ, view_size_q=tuple(size_q), cell_size_q=tuple(cell_q))
    p.update(kw)
    return p


def _arr(points):
    g = np.zeros((len(points), 4), np.int32)
    g[:, :3] = np.asarray(points, np.int64).reshape(-1, 3)
    return g, np.asarray([0, len(points)], np.int32)


def _track_list(res):
    """Canonical python view of an OracleResult: list of (view, a, b, n_tube, n_members, d2, members)."""
    out = []
    for t in res.tracks:
        m = res.members[t["member_off"]:t["member_off"] + t["n_members"]]
        out.append((int(t["view"]), int(t["seed_a"]), int(t["seed_b"]), int(t["n_tube"]), int(t["n_members"]),
                    int(t["seed_d2"]), tuple(int(x) for x in m)))
    return out


def _same(r1, r2):
    return (r1.tracks.tobytes() == r2.tracks.tobytes() and r1.members.tobytes() == r2.members.tobytes()
            and r1.track_off.tobytes() == r2.track_off.tobytes() and r1.fits.tobytes() == r2.fits.tobytes())


# --------------------------------------------------------------------------- E1 (golden)

@pytest.fixture(scope="module")
def e1():
    with open(os.path.join(HERE, "golden", "e1_constructed_example.json")) as f:
        return json.load(f)


@pytest.mark.parametrize("mode", ["brute", "cells"])
def test_e1_constructed_example(oracle_mod, e1, mode):
    g, off = _arr(e1["grains"])
    r = oracle_mod.track_views(e1["params"], g, off, mode, 1, seed_dump=True)
    assert r.counters["seeds"] == e1["n_seeds"]
    assert r.counters["candidates"] == e1["n_candidates"]
    on = [row for row in r.seed_dump if row[1] <= 8 and row[2] <= 8]
    off_track = [row for row in r.seed_dump if row[2] >= 9]
    assert len(on) == e1["n_on_track_seeds"] and all(row[3] == e1["on_track_n_tube"] for row in on)
    assert len(off_track) == e1["n_seeds"] - e1["n_on_track_seeds"]
    assert sorted(set(int(row[3]) for row in off_track)) == e1["off_track_n_tube_values"]
    assert len(r.tracks) == e1["n_tracks"] == 1
    t, tg = r.tracks[0], e1["track"]
    for k in ("seed_a", "seed_b", "n_tube", "n_members", "seed_d2"):
        assert int(t[k]) == tg[k], k
    assert list(r.members) == tg["members"]
    f, fg = r.fits[0], e1["fit"]
    assert (int(f["axis"]), int(f["n"]), int(f["u_min"]), int(f["u_max"])) == (fg["axis"], fg["n"], fg["u_min"], fg["u_max"])
    for i in range(2):
        assert abs(f["slope"][i] - fg["slope"][i]) < fg["slope_abs_tol"]
        assert abs(f["icpt"][i] - fg["icpt"][i]) < fg["icpt_abs_tol"]
    # the sums the golden file quotes, rebuilt from its own numbers
    assert Fraction(fg["num_y"], fg["den"]) == Fraction(10 * 12570000 - fg["Su"] * 10050, 10 * fg["Suu"] - fg["Su"] ** 2)
    assert abs(float(Fraction(fg["num_y"], fg["den"])) - f["slope"][0]) < 1e-15
    assert abs(float(Fraction(fg["num_z"], fg["den"])) - f["slope"][1]) < 1e-15


def test_e1_mirrored_and_permuted(oracle_mod, e1):
    pts = np.asarray(e1["grains"], np.int64)
    g, off = _arr(pts)
    r0 = oracle_mod.track_views(e1["params"], g, off, "cells", 1)
    perm = Stream(7, 7).permutation(len(pts))
    g2, _ = _arr(pts[perm][:, [1, 0, 2]])          # x <-> y swapped and rows permuted
    r1 = oracle_mod.track_views(e1["params"], g2, off, "cells", 1)
    inv = np.empty(len(perm), np.int64); inv[perm] = np.arange(len(perm))   # old row -> new row
    t0, t1 = _track_list(r0), _track_list(r1)
    assert len(t0) == len(t1) == 1
    assert {inv[t0[0][1]], inv[t0[0][2]]} == {t1[0][1], t1[0][2]}
    assert sorted(inv[list(t0[0][6])]) == list(t1[0][6])
    assert t0[0][3:6] == t1[0][3:6]


# --------------------------------------------------------------------------- exact brute force on tiny inputs

def _tiny_view(key, n_fog=36, box=(2200, 2000, 1800)):
    """A small crowded box: fog + two short noisy lines, so seeds, candidates, ties and sharing all occur."""
    st = Stream(*key)
    pts = np.floor(st.uniform(3 * n_fog).reshape(n_fog, 3) * np.asarray(box)).astype(np.int64)
    extra = []
    for (p0, d) in (((200, 300, 250), (150, 90, 60)), ((1900, 250, 300), (-140, 100, 70))):
        for i in range(11):
            j = np.floor(st.uniform(3) * 30).astype(np.int64) - 15
            extra.append([p0[0] + i * d[0] + j[0], p0[1] + i * d[1] + j[1], p0[2] + i * d[2] + j[2]])
    return np.concatenate([pts, np.asarray(extra, np.int64)])


@pytest.mark.parametrize("key", [(1, 1), (1, 2), (1, 3)])
@pytest.mark.parametrize("mode", ["brute", "cells"])
def test_all_triples_exact_rational(oracle_mod, key, mode):
    pts = _tiny_view(key)
    p = _params((2200, 2000, 1800), cell_q=(300, 512, 700), min_grains=5)
    ref = track_view_exact([tuple(int(c) for c in q) for q in pts], p)
    g, off = _arr(pts)
    r = oracle_mod.track_views(p, g, off, mode, 1, seed_dump=True)
    got = {(int(a), int(b)): int(n) for _, a, b, n in r.seed_dump}
    assert got == ref["seeds"]                                  # O2 + O3: every seed, every count
    assert r.counters["candidates"] == ref["n_candidates"]      # O4
    assert len(ref["tracks"]) >= 2
    tl = _track_list(r)                                         # O5 + O7
    assert [(t[1], t[2], t[3], t[5], t[6]) for t in tl] == \
           [(t["seed_a"], t["seed_b"], t["n_tube"], t["seed_d2"], tuple(t["members"])) for t in ref["tracks"]]
    for t, f in zip(ref["tracks"], r.fits):                     # O6
        fx = fit_exact([tuple(int(c) for c in pts[m]) for m in t["members"]])
        assert int(f["axis"]) == fx["axis"] and int(f["n"]) == fx["n"]
        assert (int(f["u_min"]), int(f["u_max"])) == (fx["u_min"], fx["u_max"])
        for i in range(2):
            assert abs(f["slope"][i] - float(fx["slope"][i])) <= 1e-12 * max(1.0, abs(float(fx["slope"][i])))
            assert abs(f["icpt"][i] - float(fx["icpt"][i])) <= 1e-9 * max(1.0, abs(float(fx["icpt"][i])))


def test_tube_boundary_witness(oracle_mod):
    """Reading Q3: r2 = 2621 = 50^2 + 11^2, closed tube: (t,50,11) is in, (t,50,12) is out."""
    base = [(0, 500, 500), (640, 500, 500)]                    # x-directed seed, 10 um apart
    for dz, expect in ((11, 3), (12, 2)):
        g, off = _arr(base + [(300, 550, 500 + dz)])
        p = _params((2000, 2000, 2000), min_grains=2)
        r = oracle_mod.track_views(p, g, off, "brute", 1, seed_dump=True)
        d = {(int(a), int(b)): int(n) for _, a, b, n in r.seed_dump}
        assert d[(0, 1)] == expect


def test_separation_window_bounds(oracle_mod):
    """Reading Q1: sep_min^2 <= D2 < sep_max^2 (lower inclusive, upper strict, "smaller than")."""
    for dist, is_seed in ((255, False), (256, True), (1279, True), (1280, False)):
        g, off = _arr([(100, 100, 100), (100 + dist, 100, 100)])
        r = oracle_mod.track_views(_params((4000, 4000, 3200), min_grains=2), g, off, "cells", 1)
        assert r.counters["seeds"] == (1 if is_seed else 0)


# --------------------------------------------------------------------------- constructions with known answers

def _line(p0, d, n):
    return [(p0[0] + i * d[0], p0[1] + i * d[1], p0[2] + i * d[2]) for i in range(n)]


@pytest.mark.parametrize("direction", [(300, 0, 0), (0, 0, 290), (200, 150, 100), (-170, 210, 40), (90, -60, 250)])
def test_exact_recovery_of_a_noiseless_track(oracle_mod, direction):
    """One isolated noiseless track with end-to-end grains -> exactly one track, members = the injected grains."""
    n = 11
    start = (4000 - 5 * direction[0], 4000 - 5 * direction[1], 1600 - 5 * direction[2])
    far_fog = [(100, 100, 100), (7900, 200, 3000), (300, 7800, 50)]          # isolated grains, far away
    b = noiseless_track_view((8000, 8000, 3200), [_line(start, direction, n)])
    g = np.concatenate([b.grains, _arr(far_fog)[0]])
    off = np.asarray([0, len(g)], np.int32)
    for mode in ("brute", "cells"):
        r = oracle_mod.track_views(_params((8000, 8000, 3200)), g, off, mode, 1)
        tl = _track_list(r)
        assert len(tl) == 1
        assert tl[0][6] == tuple(range(n)) and tl[0][3] == n and tl[0][4] == n
        f = r.fits[0]
        u = int(f["axis"])
        minors = {2: (0, 1), 0: (1, 2), 1: (0, 2)}[u]
        for i, m in enumerate(minors):                      # slope = direction ratio exactly (points are on the lattice)
            assert abs(f["slope"][i] - direction[m] / direction[u]) < 1e-12


def test_two_tracks_crossing_at_a_shared_grain(oracle_mod):
    """The shared grain goes to the track with more grains (SURVEY 8(c) O5 pins)."""
    cross = (4000, 4000, 1600)
    long_t = _line((4000 - 7 * 280, 4000, 1600), (280, 0, 0), 15)       # 15 grains along x, contains `cross`
    short_t = [q for q in _line((4000, 4000 - 5 * 270, 1600 - 5 * 60), (0, 270, 60), 11) if q != cross]  # 10 more
    pts = long_t + short_t
    g, off = _arr(pts)
    r = oracle_mod.track_views(_params((8000, 8000, 3200)), g, off, "cells", 1)
    tl = _track_list(r)
    assert len(tl) == 2
    shared = pts.index(cross)
    assert tl[0][3] == 15 and tl[0][4] == 15 and shared in tl[0][6]
    assert tl[1][3] == 11 and tl[1][4] == 10 and shared not in tl[1][6]
    assert set(tl[0][6]) == set(range(15)) and set(tl[1][6]) == set(range(15, 25))


def test_loser_grains_stay_unassigned(oracle_mod):
    """Reading Q8: one round only.  An 8-grain line crossing a 12-grain line at one shared grain is a
    candidate (n_tube = 8) but keeps only 7 members -> dropped by the second threshold, and its
    remaining 7 grains are handed to nobody."""
    main = _line((1000, 4000, 1600), (300, 0, 0), 12)
    other = [(main[5][0], main[5][1] + k * 300, main[5][2]) for k in range(-4, 4) if k != 0]   # 7 own grains
    pts = main + other
    g, off = _arr(pts)
    ref = track_view_exact(pts, _params((8000, 8000, 3200)))
    assert ref["seeds"][(12, 13)] == 8                          # the short line is a candidate ...
    for mode in ("brute", "cells"):
        r = oracle_mod.track_views(_params((8000, 8000, 3200)), g, off, mode, 1)
        tl = _track_list(r)
        assert len(tl) == 1 and tl[0][6] == tuple(range(12))    # ... but only the long line survives
        assert [(t[1], t[2], t[6]) for t in tl] == [(t["seed_a"], t["seed_b"], tuple(t["members"])) for t in ref["tracks"]]


# --------------------------------------------------------------------------- invariances on config 0

def test_cells_equal_brute_on_config0(oracle_mod, config_oracle):
    b, p, r = config_oracle(0)
    rb = oracle_mod.track_views(p, b.grains, b.view_off, "brute", 1, seed_dump=True)
    assert _same(r, rb)
    assert sorted(map(tuple, r.seed_dump)) == sorted(map(tuple, rb.seed_dump))
    assert r.counters["seeds"] == rb.counters["seeds"] and r.counters["tube_tests"] < rb.counters["tube_tests"]


@pytest.mark.parametrize("cell_um", [(3.0, 3.0, 3.0), (5.5, 13.0, 2.0), (40.0, 7.0, 60.0)])
def test_cell_size_has_no_effect(oracle_mod, config_oracle, cell_um):
    b, p, r = config_oracle(0)
    p2 = default_params(0, cell_um=cell_um)
    assert _same(r, oracle_mod.track_views(p2, b.grains, b.view_off, "cells", 1))


def test_grains_outside_the_box_are_legal(oracle_mod):
    """Reading Q13: out-of-box grains are clamped into boundary cells and take part in everything."""
    b = make_config(0)
    g = b.grains.copy()
    g[:, 0] -= 900; g[:, 1] += 700; g[:, 2] -= 300            # push a good part of the cloud outside [0,size)
    p = default_params(0)
    r1 = oracle_mod.track_views(p, g, b.view_off, "cells", 1)
    r2 = oracle_mod.track_views(p, g, b.view_off, "brute", 1)
    assert len(r1.tracks) >= 5 and _same(r1, r2)


def test_grain_order_permutation(oracle_mod, config_oracle):
    b, p, r = config_oracle(0)
    perm = Stream(5, 5).permutation(b.n_grains)
    r2 = oracle_mod.track_views(p, b.grains[perm], b.view_off, "cells", 1)
    inv = np.empty(len(perm), np.int64); inv[perm] = np.arange(len(perm))
    t1, t2 = _track_list(r), _track_list(r2)
    assert len(t1) == len(t2)
    for a, c in zip(t1, t2):
        assert a[3:6] == c[3:6]
        assert (min(inv[a[1]], inv[a[2]]), max(inv[a[1]], inv[a[2]])) == (c[1], c[2])
        assert tuple(sorted(inv[list(a[6])])) == c[6]


def test_xy_swap(oracle_mod, config_oracle):
    b, p, r = config_oracle(0)                                  # config 0's box is square in x,y
    g = b.grains[:, [1, 0, 2, 3]].copy()
    r2 = oracle_mod.track_views(p, g, b.view_off, "cells", 1)
    t1, t2 = _track_list(r), _track_list(r2)
    assert t1 == t2
    for f1, f2, t in zip(r.fits, r2.fits, r.tracks):
        assert int(f1["n"]) == int(f2["n"])
        if int(f1["axis"]) == 2:                                # minors (x,y) swap
            assert int(f2["axis"]) == 2
            assert f1["slope"][0] == f2["slope"][1] and f1["icpt"][1] == f2["icpt"][0]
        else:
            assert {int(f1["axis"]), int(f2["axis"])} == {0, 1}
            assert f1["slope"][1] == f2["slope"][1]            # z-slope on the swapped dominant axis


# --------------------------------------------------------------------------- O1 binning

def test_paper_cell_count(oracle_mod):
    """1280x1024 px x 40 frames in cells of 32x32 px x 1 frame -> 51 200 cells."""
    p = _params((1280, 1024, 40), cell_q=(32, 32, 1))
    assert oracle_mod.grid_dims(p) == (40, 32, 40)
    assert math.prod(oracle_mod.grid_dims(p)) == 51200


def test_binning_invariants(oracle_mod):
    b = make_config(3, n_views=1)
    b2 = make_batch(CONFIGS[0], 0, n_views=3)
    for batch, c in ((b, 3), (b2, 0)):
        p = default_params(c, cell_um=(8.0, 6.0, 5.0))
        g = batch.grains.copy()
        g[::17, 0] -= 2000; g[::23, 2] += 5000                 # some out-of-box grains
        srt, cs = oracle_mod.bin_grains(p, g, batch.view_off)
        nx, ny, nz = oracle_mod.grid_dims(p)
        nc = nx * ny * nz
        assert len(cs) == batch.n_views * nc + 1 and cs[0] == 0 and cs[-1] == batch.n_grains
        assert np.all(np.diff(cs) >= 0)
        assert sorted(srt[:, 3]) == list(range(batch.n_grains))         # a permutation of the rows
        assert np.array_equal(srt[:, :3], g[srt[:, 3], :3])
        for v in range(batch.n_views):
            assert cs[v * nc] == batch.view_off[v]
        # each sorted grain sits in the cell the definition gives; rows ascend inside a cell
        cell_of_slot = np.repeat(np.arange(batch.n_views * nc), np.diff(cs))
        cx = np.clip(np.floor_divide(srt[:, 0], p["cell_size_q"][0]), 0, nx - 1)
        cy = np.clip(np.floor_divide(srt[:, 1], p["cell_size_q"][1]), 0, ny - 1)
        cz = np.clip(np.floor_divide(srt[:, 2], p["cell_size_q"][2]), 0, nz - 1)
        view_of_slot = np.searchsorted(batch.view_off, np.arange(batch.n_grains), side="right") - 1
        assert np.array_equal(cell_of_slot, view_of_slot * nc + cx + nx * (cy + ny * cz))
        same_cell = cell_of_slot[1:] == cell_of_slot[:-1]
        assert np.all(srt[1:, 3][same_cell] > srt[:-1, 3][same_cell])


# --------------------------------------------------------------------------- O6 fit

def test_fit_against_polyfit_and_fractions(oracle_mod):
    st = Stream(11, 3)
    tracks, members, off = [], [], [0]
    rows = []
    for k in range(12):
        n = 8 + 3 * k
        d = (st.uniform(3) * 2 - 1)
        d /= np.linalg.norm(d)
        p0 = st.uniform(3) * np.asarray([20000, 18000, 3000])
        t = np.sort(st.uniform(n)) * 6000
        pts = np.floor(p0 + t[:, None] * d + st.normal(3 * n).reshape(n, 3) * [6, 6, 30] + 0.5).astype(np.int64)
        base = len(rows)
        rows.extend(pts.tolist())
        members.extend(range(base, base + n)); off.append(off[-1] + n)
    g, _ = _arr(rows)
    fits = oracle_mod.fit_tracks(g, members, off)
    for k, f in enumerate(fits):
        pts = np.asarray(rows[off[k]:off[k + 1]], np.float64)
        fx = fit_exact([tuple(int(c) for c in q) for q in rows[off[k]:off[k + 1]]])
        u = int(f["axis"]); assert u == fx["axis"]
        minors = {2: (0, 1), 0: (1, 2), 1: (0, 2)}[u]
        for i, m in enumerate(minors):
            s, c = np.polyfit(pts[:, u], pts[:, m], 1)          # library least squares
            assert abs(f["slope"][i] - s) <= 1e-9 * max(1.0, abs(s))
            assert abs(f["icpt"][i] - c) <= 1e-9 * max(1.0, abs(c))
            assert abs(f["slope"][i] - float(fx["slope"][i])) <= 1e-13 * max(1.0, abs(float(fx["slope"][i])))


def test_fit_degenerate_all_members_share_u(oracle_mod):
    rows = [(500, 700, 900)] * 8                                  # 8 coincident grains: den = 0
    g, _ = _arr(rows)
    f = oracle_mod.fit_tracks(g, list(range(8)), [0, 8])[0]
    assert int(f["axis"]) == (2 | 0x100) and int(f["n"]) == 8
    assert tuple(f["slope"]) == (0.0, 0.0) and tuple(f["icpt"]) == (500.0, 700.0)


# --------------------------------------------------------------------------- whole path: physics sanity

def _score(batch, res, min_grains=8):
    """findable / found / fakes (SURVEY 8(d) 'Physics quality')."""
    findable = found = fakes = 0
    per_track_cos = []
    for v in range(batch.n_views):
        lo, hi = batch.view_off[v], batch.view_off[v + 1]
        truth = batch.truth[lo:hi]
        n_true = np.bincount(truth[truth >= 0], minlength=len(batch.lines[v]))
        owners = set()
        for t in res.tracks[res.track_off[v]:res.track_off[v + 1]]:
            m = res.members[t["member_off"]:t["member_off"] + t["n_members"]]
            lab = batch.truth[m]
            lab = lab[lab >= 0]
            best = np.bincount(lab).argmax() if len(lab) else -1
            if best >= 0 and (batch.truth[m] == best).sum() >= 0.7 * len(m):
                owners.add(int(best))
            else:
                fakes += 1
        for tid in range(len(batch.lines[v])):
            if n_true[tid] >= min_grains:
                findable += 1
                ok = tid in owners
                found += ok
                per_track_cos.append((abs(batch.lines[v][tid][5]), ok))
    return findable, found, fakes, per_track_cos


def test_efficiency_and_fakes_on_generated_tracks(oracle_mod):
    """Config-0-shaped views: nearly every findable track is found, few fakes, no collapse at any angle
    (efficiency 'almost constant as a function of the track angle')."""
    batch = make_batch(CONFIGS[0], 0, n_views=12)
    res = oracle_mod.track_views(default_params(0), batch.grains, batch.view_off, "cells", 0)
    findable, found, fakes, per = _score(batch, res)
    assert findable >= 100
    assert found / findable >= 0.93
    assert fakes <= 3 * batch.n_views
    steep = [ok for c, ok in per if c >= 0.5]
    flat = [ok for c, ok in per if c < 0.5]
    assert np.mean(steep) >= 0.85 and np.mean(flat) >= 0.85
    # closed form: a vertical 50 um track carries Poisson(50/3) grains; P(n >= 8) = 99.3 % bounds what can be found
    lam = 50.0 / 3.0
    p_ge8 = 1.0 - sum(math.exp(-lam) * lam ** k / math.factorial(k) for k in range(8))
    assert abs(p_ge8 - 0.993) < 2e-3


def test_seed_density_closed_form(oracle_mod, config_oracle):
    """O2 against the closed form for uniform fog: partners per grain in the 4..20 um shell of a 50 um slab.
    rho*(4pi/3)(20^3-4^3) with the slab truncation averaged analytically over z."""
    b, p, r = config_oracle(1)
    n = b.n_grains
    vol = 350.0 * 300.0 * 50.0
    # mean over z0 in [0,50] of the shell volume inside the slab: V(R) - (pi/ (50)) * R^4 / 2  (two caps, averaged)
    def slab_ball(R, Z=50.0):
        return 4.0 / 3.0 * math.pi * R ** 3 - math.pi * R ** 4 / (2.0 * Z)
    expect_pairs = 0.5 * n * (n / vol) * (slab_ball(20.0) - slab_ball(4.0))
    # tracks add correlated pairs and the x,y edges remove some: the fog-only closed form must hold within 15 %
    assert 0.85 * expect_pairs < r.counters["seeds"] < 1.25 * expect_pairs


# --------------------------------------------------------------------------- bounded tube

@pytest.mark.parametrize("ext", [0, 200, 1280])
@pytest.mark.parametrize("mode", ["brute", "cells"])
def test_bounded_tube_all_triples_exact_rational(oracle_mod, mode, ext):
    """tube_ext_q >= 0: every seed's count and the whole track list against the exact-rational brute force, whose
    axial condition is written through the foot parameter lam = (v.d)/D2 instead of the oracle's squared products."""
    pts = _tiny_view((1, 2))
    p = _params((2200, 2000, 1800), cell_q=(300, 512, 700), min_grains=4, tube_ext_q=ext)
    ref = track_view_exact([tuple(int(c) for c in q) for q in pts], p)
    g, off = _arr(pts)
    r = oracle_mod.track_views(p, g, off, mode, 1, seed_dump=True)
    got = {(int(a), int(b)): int(n) for _, a, b, n in r.seed_dump}
    assert got == ref["seeds"]
    assert r.counters["candidates"] == ref["n_candidates"]
    tl = _track_list(r)
    assert [(t[1], t[2], t[3], t[5], t[6]) for t in tl] == \
           [(t["seed_a"], t["seed_b"], t["n_tube"], t["seed_d2"], tuple(t["members"])) for t in ref["tracks"]]
    whole = oracle_mod.track_views(dict(p, tube_ext_q=-1), g, off, mode, 1, seed_dump=True)
    w = {(int(a), int(b)): int(n) for _, a, b, n in whole.seed_dump}
    assert all(got[k] <= w[k] for k in w) and any(got[k] < w[k] for k in w)      # bounding can only remove grains


def test_bounded_tube_axial_witness(oracle_mod):
    """x-directed seed A = (1000,500,500), B = (1640,500,500) (|d| = 640), ext = 100: a grain on the line is counted
    iff its x lies in [900, 1740] (closed at both ends); ext = 0 keeps [1000, 1640]; the seed grains always count."""
    base = [(1000, 500, 500), (1640, 500, 500)]
    for ext, x, expect in ((100, 900, 3), (100, 899, 2), (100, 1740, 3), (100, 1741, 2), (0, 999, 2), (0, 1641, 2),
                           (0, 1300, 3), (-1, 100, 3), (-1, 3900, 3)):
        g, off = _arr(base + [(x, 500, 500)])
        p = _params((4000, 2000, 2000), min_grains=2, sep_min_q=640, sep_max_q=641, tube_ext_q=ext)
        r = oracle_mod.track_views(p, g, off, "brute", 1, seed_dump=True)
        d = {(int(a), int(b)): int(n) for _, a, b, n in r.seed_dump}
        assert d == {(0, 1): expect}, (ext, x)
    # a skew seed, d = (300, 400, 0), |d| = 500, ext = 50: the grain at A - 0.1 d = (-30, -40) off A is at axial
    # distance 50 (in), at A - 0.102 d it is out; exact at the boundary: s = -25 000, s^2 = 6.25e8 = 50^2 * 250 000
    A, B = (1000, 1000, 500), (1300, 1400, 500)
    for P3, expect in (((970, 960, 500), 3), ((969, 959, 500), 2)):
        g, off = _arr([A, B, P3])
        p = _params((4000, 4000, 2000), min_grains=2, sep_min_q=450, sep_max_q=550, tube_ext_q=50)
        r = oracle_mod.track_views(p, g, off, "brute", 1, seed_dump=True)
        assert {(int(a), int(b)): int(n) for _, a, b, n in r.seed_dump} == {(0, 1): expect}


def test_bounded_tube_is_orientation_and_order_free(oracle_mod, config_oracle):
    """x<->y swap and grain-order permutation leave the bounded-tube track list unchanged (after mapping)."""
    b, p, _ = config_oracle(0)
    p = dict(p, tube_ext_q=640)
    r0 = oracle_mod.track_views(p, b.grains, b.view_off, "cells", 1)
    perm = np.random.default_rng(5).permutation(len(b.grains))
    gp = b.grains[perm]
    r1 = oracle_mod.track_views(p, gp, b.view_off, "cells", 1)
    inv = perm                                   # new row i holds old row perm[i]
    t0 = sorted((min(t["seed_a"], t["seed_b"]), max(t["seed_a"], t["seed_b"]), t["n_tube"], t["n_members"]) for t in r0.tracks)
    t1 = sorted((min(inv[t["seed_a"]], inv[t["seed_b"]]), max(inv[t["seed_a"]], inv[t["seed_b"]]), t["n_tube"], t["n_members"])
                for t in r1.tracks)
    assert t0 == t1 and len(t0) > 0
    gs = b.grains.copy(); gs[:, [0, 1]] = gs[:, [1, 0]]
    ps = dict(p, view_size_q=(p["view_size_q"][1], p["view_size_q"][0], p["view_size_q"][2]),
              cell_size_q=(p["cell_size_q"][1], p["cell_size_q"][0], p["cell_size_q"][2]))
    r2 = oracle_mod.track_views(ps, gs, b.view_off, "cells", 1)
    assert r2.tracks.tobytes() == r0.tracks.tobytes() and r2.members.tobytes() == r0.members.tobytes()


# --------------------------------------------------------------------------- later keys of the order (golden)

@pytest.fixture(scope="module")
def tie_cases():
    with open(os.path.join(HERE, "golden", "tie_break_keys.json")) as f:
        return json.load(f)


def _check_golden_tracks(res, tracks):
    assert len(res.tracks) == len(tracks)
    for t, g in zip(res.tracks, tracks):
        for k in ("seed_a", "seed_b", "n_tube", "n_members", "seed_d2"):
            assert int(t[k]) == g[k], (k, int(t[k]), g[k])
        assert [int(x) for x in res.members[t["member_off"]:t["member_off"] + t["n_members"]]] == g["members"]


@pytest.mark.parametrize("mode", ["brute", "cells"])
@pytest.mark.parametrize("case", range(5))
def test_tie_break_keys_golden(oracle_mod, tie_cases, case, mode):
    """min(x,y), x, row of kmin and kmax decide: hand-derived winners, tests/golden."""
    c = tie_cases["cases"][case]
    g, off = _arr(c["grains"])
    r = oracle_mod.track_views(tie_cases["params"], g, off, mode, 1)
    assert r.counters["seeds"] == c["n_seeds"] and r.counters["candidates"] == c["n_candidates"]
    _check_golden_tracks(r, c["tracks"])


def test_tie_break_keys_mirror_images(oracle_mod, tie_cases):
    """x <-> y swap of a whole view maps k onto itself except at the x component, so the 'x decides' and 'kmax
    decides' cases must hand the shared grain to the OTHER line, and the others must not notice."""
    p = tie_cases["params"]
    for c in tie_cases["cases"]:
        g, off = _arr(c["grains"])
        gs = g.copy(); gs[:, 0], gs[:, 1] = g[:, 1].copy(), g[:, 0].copy()
        r, rs = oracle_mod.track_views(p, g, off, "brute", 1), oracle_mod.track_views(p, gs, off, "brute", 1)
        a, b = _track_list(r), _track_list(rs)
        if c["name"] in ("x_decides", "kmax_decides"):
            assert a != b and sorted(len(t[6]) for t in a) == sorted(len(t[6]) for t in b) == [8, 9]
            assert set(a[0][6]) != set(b[0][6])                      # the 9-member track is the other line
        else:
            assert a == b


@pytest.mark.parametrize("cfg", [1, 3])
def test_cells_equal_brute_on_a_full_view(oracle_mod, config_oracle, cfg):
    """Mode 'cells' (the reference of every GPU parity test and of the roofline's tests per seed) against mode
    'brute' (every seed against every grain, no cells) on one full 350 x 300 x 50 um view: config 1 (1.5 M seeds x 23.6 k
    grains = 3.5e10 integer tests) and config 3.  The brute pair loop is shared among the host cores."""
    b, p, ref = config_oracle(cfg)
    r = oracle_mod.track_views(p, b.grains, b.view_off, "brute", 0, seed_dump=True)
    assert r.counters["seeds"] == ref.counters["seeds"] and r.counters["candidates"] == ref.counters["candidates"]
    assert _same(r, ref)
    a, c = r.seed_dump, ref.seed_dump
    assert np.array_equal(a[np.lexsort((a[:, 2], a[:, 1], a[:, 0]))], c[np.lexsort((c[:, 2], c[:, 1], c[:, 0]))])


# --------------------------------------------------------------------------- NEXT-2: angle-dependent cut

@pytest.fixture(scope="module")
def angle_golden():
    with open(os.path.join(HERE, "golden", "angle_cut_tracks.json")) as f:
        return json.load(f)


@pytest.mark.parametrize("mode", ["brute", "cells"])
def test_angle_cut_golden(oracle_mod, angle_golden, mode):
    """PAPER.md:144 / Fig. 8(c): the hand-built view of tests/golden/angle_cut_tracks.json - a
    horizontal 8-grain line the table removes, a steep one it keeps, two tracks just either side of a bin edge."""
    G = angle_golden
    g, off = _arr(G["grains"])
    for case in G["cases"]:
        p = dict(G["params"], angle_min_grains=case["angle_min_grains"])
        r = oracle_mod.track_views(p, g, off, mode, 1)
        assert r.counters["seeds"] == G["n_seeds"] and r.counters["candidates"] == G["n_candidates"]
        _check_golden_tracks(r, [G["tracks"][name] for name in case["order"]])


def _cos_bin_exact(points):
    """bin of |cos theta| of the least-squares line, from the exact rational fit (cov/var form of exact_bruteforce)."""
    f = fit_exact(points)
    if f["degenerate"]:
        return -1
    u = f["axis"]
    d = {u: Fraction(1)}
    minor = {2: (0, 1), 0: (1, 2), 1: (0, 2)}[u]
    d[minor[0]], d[minor[1]] = f["slope"]
    cos2 = d[2] * d[2] / (d[0] * d[0] + d[1] * d[1] + d[2] * d[2])
    return max(k for k in range(8) if Fraction(k * k, 64) <= cos2)


def test_angle_cut_bins_against_exact_rationals(oracle_mod, config_oracle):
    """On a generated view (config 0 and config 3: smeared tracks of every direction) the tracks a one-bin table
    removes are exactly those whose exact-rational |cos theta| falls in that bin; the rest of the list, its order and
    the grains of the removed tracks (left unassigned) do not change."""
    for cfg in (0, 3):
        b, p, ref = config_oracle(cfg)
        xyz = b.grains[:, :3].astype(np.int64)
        bins = []
        for t in ref.tracks:
            m = ref.members[t["member_off"]:t["member_off"] + t["n_members"]]
            bins.append(_cos_bin_exact([tuple(int(v) for v in xyz[i]) for i in m]))
        bins = np.asarray(bins)
        assert len(set(bins.tolist())) >= 4
        for k in range(8):
            table = [0] * 8
            table[k] = 8191
            r = oracle_mod.track_views(dict(p, angle_min_grains=table), b.grains, b.view_off, "cells", 1)
            keep = np.nonzero(bins != k)[0]
            assert len(r.tracks) == len(keep)
            assert _track_list(r) == [_track_list(ref)[i] for i in keep]
        # a threshold between the member counts splits a bin
        k = int(np.bincount(bins[bins >= 0]).argmax())
        nm = np.sort(ref.tracks["n_members"][bins == k])
        thr = int(nm[len(nm) // 2]) + 1
        table = [0] * 8
        table[k] = thr
        r = oracle_mod.track_views(dict(p, angle_min_grains=table), b.grains, b.view_off, "cells", 1)
        keep = np.nonzero((bins != k) | (ref.tracks["n_members"] >= thr))[0]
        assert 0 < len(keep) < len(ref.tracks) and _track_list(r) == [_track_list(ref)[i] for i in keep]


def test_angle_cut_all_equal_table_changes_nothing(oracle_mod, e1, config_oracle):
    g, off = _arr(e1["grains"])
    base = oracle_mod.track_views(e1["params"], g, off, "brute", 1)
    for table in ([0] * 8, [8] * 8, [3] * 8):
        assert _same(base, oracle_mod.track_views(dict(e1["params"], angle_min_grains=table), g, off, "brute", 1))
    b, p, ref = config_oracle(2)
    assert _same(ref, oracle_mod.track_views(dict(p, angle_min_grains=[p["min_grains"]] * 8), b.grains, b.view_off, "cells", 1))
