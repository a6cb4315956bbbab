"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.

Bars (north_star): track lists, offsets, member lists, per-seed counts and the binning output are
bit-exact (integer work); fitted slopes / intercepts agree within 1e-5 relative.
"""
import json
import os

import numpy as np
import pytest

from emu_synth import CONFIGS, default_params, make_batch, make_config, noiseless_track_view
from gpu_helpers import assert_same_tracks, run_gpu, seed_dump_gpu

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def E():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    import paper_1311_5334_b200 as E
    E.exported_symbols()
    return E


def _mess_up(g, size_q):
    """push a share of the grains outside the box (legal, reading Q13) and set junk payloads"""
    g = g.copy()
    g[::7, 0] -= size_q[0] // 3; g[::11, 1] += size_q[1] // 2; g[::13, 2] -= 4000
    g[:, 3] = np.arange(len(g))[::-1] * 7 + 3
    return g


# (200, 200, 100) um: one cell per view with about 1 700 grains - the byte counters of the fast binning kernel
# overflow and the view is redone with 32-bit counters; (40, 2, 60) um: about 20 grains per cell (block rank sort)
@pytest.mark.parametrize("cfg,cell_um,messy", [(0, (8.0, 8.0, 8.0), False), (0, (3.0, 17.0, 5.5), True),
                                               (1, (8.0, 8.0, 8.0), False), (1, (4.0, 4.0, 4.0), True),
                                               (3, (40.0, 2.0, 60.0), False), (0, (200.0, 200.0, 100.0), False),
                                               (1, (3.0, 4.0, 4.0), False)])
def test_binning_bit_exact(E, oracle_mod, cfg, cell_um, messy):
    b = make_batch(CONFIGS[cfg], cfg, n_views=3 if cfg == 0 else 1)
    p = default_params(cfg, cell_um=cell_um)
    g = _mess_up(b.grains, p["view_size_q"]) if messy else b.grains
    srt, cs = oracle_mod.bin_grains(p, g, b.view_off)
    import torch
    prm = E.make_params(**{k: p[k] for k in ("view_size_q", "cell_size_q", "sep_min_q", "sep_max_q", "tube_r2_q", "min_grains")})
    B = E.PathBuffers(prm, len(g), b.n_views)
    E.emu_bin_grains(prm, torch.from_numpy(np.ascontiguousarray(g)).cuda(), torch.from_numpy(b.view_off).cuda(),
                     len(g), b.n_views, B.sorted, B.cell_start, B.status, B.ws)
    torch.cuda.synchronize()
    assert int(B.status.cpu()[0]) == 0
    assert np.array_equal(B.cell_start.cpu().numpy(), cs)
    assert np.array_equal(B.sorted.cpu().numpy(), srt)


# cells of 4 um and finer in y, z take the shared-memory brick kernels (4-byte grains, float test with the
# exact fallback); 8 um cells take the generic global-memory kernels.  The result may not depend on it.
CELLS = [(8.0, 8.0, 8.0), (4.0, 4.0, 4.0), (6.5, 3.0, 2.5)]


@pytest.mark.parametrize("cell_um", CELLS)
@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_per_seed_counts_bit_exact(E, config_oracle, cfg, cell_um):
    b, p, ref = config_oracle(cfg)
    p = dict(p, cell_size_q=default_params(cfg, cell_um=cell_um)["cell_size_q"])
    dump, counts = seed_dump_gpu(E, p, b.grains, b.view_off, ref.counters["seeds"] + 16)
    assert int(counts[E.EMU_CNT["seeds"]]) == ref.counters["seeds"]
    a = dump[np.lexsort((dump[:, 2], dump[:, 1], dump[:, 0]))]
    r = ref.seed_dump[np.lexsort((ref.seed_dump[:, 2], ref.seed_dump[:, 1], ref.seed_dump[:, 0]))]
    assert np.array_equal(a, r)


@pytest.mark.parametrize("cell_um", CELLS)
@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_track_list_bit_exact(E, config_oracle, cfg, cell_um):
    b, p, ref = config_oracle(cfg)
    p = dict(p, cell_size_q=default_params(cfg, cell_um=cell_um)["cell_size_q"])
    got = run_gpu(E, p, b.grains, b.view_off)
    assert_same_tracks(E, got, ref)
    assert len(got["tracks"]) > 0


@pytest.mark.parametrize("cell_um", [(2.0, 4.0, 4.0), (0.5, 4.0, 4.0)])
def test_several_bricks_per_frame(E, config_oracle, cell_um):
    """Config 1 with fine cells along u: the cell tables no longer fit one shared-memory brick.  2 um: two bricks per
    (view, frame), hit records with two ordinals; 0.5 um: more than four bricks, the records are switched off and every
    candidate is walked a second time.  Per-seed counts and the track list may not notice."""
    b, p, ref = config_oracle(1)
    p = dict(p, cell_size_q=default_params(1, cell_um=cell_um)["cell_size_q"])
    dump, counts = seed_dump_gpu(E, p, b.grains, b.view_off, ref.counters["seeds"] + 16)
    a = dump[np.lexsort((dump[:, 2], dump[:, 1], dump[:, 0]))]
    r = ref.seed_dump[np.lexsort((ref.seed_dump[:, 2], ref.seed_dump[:, 1], ref.seed_dump[:, 0]))]
    assert np.array_equal(a, r)
    assert_same_tracks(E, run_gpu(E, p, b.grains, b.view_off), ref)


@pytest.mark.parametrize("cell_um", [(4.0, 4.0, 4.0), (2.0, 16.0, 3.0), (100.0, 100.0, 50.0), (1.0, 9.0, 25.0)])
def test_cell_size_has_no_effect_on_gpu(E, config_oracle, cell_um):
    b, p, ref = config_oracle(0)
    got = run_gpu(E, default_params(0, cell_um=cell_um), b.grains, b.view_off)
    assert_same_tracks(E, got, ref)


def test_batch_of_views_in_several_chunks(E, oracle_mod):
    """7 views of config 0; a tight workspace forces several internal chunks; track_off/member_off continue."""
    b = make_batch(CONFIGS[0], 0, n_views=7)
    p = default_params(0)
    ref = oracle_mod.track_views(p, b.grains, b.view_off, "cells", 0)
    prm = E.make_params(**{k: p[k] for k in ("view_size_q", "cell_size_q", "sep_min_q", "sep_max_q", "tube_r2_q", "min_grains")})
    _, rec = E.emu_workspace_bytes(prm, b.n_grains, b.n_views)
    # the recommendation holds all 7 views at once; the minimum seed / candidate capacity (1 Mi seeds of 160 B:
    # geometry, counter and hit records) holds about 3 views of this shape at the default hint of 192 seeds per grain
    for ws in (None, 200 << 20):
        got = run_gpu(E, p, b.grains, b.view_off, find_ws_bytes=ws)
        assert_same_tracks(E, got, ref)


def test_out_of_box_grains_and_payload_ignored(E, oracle_mod):
    b = make_config(0)
    p = default_params(0)
    g = _mess_up(b.grains, p["view_size_q"])
    ref = oracle_mod.track_views(p, g, b.view_off, "cells", 1)
    assert_same_tracks(E, run_gpu(E, p, g, b.view_off), ref)


def test_e1_and_ties(E, oracle_mod):
    """The constructed example and noiseless equally spaced tracks: every candidate ties on (n_tube, D2)
    with others, so the (kmin, kmax) tie path decides."""
    with open(os.path.join(HERE, "golden", "e1_constructed_example.json")) as f:
        e1 = json.load(f)
    g = np.zeros((len(e1["grains"]), 4), np.int32); g[:, :3] = e1["grains"]
    off = np.asarray([0, len(g)], np.int32)
    got = run_gpu(E, e1["params"], g, off)
    ref = oracle_mod.track_views(e1["params"], g, off, "brute", 1)
    assert_same_tracks(E, got, ref)
    t = got["tracks"][0]
    assert (int(t["seed_a"]), int(t["seed_b"]), int(t["n_tube"])) == (0, 3, 10)

    lines = []
    for d, s in (((300, 0, 0), (500, 4000, 1600)), ((0, 280, 40), (4000, 600, 300)), ((170, 170, 170), (900, 900, 200)),
                 ((300, 0, 0), (500, 4000, 1650))):          # the last one runs 50 q beside the first: shared grains
        lines.append([(s[0] + i * d[0], s[1] + i * d[1], s[2] + i * d[2]) for i in range(14)])
    b = noiseless_track_view((8000, 8000, 3200), lines, n_fog=300)
    p = dict(e1["params"], view_size_q=(8000, 8000, 3200))
    ref = oracle_mod.track_views(p, b.grains, b.view_off, "brute", 1)
    assert len(ref.tracks) >= 3
    assert_same_tracks(E, run_gpu(E, p, b.grains, b.view_off), ref)


def test_degenerate_inputs(E, oracle_mod):
    p = default_params(0)
    # no grains at all, one view / three views with an empty one in the middle / a single grain
    for grains, off in ((np.zeros((0, 4), np.int32), [0, 0]),
                        (make_config(0).grains, None),
                        (np.asarray([[5, 5, 5, 0]], np.int32), [0, 1])):
        if off is None:
            n = len(grains)
            off = [0, n // 2, n // 2, n]
        off = np.asarray(off, np.int32)
        ref = oracle_mod.track_views(p, grains, off, "cells", 1)
        got = run_gpu(E, p, grains, off)
        assert_same_tracks(E, got, ref)
    # all grains coincide (D2 = 0 is never a seed, reading Q12) / all in one cell
    g = np.zeros((50, 4), np.int32); g[:, :3] = (777, 888, 999)
    off = np.asarray([0, 50], np.int32)
    assert_same_tracks(E, run_gpu(E, p, g, off), oracle_mod.track_views(p, g, off, "brute", 1))
    b = make_config(0)
    p1 = default_params(0, cell_um=(200.0, 200.0, 100.0))
    assert_same_tracks(E, run_gpu(E, p1, b.grains, b.view_off), oracle_mod.track_views(p1, b.grains, b.view_off, "cells", 1))


def test_capacity_and_range_errors_are_reported(E):
    import torch
    b = make_config(0)
    p = default_params(0, max_tracks_per_view=3)
    got = run_gpu(E, p, b.grains, b.view_off)
    assert int(got["counts"][E.EMU_CNT["status"]]) & E.EMU_ST["track_overflow"]
    g = b.grains.copy(); g[5, 0] = 1 << 17
    got = run_gpu(E, default_params(0), g, b.view_off)
    assert int(got["counts"][E.EMU_CNT["status"]]) & E.EMU_ST["coord"]
    prm = E.make_params((6400, 6400, 3200), (512, 512, 512), 256, 1280, 2621, 8, tube_ext_q=-2)
    with pytest.raises(E.EmuError):
        E.emu_workspace_bytes(prm, 10, 1)


def test_bench_workload_sampled_views(E, oracle_mod):
    """BASELINE.json configs[4] as bench.py runs it (same generator, parameters, 3x4x4 um cells, recommended workspace,
    hence the same kernels, frames, three bricks per frame and several internal chunks): 20 views through the CUDA
    path; views 0, 9 and 19 are compared with the oracle element by element, and the properties that hold at any
    size are checked on all of them."""
    import bench
    V = 20
    grains, off = bench.make_workload(0, V)
    p = bench.params_dict()
    got = run_gpu(E, p, grains, off)
    counts = got["counts"]
    assert int(counts[E.EMU_CNT["status"]]) == 0
    toff, tr, mem = got["track_off"], got["tracks"], got["members"]
    assert toff[0] == 0 and np.all(np.diff(toff) >= 0) and toff[-1] == len(tr) == int(counts[E.EMU_CNT["tracks"]])
    assert np.all(np.repeat(np.arange(V), np.diff(toff)) == tr["view"])
    assert np.all(tr["n_members"] >= p["min_grains"]) and np.all(tr["n_tube"] >= tr["n_members"])
    assert np.array_equal(tr["member_off"], np.concatenate(([0], np.cumsum(tr["n_members"])[:-1])))
    assert len(mem) == int(tr["n_members"].sum()) and len(np.unique(mem)) == len(mem)        # exclusive association
    mview = np.searchsorted(off, mem, side="right") - 1
    assert np.array_equal(mview, np.repeat(tr["view"], tr["n_members"]))                     # members stay in their view
    sample = [0, 9, 19]
    sub = np.concatenate([grains[off[v]:off[v + 1]] for v in sample])
    soff = np.zeros(len(sample) + 1, np.int32)
    soff[1:] = np.cumsum([off[v + 1] - off[v] for v in sample])
    ref = oracle_mod.track_views(p, sub, soff, "cells", len(sample))
    for k, v in enumerate(sample):
        shift = int(off[v]) - int(soff[k])
        g = tr[toff[v]:toff[v + 1]]
        r = ref.tracks[ref.track_off[k]:ref.track_off[k + 1]]
        assert len(g) == len(r) and len(g) > 500
        for f in ("n_tube", "n_members", "seed_d2"):
            assert np.array_equal(g[f], r[f]), (v, f)
        assert np.array_equal(g["seed_a"] - shift, r["seed_a"]) and np.array_equal(g["seed_b"] - shift, r["seed_b"])
        gm = mem[g["member_off"][0]:g["member_off"][-1] + g["n_members"][-1]] - shift
        rm = ref.members[r["member_off"][0]:r["member_off"][-1] + r["n_members"][-1]]
        assert np.array_equal(gm, rm)
        gf, rf = got["fits"][toff[v]:toff[v + 1]], ref.fits[ref.track_off[k]:ref.track_off[k + 1]]
        for f in ("axis", "n", "u_min", "u_max"):
            assert np.array_equal(gf[f], rf[f])
        assert np.all(np.abs(gf["slope"] - rf["slope"]) <= 1e-5 * np.maximum(np.abs(gf["slope"]), np.abs(rf["slope"])) + 1e-12)
        assert np.all(np.abs(gf["icpt"] - rf["icpt"]) <= 1e-5 * np.maximum(np.abs(gf["icpt"]), np.abs(rf["icpt"])) + 1e-6)


@pytest.mark.parametrize("cell_um", [(8.0, 8.0, 8.0), (4.0, 4.0, 4.0), (3.0, 4.0, 2.5)])
@pytest.mark.parametrize("cfg,ext_q", [(0, 0), (0, 640), (2, 320), (3, 1280)])
def test_bounded_tube_bit_exact(E, oracle_mod, cfg, ext_q, cell_um):
    """tube_ext_q >= 0 (a grain counts only if its foot lies between the seed grains or at most
    tube_ext_q beyond either).  Per-seed counts and the track list against the oracle; 8 um cells take the generic
    global-memory kernels, the finer ones the shared-memory brick kernels (clipped walk, float axial test with the
    exact fallback)."""
    b = make_config(cfg)
    p = dict(default_params(cfg, cell_um=cell_um), tube_ext_q=ext_q)
    ref = oracle_mod.track_views(p, b.grains, b.view_off, "cells", 1, seed_dump=True)
    dump, counts = seed_dump_gpu(E, p, b.grains, b.view_off, ref.counters["seeds"] + 16)
    assert int(counts[E.EMU_CNT["seeds"]]) == ref.counters["seeds"]
    a = dump[np.lexsort((dump[:, 2], dump[:, 1], dump[:, 0]))]
    r = ref.seed_dump[np.lexsort((ref.seed_dump[:, 2], ref.seed_dump[:, 1], ref.seed_dump[:, 0]))]
    assert np.array_equal(a, r)
    got = run_gpu(E, p, b.grains, b.view_off, tube_ext_q=ext_q)
    assert_same_tracks(E, got, ref)
    whole = oracle_mod.track_views(default_params(cfg), b.grains, b.view_off, "cells", 1)
    assert ref.counters["candidates"] < whole.counters["candidates"]
