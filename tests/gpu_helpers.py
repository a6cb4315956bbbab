"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI binding."""
import numpy as np


def gpu_params(E, p: dict, **kw):
    d = dict(view_size_q=p["view_size_q"], cell_size_q=p["cell_size_q"], sep_min_q=p["sep_min_q"],
             sep_max_q=p["sep_max_q"], tube_r2_q=p["tube_r2_q"], min_grains=p["min_grains"],
             max_tracks_per_view=p.get("max_tracks_per_view", 4096), tube_ext_q=p.get("tube_ext_q", -1),
             angle_min_grains=p.get("angle_min_grains"))
    d.update(kw)
    return E.make_params(**d)


def run_gpu(E, p: dict, grains: np.ndarray, view_off: np.ndarray, find_ws_bytes=None, **kw):
    import torch
    prm = gpu_params(E, p, **kw)
    n_views = len(view_off) - 1
    g = np.ascontiguousarray(grains, np.int32).reshape(-1, 4)
    d_grains = torch.from_numpy(g).cuda() if len(g) else torch.empty((0, 4), dtype=torch.int32, device="cuda")
    d_off = torch.from_numpy(np.ascontiguousarray(view_off, np.int32)).cuda()
    B = E.PathBuffers(prm, len(g), n_views, find_ws_bytes=find_ws_bytes)
    res = E.run_path(prm, d_grains, d_off, n_views, B)
    torch.cuda.synchronize()
    out = res.host()
    out["sorted"] = B.sorted[:len(g)].cpu().numpy()
    out["cell_start"] = B.cell_start.cpu().numpy()
    return out


def seed_dump_gpu(E, p: dict, grains: np.ndarray, view_off: np.ndarray, capacity: int):
    import torch
    prm = gpu_params(E, p)
    n_views = len(view_off) - 1
    g = np.ascontiguousarray(grains, np.int32).reshape(-1, 4)
    d_grains = torch.from_numpy(g).cuda()
    d_off = torch.from_numpy(np.ascontiguousarray(view_off, np.int32)).cuda()
    B = E.PathBuffers(prm, len(g), n_views)
    E.emu_bin_grains(prm, d_grains, d_off, len(g), n_views, B.sorted, B.cell_start, B.status, B.ws)
    dump = torch.zeros((capacity, 4), dtype=torch.int32, device="cuda")
    E.emu_count_seeds(prm, B.sorted, B.cell_start, d_off, len(g), n_views, dump, B.counts, B.ws)
    torch.cuda.synchronize()
    counts = B.counts.cpu().numpy()
    n = int(counts[E.EMU_CNT["seeds"]])
    return dump[:min(n, capacity)].cpu().numpy(), counts


def assert_same_tracks(E, got: dict, ref, fit_rtol=1e-5):
    """GPU result vs OracleResult: track list, offsets, members memcmp-equal; fits within north_star's 1e-5."""
    counts = got["counts"]
    assert int(counts[E.EMU_CNT["status"]]) == 0, f"status {int(counts[E.EMU_CNT['status']])}"
    assert np.array_equal(got["track_off"], ref.track_off)
    assert got["tracks"].tobytes() == ref.tracks.tobytes()
    assert got["members"].tobytes() == ref.members.tobytes()
    assert int(counts[E.EMU_CNT["seeds"]]) == ref.counters["seeds"]
    assert int(counts[E.EMU_CNT["candidates"]]) == ref.counters["candidates"]
    f, r = got["fits"], ref.fits
    assert len(f) == len(r)
    for k in ("axis", "n", "u_min", "u_max"):
        assert np.array_equal(f[k], r[k]), k
    ds = np.abs(f["slope"] - r["slope"]); di = np.abs(f["icpt"] - r["icpt"])
    assert np.all(ds <= fit_rtol * np.maximum(np.abs(f["slope"]), np.abs(r["slope"])) + 1e-12)
    assert np.all(di <= fit_rtol * np.maximum(np.abs(f["icpt"]), np.abs(r["icpt"])) + 1e-6)
