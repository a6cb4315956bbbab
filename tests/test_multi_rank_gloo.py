"""The N > 1 path on CPU: two gloo ranks shard the views as bench.py does, each runs its shard (the oracle stands in
for the kernels here - the plumbing is what is tested), and the reductions / gather reproduce the one-rank result."""
import os
import socket

import numpy as np
import pytest


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, views_per_rank, out_dir):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from emu_synth import CONFIGS, default_params, make_batch
        from paper_1311_5334_b200 import shard
        first, n = shard.view_range(rank, world, views_per_rank)
        b = make_batch(CONFIGS[0], 0, n_views=n, first_view=first)
        r = oracle.track_views(default_params(0), b.grains, b.view_off, "cells", 1)
        ms, (n_grains, n_tracks) = shard.reduce_step(10.0 + rank, [b.n_grains, len(r.tracks)])
        off = shard.gather_track_off(r.track_off)
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), ms=ms, n_grains=n_grains, n_tracks=n_tracks, off=off,
                 local_tracks=len(r.tracks))
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_reduce_gather(tmp_path, oracle_mod):
    import torch.multiprocessing as mp
    from emu_synth import CONFIGS, default_params, make_batch
    world, vpr = 2, 2
    mp.spawn(_worker, args=(world, _free_port(), vpr, str(tmp_path)), nprocs=world, join=True)
    whole = make_batch(CONFIGS[0], 0, n_views=world * vpr)
    ref = oracle_mod.track_views(default_params(0), whole.grains, whole.view_off, "cells", 1)
    got = [np.load(os.path.join(tmp_path, f"rank{r}.npz")) for r in range(world)]
    for g in got:
        assert float(g["ms"]) == 11.0                               # max over ranks
        assert int(g["n_grains"]) == whole.n_grains                 # sum over ranks
        assert int(g["n_tracks"]) == len(ref.tracks)
        assert np.array_equal(g["off"], ref.track_off.astype(np.int64))   # the gathered global track_off
    assert sum(int(g["local_tracks"]) for g in got) == len(ref.tracks)


def test_split_views_covers_everything():
    from paper_1311_5334_b200 import shard
    for n, w in ((1024, 8), (10, 3), (2, 4), (0, 2)):
        parts = shard.split_views(n, w)
        assert len(parts) == w and parts[0][0] == 0
        assert sum(k for _, k in parts) == n
        assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(w - 1))
        assert max(k for _, k in parts) - min(k for _, k in parts) <= 1
    # balanced by sum N^2: one dense view weighs as much as four views of half its grains
    n = [100] * 8 + [200] * 2
    parts = shard.split_views(10, 2, n)
    assert parts == [(0, 8), (8, 2)]
    assert sum(k for _, k in parts) == 10
    for nv, w in ((7, 3), (3, 5), (64, 8)):
        rng = np.random.default_rng(nv)
        g = rng.integers(1000, 70000, nv)
        parts = shard.split_views(nv, w, g)
        assert len(parts) == w and parts[0][0] == 0 and sum(k for _, k in parts) == nv
        assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(w - 1))
        if nv >= w:
            assert all(k >= 1 for _, k in parts)
            loads = [float((g[a:a + k].astype(float) ** 2).sum()) for a, k in parts]
            assert max(loads) <= sum(loads) / w + float(g.max()) ** 2          # within one view of the ideal share
    assert shard.view_range(3, 8, 128) == (384, 128)
    with pytest.raises(ValueError):
        shard.view_range(8, 8, 1)
