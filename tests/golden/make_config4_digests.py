"""Writes tests/golden/config4_view_digests.json: the ORACLE's track list for every one of the 1 024 views of
BASELINE.json configs[4] (the batch bench.py times), as one SHA-256 per view.

Why: north_star asks for track lists bit-identical to the oracle on all five configs, and the oracle needs about 36 s
of one core per config-4 view - some 40 minutes on 16 cores for the whole batch - so the GPU tests cannot run it on
every view each time.  This script runs it once, on the CPU box, in slices that can be resumed
(`python tests/golden/make_config4_digests.py [first_view [n_views]]`, progress in config4_view_digests.partial.jsonl;
slices may run on several machines with EMU_DIGEST_PARTIAL=<file> and be concatenated into that file afterwards),
and tests/test_gpu_config4_all_views.py compares the CUDA path's output for all 1 024 views with the stored digests.

It imports `oracle` and `emu_synth` only - nothing of the CUDA path, no bench.py.  The workload is restated here:
views (4, v) of emu_synth.make_view, default_params(4) with the contract's whole-line tube.  (The cell size has no
effect on the track list - reading Q10 - so the oracle's default cells serve.)

Digest of a view = SHA-256 over, in this order, with everything made relative to the view (view := 0, rows minus the
view's first row, member_off minus the view's first member offset):
  tracks.tobytes() (emu_track records, best first) + members.tobytes() (int32 rows) + the integer fields of the fits
  (axis, n, u_min, u_max as int32[T][4]).tobytes()
The floating-point fit fields are not part of it (they are compared at 1e-5 on sampled views elsewhere).
"""
from __future__ import annotations

import hashlib
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

CFG = 4
N_VIEWS = 1024
OUT = os.path.join(HERE, "config4_view_digests.json")
PARTIAL = os.path.join(HERE, "config4_view_digests.partial.jsonl")


def workload_params() -> dict:
    from emu_synth import default_params
    p = default_params(CFG, max_tracks_per_view=4096)
    p["tube_ext_q"] = -1
    return p


def view_digests(tracks: np.ndarray, track_off: np.ndarray, members: np.ndarray, fits: np.ndarray, view_off: np.ndarray) -> list:
    """one dict per view of a batch result (oracle's or the CUDA path's: same record layouts)"""
    out = []
    for v in range(len(view_off) - 1):
        t0, t1 = int(track_off[v]), int(track_off[v + 1])
        t = tracks[t0:t1].copy()
        f = fits[t0:t1]
        m0 = int(t["member_off"][0]) if t1 > t0 else 0
        nm = int(t["n_members"].sum())
        m = members[m0:m0 + nm].astype(np.int32) - np.int32(view_off[v])
        t["view"] -= v
        t["seed_a"] -= view_off[v]; t["seed_b"] -= view_off[v]
        t["member_off"] -= m0
        fi = np.stack([f["axis"], f["n"], f["u_min"], f["u_max"]], axis=1).astype(np.int32) if t1 > t0 else np.zeros((0, 4), np.int32)
        h = hashlib.sha256()
        h.update(np.ascontiguousarray(t).tobytes()); h.update(np.ascontiguousarray(m).tobytes()); h.update(np.ascontiguousarray(fi).tobytes())
        out.append(dict(n_grains=int(view_off[v + 1] - view_off[v]), n_tracks=t1 - t0, n_members=nm, sha256=h.hexdigest()))
    return out


def main(first: int = 0, count: int = N_VIEWS, slice_views: int = 16):
    global PARTIAL
    PARTIAL = os.environ.get("EMU_DIGEST_PARTIAL", PARTIAL)      # (slices run on another machine write elsewhere; concatenate them)
    import oracle
    from emu_synth import CONFIGS, make_view
    oracle.build()
    p = workload_params()
    done = {}
    if os.path.exists(PARTIAL):
        for line in open(PARTIAL):
            r = json.loads(line)
            done[r["view"]] = r
    t_start = time.time()
    for v0 in range(first, min(N_VIEWS, first + count), slice_views):
        vs = [v for v in range(v0, min(N_VIEWS, first + count, v0 + slice_views)) if v not in done]
        if not vs:
            continue
        gs = [make_view(CONFIGS[CFG], CFG, v)[0] for v in vs]
        off = np.zeros(len(vs) + 1, np.int32)
        off[1:] = np.cumsum([len(g) for g in gs])
        r = oracle.track_views(p, np.concatenate(gs), off, "cells", 0)
        with open(PARTIAL, "a") as fh:
            for v, d in zip(vs, view_digests(r.tracks, r.track_off, r.members, r.fits, off)):
                d["view"] = v
                done[v] = d
                fh.write(json.dumps(d) + "\n")
        print(f"views {vs[0]}..{vs[-1]} done, {len(done)} of {N_VIEWS}, {time.time() - t_start:.0f} s", flush=True)
    if len(done) == N_VIEWS:
        p_out = {k: (list(v) if isinstance(v, (list, tuple)) else v) for k, v in p.items() if k != "cell_size_q" and v is not None}
        views = [{k: done[v][k] for k in ("n_grains", "n_tracks", "n_members", "sha256")} for v in range(N_VIEWS)]
        doc = dict(source="oracle.track_views (mode cells) on emu_synth views (4, v), v = 0..1023; written by "
                          "tests/golden/make_config4_digests.py, which imports only oracle/ and emu_synth/",
                   config=CFG, params=p_out, n_views=N_VIEWS, total_tracks=sum(x["n_tracks"] for x in views),
                   total_members=sum(x["n_members"] for x in views), views=views)
        with open(OUT, "w") as fh:
            json.dump(doc, fh, indent=0)
        print("wrote", OUT)


if __name__ == "__main__":
    a = [int(x) for x in sys.argv[1:]]
    main(*a)
