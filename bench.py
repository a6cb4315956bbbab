#!/usr/bin/env python
"""bench.py - one "step" = one pass of the whole hot path (A1 bin -> A2..A5,A7 find -> A6 fit) over the
throughput batch of BASELINE.json configs[4]: 1,024 independent views of 350x300x50 um, fog 10 per 1000 um^3,
300 isotropic through-going tracks per view (about 64 k grains per view, 66 M grains per GPU), seeded synthetic.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--views V] [--impl reference]

N > 1 is launched by torchrun, one rank per GPU; every rank processes its own V views (weak scaling, no
data-path collective - the views are independent).  Rank 0 prints ONE JSON line.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload instead.
Extras measured after the timed step (none changes it; 0 switches one off): --latency-views (single views through
the host call, default 8), --recognize-views (emu_recognize_grains on rendered voxel stacks, default 4);
--tube-ext-um runs the bounded tube of SURVEY 8(f) NEXT-1 instead of the contract's whole line.  DESIGN.md section 8 states every formula used here.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

CFG = 4                          # BASELINE.json configs[4] "throughput batch"
CELL_UM = (3.0, 4.0, 4.0)        # cell size of the 3D hash (a pure speed knob: no effect on the track list)
VIEW_AREA_CM2 = 350e-4 * 300e-4  # 350 x 300 um = 1.05e-3 cm^2 per view
# Algorithmic work of the voting kernel: lane-instructions per seed
#   = tests/seed * 18 + pair-tests/seed * 10, with tests/seed and pair-tests/seed the ORACLE's own counters
# (oracle mode "cells", same cell size) on views 0..7 of this workload.  The cpu_baseline leg re-measures
# them live; the constants serve the runs that have no such leg (N > 1).
ALG_PER_SEED = {(8.0, 8.0, 8.0): (317.7, 2.88), (3.0, 4.0, 4.0): (102.1, 2.26)}
INSTR_PER_TEST, INSTR_PER_PAIR = 18, 10    # read off the SASS: profiles/r2_sass_counts.md
MIX_PEAK_SHARE = 99.3 / 128.0    # measured issue rate of the tube-test instruction mix / nominal issue rate: the committed
                                 # round-2 run (profiles/r2_mb_pipes.md).  Used only when the live leg below is off or fails.
MIX_SASS_PER_PAIR = 52           # SASS instructions of one pair-iteration of k_mix (profiles/r2_mb_pipes.md: 104 per two)
BIN_BYTES_PER_GRAIN = 32.0       # 16 B read + 16 B written per grain; + 4 B per cell of the grid
# DRAM bytes (read + write) of one k_brick<kVote> launch per view of the launch, from the committed ncu --set full
# capture profiles/r2_k_brick_full.txt (33 views: 50.48 GB read + 28.86 GB written)
VOTE_DRAM_BYTES_PER_VIEW = (50.478269e9 + 28.861403e9) / 33
# DRAM bytes of the two binning kernels per grain, from profiles/r2_k_bin_full.txt (65 792 077 grains:
# k_bin_split 1.055 + 1.004 GB, k_bin_chunk 1.061 + 1.467 GB)
BIN_DRAM_BYTES_PER_GRAIN = (1.054695e9 + 1.003755e9 + 1.060990e9 + 1.466883e9) / 65792077


def _gen_view(v):
    from emu_synth import CONFIGS, make_view
    g, _, _ = make_view(CONFIGS[CFG], CFG, v)
    return g


def make_workload(first_view: int, n_views: int):
    """grains int32 [N,4], view_off int32 [n_views+1] for views first_view.. of config 4 (key (4, v))."""
    import multiprocessing as mp
    nproc = max(1, min(len(os.sched_getaffinity(0)), 32, n_views))
    if nproc > 1:
        with mp.get_context("fork").Pool(nproc) as pool:
            gs = pool.map(_gen_view, range(first_view, first_view + n_views), chunksize=max(1, n_views // (4 * nproc)))
    else:
        gs = [_gen_view(v) for v in range(first_view, first_view + n_views)]
    off = np.zeros(n_views + 1, np.int32)
    off[1:] = np.cumsum([len(g) for g in gs])
    return np.concatenate(gs), off


TUBE_EXT_Q = -1                  # -1 = the contract (whole line); >= 0: the bounded tube of SURVEY 8(f) NEXT-1 (--tube-ext-um)


def params_dict():
    from emu_synth import default_params
    p = default_params(CFG, cell_um=CELL_UM, max_tracks_per_view=4096)
    p["tube_ext_q"] = TUBE_EXT_Q
    return p


def measure_mix_peak():
    """The measured issue peak of the voting kernel's own instruction mix, from THIS run: compile
    microbench/mb_pipes.cu to a temporary directory, run it on the current GPU and read its k_mix line."""
    import re
    import tempfile
    from paper_1311_5334_b200 import build as lib_build
    with tempfile.TemporaryDirectory() as tmp:
        exe = lib_build.build_microbench(tmp)
        out = subprocess.run([exe], check=True, capture_output=True, text=True, timeout=120).stdout      # device 0, as the N = 1 run
    pairs = float(re.search(r"=\s*([0-9.]+) lane-pairs / clk / SM", out).group(1))
    ffma = re.search(r"^FFMA\s+[0-9.]+\s+([0-9.]+)", out, flags=re.M)
    per_clk = pairs * MIX_SASS_PER_PAIR
    return {"lane_instr_per_clk_sm": per_clk, "share_of_nominal": per_clk / 128.0, "lane_pairs_per_clk_sm": pairs,
            "sass_instr_per_pair": MIX_SASS_PER_PAIR, "ffma_lane_ops_per_clk_sm": float(ffma.group(1)) if ffma else None,
            "source": "microbench/mb_pipes.cu (k_mix) compiled and run inside this bench run"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "_source": "fallback"}


def oracle_sample(n_sample_views: int, threads: int):
    """The oracle as it stands (mode 'cells', g++ -O2, one OpenMP thread per view) on the first views of the
    workload.  Returns (seconds, grains, counters)."""
    import oracle
    oracle.build()
    grains, off = make_workload(0, n_sample_views)
    # untimed warm-up: library load, OpenMP team, page faults (one tiny config-0 view per thread)
    from emu_synth import CONFIGS, default_params, make_batch
    wb = make_batch(CONFIGS[0], 0, n_views=max(1, min(threads, n_sample_views)))
    oracle.track_views(default_params(0), wb.grains, wb.view_off, "cells", threads)
    t0 = time.perf_counter()
    r = oracle.track_views(params_dict(), grains, off, "cells", threads)
    dt = time.perf_counter() - t0
    return dt, int(off[-1]), r.counters, r


def first_views(out: dict, nv: int) -> dict:
    """tracks / fits / members / track_off of views 0..nv-1 of a batch result (host arrays)."""
    toff = np.asarray(out["track_off"])[:nv + 1].copy()
    nt = int(toff[-1])
    tr = np.asarray(out["tracks"])[:nt].copy()
    nm = int(tr["member_off"][-1] + tr["n_members"][-1]) if nt else 0
    return dict(track_off=toff, tracks=tr, fits=np.asarray(out["fits"])[:nt].copy(), members=np.asarray(out["members"])[:nm].copy())


def same_as_oracle(got: dict, ref) -> bool:
    """SURVEY 8(c) comparison rule: offsets, every track field and every member index bit-equal; fits: integer fields
    equal, slopes / intercepts within 1e-5 relative (BASELINE.json north_star)."""
    if not (np.array_equal(got["track_off"], ref.track_off) and got["tracks"].tobytes() == ref.tracks.tobytes()
            and got["members"].tobytes() == ref.members.tobytes() and len(got["fits"]) == len(ref.fits)):
        return False
    f, r = got["fits"], ref.fits
    for k in ("axis", "n", "u_min", "u_max"):
        if not np.array_equal(f[k], r[k]):
            return False
    ok_s = np.abs(f["slope"] - r["slope"]) <= 1e-5 * np.maximum(np.abs(f["slope"]), np.abs(r["slope"])) + 1e-12
    ok_i = np.abs(f["icpt"] - r["icpt"]) <= 1e-5 * np.maximum(np.abs(f["icpt"]), np.abs(r["icpt"])) + 1e-6
    return bool(np.all(ok_s) and np.all(ok_i))


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, same metric / unit / config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = len(os.sched_getaffinity(0))
    nv = args.sample_views if args.sample_views else max(1, min(cores, 16))
    times = []
    cnt, ng = None, 0
    for _ in range(args.warmup if args.reference_warmup else 0):
        oracle_sample(nv, cores)
    for _ in range(max(1, min(args.steps, args.reference_steps))):
        dt, ng, cnt, _ = oracle_sample(nv, cores)
        times.append(dt)
    t = float(np.mean(times))
    val = ng / t
    line = {
        "impl": "reference", "metric": "grains_per_s", "value": val, "unit": "grains/s", "n_gpus": args.gpus,
        "steps": len(times), "warmup": 0, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": workload_config(nv, 1),
        "views_per_s": nv / t, "cm2_per_hour": nv / t * 3600 * VIEW_AREA_CM2,
        "cpu_baseline": {"value": val, "unit": "grains/s", "cores": min(cores, nv), "kind": "oracle",
                         "sample": f"views 0..{nv - 1} of the workload ({ng} grains), one OpenMP thread per view, "
                                   f"oracle mode 'cells' at cell {CELL_UM} um; each step = this sample"},
        "e2e": {"value": val, "unit": "grains/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "oracle_counters": cnt,
    }
    print(json.dumps(line))


def workload_config(views_per_gpu: int, n_gpus: int) -> dict:
    return {"workload": "BASELINE.json configs[4] throughput batch: independent 350x300x50 um views, fog 10/1000 um^3, "
                        "300 isotropic through tracks per view, int32 coords at 1/64 um, seeded synthetic (key (4, view))",
            "views_per_gpu": views_per_gpu, "views_total": views_per_gpu * n_gpus,
            "tracking": "tube r2 2621 q^2 (0.8 um), pair separation 256..1280 q (4..20 um), min 8 grains, " +
                        ("whole-line tube" if TUBE_EXT_Q < 0 else f"bounded tube, {TUBE_EXT_Q} q beyond the seed grains (NEXT-1, not the contract)"),
            "cell_um": list(CELL_UM), "parallelism": f"views sharded over {n_gpus} GPU(s), no collective",
            "l2": "inputs (about 1 GB of grains per step) exceed the 126 MB L2; no flush needed"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--views", type=int, default=1024, help="views per GPU (BASELINE.json configs[4]: 1024)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--sample-views", type=int, default=0, help="views in the oracle sample (default: one per core, <= 16)")
    ap.add_argument("--reference-steps", type=int, default=2)
    ap.add_argument("--reference-warmup", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cell-um", type=float, nargs=3, default=None, help="override the cell size of the 3D hash (um)")
    ap.add_argument("--mix-peak", type=int, default=1,
                    help="1: compile and run microbench/mb_pipes.cu and report the measured issue peak of the voting kernel's "
                         "instruction mix as roofline.mix_peak_measured (N = 1 only); 0: the committed round-2 figure")
    ap.add_argument("--latency-views", type=int, default=8,
                    help="also time single views one at a time through the host call (SURVEY 8(f) NEXT-3: the microscope "
                         "delivers one view every 0.2 s, P:102); adds the key single_view to the JSON line")
    ap.add_argument("--recognize-views", type=int, default=4,
                    help="also time emu_recognize_grains (SURVEY 8(f) NEXT-4) on this many synthetic 1280 x 1024 x 40 voxel "
                         "stacks rendered from config-1 views; adds the key recognize to the JSON line")
    ap.add_argument("--find-ws-gib", type=float, default=None,
                    help="workspace given to emu_find_tracks in GiB (default: what emu_workspace_bytes recommends, about "
                         "100 GiB for the full batch); the views are then processed in smaller internal chunks")
    ap.add_argument("--stream-views", type=int, default=1024,
                    help="also run this many views of the workload in batches through emu_stream_* (copies overlapped with "
                         "the kernels, SURVEY 8(f) NEXT-3) and 32 config-1 views one per batch; adds the key stream; 0 = off")
    ap.add_argument("--stream-batch", type=int, default=48, help="views per streamed batch")
    ap.add_argument("--tube-ext-um", type=float, default=None,
                    help="bounded tube (SURVEY 8(f) NEXT-1): axial extent beyond the seed grains in um; default: whole line")
    args = ap.parse_args()
    if args.cell_um is not None:
        global CELL_UM
        CELL_UM = tuple(float(x) for x in args.cell_um)
    if args.tube_ext_um is not None:
        global TUBE_EXT_Q
        TUBE_EXT_Q = int(round(args.tube_ext_um * 64))
    if args.impl == "reference":
        run_reference(args)
        return

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU, rendezvous on 127.0.0.1)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--standalone", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--local-addr", "127.0.0.1", os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))

    import torch
    import torch.distributed as dist
    import paper_1311_5334_b200 as E   # raises if libemu4pi.so is missing: there is no fallback
    E.exported_symbols()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    assert world == args.gpus, f"--gpus {args.gpus} but WORLD_SIZE={world}: launch with torchrun"

    from paper_1311_5334_b200 import shard
    p = params_dict()
    V = args.views
    first_view, _ = shard.view_range(rank, world, V)          # weak scaling: every rank owns V views of its own
    grains, off = make_workload(first_view, V)
    n = int(off[-1])
    prm = E.make_params(**{k: p[k] for k in ("view_size_q", "cell_size_q", "sep_min_q", "sep_max_q", "tube_r2_q",
                                             "min_grains", "max_tracks_per_view", "tube_ext_q")})
    d_grains = torch.from_numpy(grains).cuda()
    d_off = torch.from_numpy(off).cuda()
    find_ws = int(args.find_ws_gib * (1 << 30)) if args.find_ws_gib else None
    B = E.PathBuffers(prm, n, V, find_ws_bytes=find_ws)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    B_ws_bytes = B.ws.numel()
    for _ in range(args.warmup):
        E.run_path(prm, d_grains, d_off, V, B)
    barrier()
    counts = B.counts.cpu().numpy().copy()
    status = int(counts[E.EMU_CNT["status"]]) | int(B.status.cpu()[0])
    assert status == 0, f"device status {status} (capacity / range): the step is not valid"

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    prof = E.Profile()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    with prof:
        for _ in range(args.steps):
            E.run_path(prm, d_grains, d_off, V, B)
    ev1.record()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if rank == 0 else None
    stage_ms, stage_launches = prof.read()
    ms_total, (n_total,) = shard.reduce_step(ms_total, [n], device="cuda")    # max over ranks / sum over ranks
    ms_step = ms_total / args.steps
    counts = B.counts.cpu().numpy().copy()
    cores = len(os.sched_getaffinity(0))
    nv_s = args.sample_views if args.sample_views else max(1, min(cores, 16, V))      # views the oracle leg will check
    dev_first = first_views(E.PathResult(B).host(), nv_s) if rank == 0 else None      # of the LAST timed step

    # end to end: ONE C-ABI call on pinned host buffers per step (H2D + path + D2H inside the call)
    e2e, e2e_first = None, None
    if not args.no_e2e:
        del B                                               # one workspace at a time (each is sized for 180 GB of HBM)
        torch.cuda.empty_cache()
        H = E.HostPath(prm, n, V)
        H.h_grains[:n].copy_(torch.from_numpy(grains))
        H.h_view_off.copy_(torch.from_numpy(off))
        nt, nm = H.call()                                   # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            nt, nm = H.call()                               # synchronous: returns with the outputs on the host
        barrier()
        dt = time.perf_counter() - t0
        dt_max, _ = shard.reduce_step(dt, [0], device="cuda")
        e2e = {"value": n_total * args.steps / dt_max, "unit": "grains/s",
               "h2d_bytes_per_step": H.h2d_bytes(), "d2h_bytes_per_step": H.d2h_bytes(nt, nm),
               "ms_per_step": dt_max / args.steps * 1e3,
               "call": "emu_track_views_host (pinned host buffers; copies inside the timed call)"}
        assert int(H.h_counts[E.EMU_CNT["status"]]) == 0
        assert nt == int(counts[E.EMU_CNT["tracks"]]), "host path and device path disagree"
        e2e_first = first_views(H.result(nt, nm), nv_s) if rank == 0 else None           # of the LAST timed call
        del H

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = measured_peaks()
    seeds = int(counts[E.EMU_CNT["seeds"]])
    cpu = None
    alg = ALG_PER_SEED.get(tuple(CELL_UM))
    parity = None
    ref_tracks = None                                         # the oracle's result for views 0..nv_s-1 (kept for the streamed leg)
    if world == 1 and not args.no_cpu_baseline:
        dt, ng, cnt, ref = oracle_sample(nv_s, cores)
        ref_tracks = ref
        # parity of what was TIMED: views 0..nv_s-1 of the last timed device step and of the last timed host call
        # against the oracle, element by element (SURVEY 8(c) comparison rule)
        parity = {"views_checked": nv_s, "tracks_checked": int(len(ref.tracks)), "members_checked": int(len(ref.members)),
                  "device_path": same_as_oracle(dev_first, ref),
                  "e2e_host_call": same_as_oracle(e2e_first, ref) if e2e_first is not None else None,
                  "rule": "track_off, tracks, members bit-equal; fits: integer fields equal, slope / icpt within 1e-5 relative"}
        parity["identical"] = bool(parity["device_path"] and parity["e2e_host_call"] is not False)
        cpu = {"value": ng / dt, "unit": "grains/s", "cores": min(cores, nv_s), "kind": "oracle",
               "sample": f"views 0..{nv_s - 1} of the workload ({ng} grains), one OpenMP thread per view, oracle mode "
                         f"'cells' at cell {CELL_UM} um, {dt:.1f} s after an untimed warm-up on config-0 views",
               "views_per_s": nv_s / dt}
        alg = (cnt["tube_tests"] / cnt["seeds"], cnt["pair_tests"] / cnt["seeds"])

    sm_max = float(peaks.get("sm_max_mhz") or 1965.0)
    alu_peak = 148 * 4 * 32 * sm_max * 1e6 / 1e12            # Tlane-instr/s
    mix_peak = None
    if args.mix_peak and world == 1:
        try:
            mix_peak = measure_mix_peak()
        except Exception as exc:                              # an extra leg may not take the headline down with it
            mix_peak = {"error": f"{type(exc).__name__}: {exc}"}
    mix_share = mix_peak["share_of_nominal"] if mix_peak and "share_of_nominal" in mix_peak else MIX_PEAK_SHARE
    vote_ms = stage_ms["vote"] / max(1, stage_launches["vote"])
    roofline = None
    if alg is not None and stage_launches["vote"]:
        alg_instr = seeds * (alg[0] * INSTR_PER_TEST + alg[1] * INSTR_PER_PAIR)   # per step, all vote launches
        achieved = alg_instr / (stage_ms["vote"] / args.steps * 1e-3) / 1e12
        views_per_launch = V * args.steps / stage_launches["vote"]
        captured = tuple(CELL_UM) == (3.0, 4.0, 4.0) and TUBE_EXT_Q < 0     # the configuration of the committed ncu capture
        gpu_tests = float(counts[E.EMU_CNT["tests"]]) / max(1, seeds)
        roofline = {"kernel": "k_brick<kVote> (A3 tube count + hit records on shared-memory bricks, three frames; the seeds of "
                              "A2 arrive as per-brick lists of prepared records)", "bound": "alu", "achieved": achieved, "peak": alu_peak,
                    "unit": "Tlane-instr/s", "frac": achieved / alu_peak,
                    "frac_of_mix_peak": achieved / (alu_peak * mix_share),
                    "mix_peak_measured": mix_peak,
                    "mix_peak_source": ("measured in this run (mix_peak_measured)" if mix_share is not MIX_PEAK_SHARE else
                                        "profiles/r2_mb_pipes.md (round-2 capture): the tube-test instruction mix sustains 99.3 of "
                                        "128 lane-instr per clock and SM"),
                    "frac_on_kernel_tests": achieved / alu_peak * (gpu_tests * INSTR_PER_TEST + alg[1] * INSTR_PER_PAIR)
                                            / (alg[0] * INSTR_PER_TEST + alg[1] * INSTR_PER_PAIR),
                    "traffic": VOTE_DRAM_BYTES_PER_VIEW * views_per_launch if captured else None,
                    "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of profiles/r2_k_brick_full.txt per view "
                                      "x views per launch",
                    "peak_source": f"148 SM x 4 schedulers x 32 lanes x {sm_max:.0f} MHz ({peaks['_source']} max SM clock)",
                    "algorithmic": f"{seeds} seeds x ({alg[0]:.1f} tests x {INSTR_PER_TEST} + {alg[1]:.2f} pair tests x "
                                   f"{INSTR_PER_PAIR}) lane-instr, oracle counters at the same cell size",
                    "launches_per_step": stage_launches["vote"] / args.steps, "avg_launch_ms": vote_ms,
                    "share_of_step": stage_ms["vote"] / args.steps / ms_step}
    bin_ms = sum(stage_ms[k] for k in ("bin_count", "bin_scan", "bin_scatter", "bin_place")) / args.steps
    hbm = float(peaks["hbm_gbs"])
    ncell = int(E.emu_grid_cells(prm)[0])
    bin_bytes = BIN_BYTES_PER_GRAIN * n + 4.0 * ncell * V
    bin_gbs = bin_bytes / (bin_ms * 1e-3) / 1e9 if bin_ms > 0 else 0.0
    roofline_bin = {"kernel": "emu_bin_grains: k_bin_split + k_bin_chunk (two passes: chunks of cells through a scratch array, then one chunk per block in shared memory)", "bound": "hbm",
                    "achieved": bin_gbs, "peak": hbm, "unit": "GB/s", "frac": bin_gbs / hbm,
                    "traffic": BIN_DRAM_BYTES_PER_GRAIN * n if tuple(CELL_UM) == (3.0, 4.0, 4.0) else None, "traffic_source": "profiles/r2_k_bin_full.txt, both passes, per grain x grains",
                    "algorithmic_bytes": bin_bytes, "ms": bin_ms,
                    "algorithmic_bytes_per_grain": bin_bytes / max(1, n),
                    "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peaks['_source']})"}

    single = None
    if args.latency_views > 0:
        try:
            # one view per host call (H2D + path + D2H inside), config 4 (the bench density) and config 1 (one microscope view)
            from emu_synth import CONFIGS, default_params, make_view
            single = {}
            for cfg_i in (CFG, 1):
                pp = default_params(cfg_i, cell_um=CELL_UM, max_tracks_per_view=4096)
                pp["tube_ext_q"] = TUBE_EXT_Q
                pr = E.make_params(**{k: pp[k] for k in ("view_size_q", "cell_size_q", "sep_min_q", "sep_max_q", "tube_r2_q",
                                                          "min_grains", "max_tracks_per_view", "tube_ext_q")})
                views = [make_view(CONFIGS[cfg_i], cfg_i, v)[0] for v in range(args.latency_views)]
                nmax = max(len(g) for g in views)
                H1 = E.HostPath(pr, nmax, 1)
                ts = []
                for rep_i in range(2):                                  # the first round warms up
                    for g in views:
                        H1.n_grains = len(g)
                        H1.h_grains[:len(g)].copy_(torch.from_numpy(g))
                        H1.h_view_off.copy_(torch.tensor([0, len(g)], dtype=torch.int32))
                        torch.cuda.synchronize()
                        t0 = time.perf_counter()
                        H1.call()
                        if rep_i:
                            ts.append((time.perf_counter() - t0) * 1e3)
                single[f"config{cfg_i}"] = {"views": len(views), "grains_per_view": int(np.mean([len(g) for g in views])),
                                            "ms_median": float(np.median(ts)), "ms_max": float(np.max(ts))}
                del H1
                torch.cuda.empty_cache()
        except Exception as exc:                              # an extra leg may not take the headline down with it
            single = {"error": f"{type(exc).__name__}: {exc}"}
            torch.cuda.empty_cache()

    stream = None
    if args.stream_views > 0 and world == 1:
        try:
            # the same workload in batches through emu_stream_* (H2D of batch k+1 and D2H of batch k-1
            # behind the kernels of batch k), and config-1 views one per batch as a microscope would deliver them
            from emu_synth import CONFIGS, default_params, make_view
            stream = {}
            torch.cuda.empty_cache()
            SV, BV = min(args.stream_views, V), args.stream_batch
            nb = (SV + BV - 1) // BV
            bounds = [(b * BV, min(SV, (b + 1) * BV)) for b in range(nb)]
            S = E.StreamPath(prm, max(int(off[b1] - off[b0]) for b0, b1 in bounds), BV)

            def batch(b):
                b0, b1 = bounds[b]
                return grains[off[b0]:off[b1]], (off[b0:b1 + 1] - off[b0]).astype(np.int32)
            for rep_i in range(2):                                             # the first round warms up
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                nt_s = 0
                S.submit(*batch(0))
                for b in range(1, nb):
                    S.submit(*batch(b))
                    nt_s += S.collect(copy=False)["n_tracks"]
                nt_s += S.collect(copy=False)["n_tracks"]
                dt = time.perf_counter() - t0
            assert SV < V or nt_s == int(counts[E.EMU_CNT["tracks"]]), "the streamed batches and the one-call path disagree"
            # parity of the streamed path itself, element by element: views 0..nv_s-1 as ONE batch through the same
            # emu_stream object (the timed rounds above read only the counts back), against the oracle's result
            if parity is not None and ref_tracks is not None and nv_s <= min(BV, SV):
                S.submit(grains[:off[nv_s]], off[:nv_s + 1].astype(np.int32))
                parity["stream"] = same_as_oracle(S.collect(copy=True), ref_tracks)
                parity["identical"] = bool(parity["identical"] and parity["stream"])
            stream["config4"] = {"views": SV, "views_per_batch": BV, "grains_per_s": float(off[SV]) / dt, "views_per_s": SV / dt,
                                 "ms_per_view": dt / SV * 1e3, "tracks": nt_s,
                                 "call": "emu_stream_submit / emu_stream_collect, two batches in flight, pinned host buffers"}
            S.close(); del S
            torch.cuda.empty_cache()
            pp = default_params(1, cell_um=CELL_UM, max_tracks_per_view=4096)
            pp["tube_ext_q"] = TUBE_EXT_Q
            pr1 = E.make_params(**{k: pp[k] for k in ("view_size_q", "cell_size_q", "sep_min_q", "sep_max_q", "tube_r2_q",
                                                       "min_grains", "max_tracks_per_view", "tube_ext_q")})
            views = [make_view(CONFIGS[1], 1, v)[0] for v in range(32)]
            offs = [np.asarray([0, len(g)], np.int32) for g in views]
            S = E.StreamPath(pr1, max(len(g) for g in views), 1)
            for rep_i in range(2):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                S.submit(views[0], offs[0])
                for b in range(1, len(views)):
                    S.submit(views[b], offs[b])
                    S.collect(copy=False)
                S.collect(copy=False)
                dt = time.perf_counter() - t0
            stream["config1"] = {"views": len(views), "views_per_batch": 1, "views_per_s": len(views) / dt,
                                 "ms_per_view": dt / len(views) * 1e3, "microscope_rate_hz": 5.0}
            S.close(); del S
            torch.cuda.empty_cache()
        except Exception as exc:                              # an extra leg may not take the headline down with it
            stream = {"error": f"{type(exc).__name__}: {exc}"}
            torch.cuda.empty_cache()

    recog = None
    if args.recognize_views > 0:
        try:
            from emu_synth import CONFIGS, make_view
            from emu_synth.voxels import PITCH_Q, THRESHOLD, render_stack
            shape = (40, 1024, 1280)                                   # the paper's view: 1280 x 1024 px x 40 frames
            NV = args.recognize_views
            stacks = []
            for v in range(NV):
                g = make_view(CONFIGS[1], 1, v)[0].astype(np.int64)
                g = g[(g[:, 0] < shape[2] * PITCH_Q[0]) & (g[:, 1] < shape[1] * PITCH_Q[1])]      # the part of the view the stack covers
                stacks.append(render_stack(shape, g, key=(8, v)))
            vox = np.stack(stacks)
            d_vox = torch.from_numpy(vox).cuda()
            cap = 1 << 20
            d_g = torch.empty((cap, 4), dtype=torch.int32, device="cuda"); d_o = torch.empty(NV + 1, dtype=torch.int32, device="cuda")
            d_c = torch.zeros(1, dtype=torch.int64, device="cuda"); d_s = torch.zeros(1, dtype=torch.int64, device="cuda")
            ws = torch.empty(E.emu_recognize_ws_bytes(NV, shape[1], shape[0], cap), dtype=torch.uint8, device="cuda")
            for _ in range(3):
                E.emu_recognize_grains(d_vox, THRESHOLD, PITCH_Q, d_g, d_o, d_c, d_s, ws)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                E.emu_recognize_grains(d_vox, THRESHOLD, PITCH_Q, d_g, d_o, d_c, d_s, ws)
            e1.record(); torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / 5
            ng = int(d_c.cpu()[0])
            from oracle.recognize import recognize_grains as oracle_recognize     # the reported CPU baseline of this stage
            t0 = time.perf_counter(); ref = oracle_recognize(vox[0], THRESHOLD, PITCH_Q); t_or = time.perf_counter() - t0
            n0 = int(d_o.cpu()[1])
            same = bool(n0 == len(ref) and np.array_equal(d_g[:n0].cpu().numpy(), ref))
            alg = vox.size + 16.0 * ng + 4.0 * NV * shape[0] * shape[1]
            recog = {"views": NV, "voxels_per_view": int(vox[0].size), "grains": ng, "ms": ms, "views_per_s": NV / (ms * 1e-3),
                     "roofline": {"bound": "hbm", "achieved": alg / (ms * 1e-3) / 1e9, "peak": float(peaks["hbm_gbs"]), "unit": "GB/s",
                                  "frac": alg / (ms * 1e-3) / 1e9 / float(peaks["hbm_gbs"]),
                                  "algorithmic": "1 B per voxel + 16 B per grain + 4 B per row of voxels"},
                     "cpu_baseline": {"kind": "oracle (numpy)", "views_per_s": 1.0 / t_or, "cores": 1},
                     "first_view_identical_to_oracle": same}
            del d_vox
        except Exception as exc:                              # an extra leg may not take the headline down with it
            recog = {"error": f"{type(exc).__name__}: {exc}"}
            torch.cuda.empty_cache()

    val = n_total / (ms_step * 1e-3)
    line = {
        "metric": "grains_per_s", "value": val, "unit": "grains/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic", "config": workload_config(V, world),
        "views_per_s": V * world / (ms_step * 1e-3),
        "cm2_per_hour": V * world / (ms_step * 1e-3) * 3600 * VIEW_AREA_CM2,
        "find_workspace_gib": float(B_ws_bytes) / (1 << 30),
        "grains_per_gpu": n, "seeds": seeds, "candidates": int(counts[E.EMU_CNT["candidates"]]),
        "tracks": int(counts[E.EMU_CNT["tracks"]]),
        "tests_per_seed_gpu": float(counts[E.EMU_CNT["tests"]]) / max(1, seeds),
        "gpu_launches": int(sum(stage_launches.values())),
        "stage_ms_per_step": {k: v / args.steps for k, v in stage_ms.items()},
        "roofline": roofline, "roofline_bin": roofline_bin, "cpu_baseline": cpu, "e2e": e2e, "clocks": clocks,
        "single_view": single, "stream": stream, "recognize": recog, "parity": parity,
        "timing_note": "emu_profile is active inside the timed region: a pair of CUDA events around every launch of the "
                       "library (the per-stage times and gpu_launches come from them); value is therefore conservative",
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    if parity is not None and not parity["identical"]:
        sys.exit("bench.py: the timed run is NOT identical to the oracle on the checked views: " + json.dumps(parity))


if __name__ == "__main__":
    main()
