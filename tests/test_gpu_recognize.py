"""Parity of emu_recognize_grains against oracle/recognize.py: integer work, bit-exact, order
included (raster order of the defining voxel, view after view)."""
import numpy as np
import pytest

from emu_synth.voxels import PITCH_Q, THRESHOLD, random_grains_q, render_stack

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def E():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    import paper_1311_5334_b200 as E
    E.exported_symbols()
    return E


def _gpu(E, vox, thr, pitch, capacity=None):
    import torch
    d_vox = torch.from_numpy(np.ascontiguousarray(vox)).cuda()
    nv, nz, ny, nx = vox.shape
    cap = capacity if capacity is not None else max(1, vox.size // 8)
    d_g = torch.zeros((cap, 4), dtype=torch.int32, device="cuda")
    d_off = torch.zeros(nv + 1, dtype=torch.int32, device="cuda")
    d_cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    d_st = torch.zeros(1, dtype=torch.int64, device="cuda")
    ws = torch.empty(E.emu_recognize_ws_bytes(nv, ny, nz, cap), dtype=torch.uint8, device="cuda")
    E.emu_recognize_grains(d_vox, thr, pitch, d_g, d_off, d_cnt, d_st, ws)
    torch.cuda.synchronize()
    n = int(d_cnt.cpu()[0])
    return d_g[:min(n, cap)].cpu().numpy(), d_off.cpu().numpy(), n, int(d_st.cpu()[0])


def _oracle(vox, thr, pitch):
    from oracle.recognize import recognize_grains
    parts = [recognize_grains(v, thr, pitch) for v in vox]
    off = np.zeros(len(vox) + 1, np.int32)
    off[1:] = np.cumsum([len(p) for p in parts])
    return np.concatenate(parts) if parts else np.zeros((0, 4), np.int32), off


@pytest.mark.parametrize("shape", [(3, 12, 70, 133), (1, 40, 64, 260), (2, 5, 33, 128)])
def test_rendered_stacks_bit_exact(E, shape):
    """ragged row lengths (133, 260: not multiples of the 128 voxels a warp takes per step), several views"""
    nv, nz, ny, nx = shape
    vox = np.stack([render_stack((nz, ny, nx), random_grains_q((nz, ny, nx), 150, key=(7, 10 + v)), key=(7, 20 + v))
                    for v in range(nv)])
    ref, roff = _oracle(vox, THRESHOLD, PITCH_Q)
    got, off, n, st = _gpu(E, vox, THRESHOLD, PITCH_Q)
    assert st == 0 and n == len(ref) > 50 * nv
    assert np.array_equal(off, roff) and np.array_equal(got, ref)


def test_random_noise_with_ties_and_borders(E):
    """dense random stacks: many equal maxima (the raster tie rule decides), grains on every face of the stack"""
    rng = np.random.default_rng(3)
    vox = rng.integers(0, 40, size=(2, 7, 37, 150)).astype(np.uint8)
    vox[rng.random(vox.shape) < 0.02] = 200
    vox[0, 2:4, 10:13, 20:24] = 133
    for thr, pitch in ((20, PITCH_Q), (0, (64, 64, 64)), (199, (1, 4096, 7))):
        ref, roff = _oracle(vox, thr, pitch)
        got, off, n, st = _gpu(E, vox, thr, pitch)
        assert st == 0 and n == len(ref) > 0
        assert np.array_equal(off, roff) and np.array_equal(got, ref)


def test_empty_and_capacity(E):
    vox = np.zeros((2, 3, 8, 16), np.uint8)
    got, off, n, st = _gpu(E, vox, 10, PITCH_Q)
    assert n == 0 and st == 0 and off.tolist() == [0, 0, 0]
    vox[:, 1, 4, ::4] = 90
    got, off, n, st = _gpu(E, vox, 10, PITCH_Q, capacity=3)
    assert n == 8 and st & E.EMU_ST["grain_overflow"]


def test_recognized_grains_feed_the_track_path(E, oracle_mod):
    """the chain A0 -> A1..A7 on the device: a stack rendered from a noiseless track plus fog is recognised and the
    grain list goes straight into emu_bin_grains / emu_find_tracks / emu_fit_tracks; the track list equals the
    oracle's on the oracle's own recognised grains."""
    import torch
    shape = (24, 160, 200)                                       # 3000 x 2560 x 1920 q
    line = np.asarray([[300 + 190 * i, 400 + 120 * i, 300 + 90 * i] for i in range(12)], np.int32)
    fog = random_grains_q(shape, 40, key=(7, 31))
    vox = render_stack(shape, np.concatenate([line, fog]), key=(7, 32))[None]
    ref_g, ref_off = _oracle(vox, THRESHOLD, PITCH_Q)
    got_g, off, n, st = _gpu(E, vox, THRESHOLD, PITCH_Q)
    assert np.array_equal(got_g, ref_g)
    p = dict(view_size_q=(3000, 2560, 1920), cell_size_q=(256, 256, 256), sep_min_q=128, sep_max_q=1280, tube_r2_q=2621,
             tube_ext_q=-1, min_grains=8, max_tracks_per_view=64)
    from gpu_helpers import assert_same_tracks, run_gpu
    ref = oracle_mod.track_views(p, ref_g, ref_off, "brute", 1)
    assert len(ref.tracks) >= 1
    assert_same_tracks(E, run_gpu(E, p, got_g, off), ref)
