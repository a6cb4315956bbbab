"""Pins of the grain-recognition oracle (oracle/recognize.py): hand-made stacks
whose answer follows from the definition, the plain-loop / exact-Fraction restatement on small random stacks, and the
recovery of rendered grains.  All CPU (-m "not gpu")."""
import numpy as np
import pytest

from emu_synth.voxels import PITCH_Q, THRESHOLD, random_grains_q, render_stack
from oracle.recognize import recognize_grains, recognize_grains_loops


def _stack(shape=(5, 7, 9)):
    return np.zeros(shape, np.uint8)


def test_single_voxel_and_threshold_is_strict():
    v = _stack(); v[2, 3, 4] = 41
    r = recognize_grains(v, 40, PITCH_Q)
    # one voxel above the threshold: the grain sits at the centre of that voxel, (i + 1/2) * pitch, rounded half up
    assert r.tolist() == [[int(4.5 * 15 + 0.5), int(3.5 * 16 + 0.5), int(2.5 * 80 + 0.5), 41]]
    v[2, 3, 4] = 40
    assert len(recognize_grains(v, 40, PITCH_Q)) == 0          # "higher than a given threshold"


def test_symmetric_blob_gives_the_centre_and_one_grain():
    v = _stack()
    v[1:4, 2:5, 3:6] = 60; v[2, 3, 4] = 200                     # a 3x3x3 shell round one maximum
    r = recognize_grains(v, 40, PITCH_Q)
    assert r.tolist() == [[68, 56, 200, 200]]                   # (4.5*15, 3.5*16, 2.5*80) = (67.5 -> 68, 56, 200)


def test_centre_of_mass_closed_form():
    """weights 100 at x = 4 and 50 at x = 5 (both above the threshold): centre of mass index 4 + 1/3, so
    x = 15 * (4.8333..) = 72.5 -> 73 exactly at the rounding boundary (half up); a weight at or below the threshold
    does not pull."""
    v = _stack(); v[2, 3, 4] = 100; v[2, 3, 5] = 50
    assert recognize_grains(v, 40, PITCH_Q)[0].tolist() == [73, 56, 200, 100]
    v[2, 3, 5] = 40
    assert recognize_grains(v, 40, PITCH_Q)[0].tolist() == [68, 56, 200, 100]
    v[2, 3, 5] = 50; v[3, 3, 4] = 100                            # an equal neighbour one frame deeper: z index 2.4
    r = recognize_grains(v, 40, PITCH_Q)
    assert len(r) == 1 and r[0].tolist() == [int(15 * (4 + 50 / 250 + 0.5) + 0.5), 56, int(80 * (2 + 100 / 250 + 0.5) + 0.5), 100]


def test_plateau_gives_exactly_one_grain_the_first_in_raster_order():
    v = _stack(); v[2, 3, 4] = 90; v[2, 3, 5] = 90; v[2, 4, 4] = 90; v[3, 3, 4] = 90
    r = recognize_grains(v, 40, PITCH_Q)
    assert len(r) == 1
    # the winner is voxel (z, y, x) = (2, 3, 4); centre of mass of the four equal weights
    assert r[0].tolist() == [int(15 * (4.25 + 0.5) + 0.5), int(16 * (3.25 + 0.5) + 0.5), int(80 * (2.25 + 0.5) + 0.5), 90]


def test_border_voxels_and_two_separate_grains():
    v = _stack(); v[0, 0, 0] = 77; v[4, 6, 8] = 99; v[4, 6, 6] = 98    # two voxels apart: not neighbours
    r = recognize_grains(v, 40, PITCH_Q)
    assert r[:, 3].tolist() == [77, 98, 99]                      # raster order of the defining voxels
    assert r[0, :3].tolist() == [8, 8, 40]


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_numpy_oracle_equals_plain_loops(seed):
    rng = np.random.default_rng(seed)
    v = rng.integers(0, 256, size=(6, 9, 11)).astype(np.uint8)
    v[rng.random(v.shape) < 0.5] //= 8                          # a mix of background and bright voxels, many ties
    v[2:4, 3:6, 4:7] = 133                                       # a plateau
    a, b = recognize_grains(v, 60, PITCH_Q), recognize_grains_loops(v, 60, PITCH_Q)
    assert len(a) > 5 and np.array_equal(a, b)
    a, b = recognize_grains(v, 0, (64, 64, 64)), recognize_grains_loops(v, 0, (64, 64, 64))
    assert np.array_equal(a, b)


def test_rendered_grains_are_recovered():
    """Grains rendered by the generator (Gaussian blobs on a flat background) come back one for one when they are
    well separated, within half a voxel of where they were put."""
    shape = (16, 96, 128)
    g = random_grains_q(shape, 60, key=(7, 5))
    d = np.abs(g[:, None, :] - g[None, :, :]) / np.asarray(PITCH_Q)
    keep = [i for i in range(len(g)) if all(d[i, j].max() > 9 for j in range(len(g)) if j != i)]
    g = g[keep]
    v = render_stack(shape, g, key=(7, 6))
    r = recognize_grains(v, THRESHOLD, PITCH_Q)
    assert len(r) == len(g) > 10
    for p in g:
        e = np.abs(r[:, :3] - p[:3]) / np.asarray(PITCH_Q)
        assert e.max(axis=1).min() <= 0.5
