"""Seeded synthetic voxel stacks of one emulsion view (inputs only).

Stand-in for the filtered camera frames of the paper (1280 x 1024 pixels x 40 frames for a view of
300 x 250 x 50 um, i.e. about 0.234 x 0.244 um pixels and 1.25 um frames; "a grain produces a signal of a few pixels
in X, Y and a few frames in depth").  Recipe:

* voxel pitch 15 x 16 x 80 q (0.234 x 0.25 x 1.25 um at q = 1/64 um);
* every grain is a Gaussian blob, sigma 1.3 px in x and y and 0.9 frames in z, peak pulse height uniform in [90, 250],
  centred at the grain's position; blobs add up;
* background: independent pulse heights uniform in [0, noise_max] (after the paper's filtering the background is
  low and flat); everything is clipped to [0, 255] and stored as uint8;
* the recognition threshold that goes with it: 40.

No recognition arithmetic lives here; the random numbers come from the counter-based stream of views.py.
"""
from __future__ import annotations

import numpy as np

from .views import Stream

PITCH_Q = (15, 16, 80)
THRESHOLD = 40


def render_stack(shape, grains_q: np.ndarray, key=(7, 0), noise_max: int = 12, sigma_px=(1.3, 1.3, 0.9)) -> np.ndarray:
    """shape = (nz, ny, nx); grains_q int [n, >=3] positions in q.  Returns the uint8 stack."""
    nz, ny, nx = shape
    st = Stream(*key)
    img = np.floor(st.uniform(nz * ny * nx) * (noise_max + 1)).astype(np.float32).reshape(nz, ny, nx)
    n = len(grains_q)
    amp = 90.0 + st.uniform(max(n, 1))[:n] * 160.0
    rx, ry, rz = (int(np.ceil(3 * s)) for s in sigma_px)
    for g, a in zip(np.asarray(grains_q, np.float64), amp):
        c = [g[i] / PITCH_Q[i] - 0.5 for i in range(3)]          # centre in voxel index units (voxel i spans [i, i+1) p)
        ix, iy, iz = (int(round(v)) for v in c)
        x0, x1 = max(ix - rx, 0), min(ix + rx + 1, nx)
        y0, y1 = max(iy - ry, 0), min(iy + ry + 1, ny)
        z0, z1 = max(iz - rz, 0), min(iz + rz + 1, nz)
        if x0 >= x1 or y0 >= y1 or z0 >= z1:
            continue
        ex = np.exp(-0.5 * ((np.arange(x0, x1) - c[0]) / sigma_px[0]) ** 2)
        ey = np.exp(-0.5 * ((np.arange(y0, y1) - c[1]) / sigma_px[1]) ** 2)
        ez = np.exp(-0.5 * ((np.arange(z0, z1) - c[2]) / sigma_px[2]) ** 2)
        img[z0:z1, y0:y1, x0:x1] += a * ez[:, None, None] * ey[None, :, None] * ex[None, None, :]
    return np.clip(np.floor(img + 0.5), 0, 255).astype(np.uint8)


def random_grains_q(shape, n: int, key=(7, 1), margin_px: int = 4) -> np.ndarray:
    """n grain positions (q) uniform inside the stack, margin_px voxels away from its faces."""
    nz, ny, nx = shape
    st = Stream(*key)
    u = st.uniform(3 * n).reshape(n, 3)
    lo = np.asarray([margin_px * PITCH_Q[0], margin_px * PITCH_Q[1], min(margin_px, nz // 4) * PITCH_Q[2]], np.float64)
    hi = np.asarray([nx * PITCH_Q[0], ny * PITCH_Q[1], nz * PITCH_Q[2]], np.float64) - lo
    return np.floor(lo + u * (hi - lo)).astype(np.int32)
