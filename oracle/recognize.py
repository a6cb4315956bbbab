"""CPU oracle of the 3D grain recognition (section 2).

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as the rest of oracle/): plain numpy, the definition written out,
no tiling, no shared code with paper_1311_5334_b200.

The paper: "Each pixel with a pulse height higher than a given threshold is compared to the 3 x 3 x 3
neighboring pixels; the pixel with the highest pulse height among these will be defining the grain.  The spatial
coordinates of the grains are then computed with a center-of-mass method using the pulse height of each pixel."

Readings (the paper gives no formula; DESIGN.md section 3b lists them):
  R1  input: one view as a stack of filtered frames vox[nz][ny][nx], uint8 pulse heights (x fastest).
  R2  a voxel v DEFINES A GRAIN iff I(v) > thr and I(v) is the highest of its 3x3x3 neighbourhood; voxels outside the
      stack count as 0.  Ties (a plateau of equal maxima) must give ONE grain: v wins against an equal neighbour only
      if v comes first in raster order (z, then y, then x), i.e. I(v) > I(n) for neighbours n before v and
      I(v) >= I(n) for neighbours after v.
  R3  centre of mass over the same 3x3x3 neighbourhood, weight w(n) = I(n) if I(n) > thr else 0 ("using the pulse
      height of each pixel"; pixels at or below the threshold carry none after the filtering).
  R4  coordinates in q = 1/64 um: the centre of voxel index i along an axis of pitch p q is (i + 1/2) p, so
      pos_q = floor(p * (sum w i / sum w + 1/2) + 1/2) = (2 p sum(w i) + p sum(w) + sum(w)) // (2 sum(w)), exact
      in integers.
  R5  output: one record (x_q, y_q, z_q, I(v)) per grain, listed in raster order of the defining voxel.
"""
from __future__ import annotations

import numpy as np


def recognize_grains(vox: np.ndarray, thr: int, pitch_q) -> np.ndarray:
    """vox: uint8 [nz, ny, nx]; returns int32 [n, 4] = (x_q, y_q, z_q, peak), raster order of the peak voxel."""
    vox = np.ascontiguousarray(vox, np.uint8)
    nz, ny, nx = vox.shape
    I = np.zeros((nz + 2, ny + 2, nx + 2), np.int64)          # a border of zeros: voxels outside the stack (R2)
    I[1:-1, 1:-1, 1:-1] = vox
    C = I[1:-1, 1:-1, 1:-1]
    peak = C > int(thr)
    W = np.where(I > int(thr), I, 0)                           # weights (R3)
    sw = np.zeros(C.shape, np.int64)
    swi = [np.zeros(C.shape, np.int64) for _ in range(3)]      # sum of w * (offset along x, y, z)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                N = I[1 + dz:nz + 1 + dz, 1 + dy:ny + 1 + dy, 1 + dx:nx + 1 + dx]
                if (dz, dy, dx) < (0, 0, 0):
                    peak &= C > N                              # a neighbour before v in raster order: strictly higher
                elif (dz, dy, dx) > (0, 0, 0):
                    peak &= C >= N                             # a neighbour after v: at least as high
                w = W[1 + dz:nz + 1 + dz, 1 + dy:ny + 1 + dy, 1 + dx:nx + 1 + dx]
                sw += w
                swi[0] += w * dx; swi[1] += w * dy; swi[2] += w * dz
    zz, yy, xx = np.nonzero(peak)                              # raster order (R5)
    idx = (xx, yy, zz)
    out = np.zeros((len(zz), 4), np.int32)
    s = sw[zz, yy, xx]
    for a in range(3):
        p = int(pitch_q[a])
        swa = swi[a][zz, yy, xx] + s * idx[a]                  # sum of w * absolute index
        out[:, a] = (2 * p * swa + p * s + s) // (2 * s)      # R4
    out[:, 3] = C[zz, yy, xx]
    return out


def recognize_grains_loops(vox: np.ndarray, thr: int, pitch_q) -> np.ndarray:
    """The same definition as plain Python loops with exact Fractions (tiny stacks only): the pin of the numpy version."""
    from fractions import Fraction
    nz, ny, nx = vox.shape

    def at(z, y, x):
        return int(vox[z, y, x]) if 0 <= z < nz and 0 <= y < ny and 0 <= x < nx else 0

    out = []
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                c = at(z, y, x)
                if c <= thr:
                    continue
                ok, sw, sx, sy, sz = True, 0, 0, 0, 0
                for dz in (-1, 0, 1):
                    for dy in (-1, 0, 1):
                        for dx in (-1, 0, 1):
                            n = at(z + dz, y + dy, x + dx)
                            before = (z + dz, y + dy, x + dx) < (z, y, x)
                            if (dz, dy, dx) != (0, 0, 0) and (n > c or (before and n == c)):
                                ok = False
                            w = n if n > thr else 0
                            sw += w; sx += w * (x + dx); sy += w * (y + dy); sz += w * (z + dz)
                if ok:
                    pos = [int((Fraction(p) * (Fraction(sa, sw) + Fraction(1, 2)) + Fraction(1, 2)).__floor__())
                           for p, sa in zip(pitch_q, (sx, sy, sz))]
                    out.append(pos + [c])
    return np.asarray(out, np.int32).reshape(-1, 4)
