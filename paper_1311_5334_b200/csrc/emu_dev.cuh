// emu_dev.cuh - device-side parameter block, cell arithmetic and the tube walker shared by the
// kernels of libemu4pi.  Product code: shares nothing with oracle/.
//
// Citations: P:NN = PAPER.md line NN; "reading Qn" = DESIGN.md section 3.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/emu.h"

#define EMU_FULL 0xffffffffu

// Frames.  The tube walk of emu_find.cu wants the line's dominant axis to be the axis the rows of cells
// run along, so every view is binned three times, once per choice of the first axis:
//   frame 0: (u,v,w) = (x,y,z)   frame 1: (u,v,w) = (y,x,z)   frame 2: (u,v,w) = (z,x,y)
// (w = z wherever possible: a view is flat, a line crosses few z layers, and w is the outer loop of the walk)
// The cell size triple cs[] applies to (u,v,w) in every frame; frame 0 is the binning the C ABI defines.
struct EmuFrame { int n[3]; int ncell; };

struct EmuDev {           // passed by value to every kernel
  EmuFrame fr[3];         // grid of every frame: n = ceil(view_size[perm] / cs); fr[0] = {n, ncell}
  int n[3];               // cells per axis = ceil(view_size / cell_size)
  int cs[3];              // cell size, q
  float inv_cs[3];
  int ncell;              // per view
  int sep_max;            // q
  int sep_min2, sep_max2; // q^2 (sep_max <= 2048 -> < 2^22)
  int r2;                 // tube radius^2, q^2
  float Rw;               // walk radius: ceil(sqrt(r2)) + 2 q of slack for the float bounds
  int min_grains;
  int max_tracks;
  int ext;                // tube_ext_q: -1 = whole line, >= 0 = bounded tube
  // brick kernels (emu_find.cu): cell index of a dilated bound without a float->int conversion,
  //   lo = rn(x * inv_cs + klo), hi = rn(x * inv_cs + khi), klo = -(Rw * inv_cs + 0.5), khi = Rw * inv_cs - 0.5
  float klo[3], khi[3];
  float csf[3];           // cell size as float
  float Rup;              // ceil(sqrt(r2)) as float (error band of the float tube test)
  int packed_ok;          // 1: the 4-byte grain format of the brick kernels can hold a view of this grid
  int angle_min[8];       // angle-dependent cut: minimum members per bin of |cos theta|, 0 = none
  int angle_cut;          // 1: some entry of angle_min exceeds min_grains (the cut can remove a track)
};

// lab axis of coordinate i of frame f
__host__ __device__ __forceinline__ int emu_frame_axis(int f, int i) {
  return f == 0 ? i : (f == 1 ? (i == 0 ? 1 : (i == 1 ? 0 : 2)) : (i == 0 ? 2 : i - 1));
}

// lab coordinates -> frame coordinates (w is carried along)
__host__ __device__ __forceinline__ int4 emu_to_frame(int f, int4 g) {
  if (f == 1) return make_int4(g.y, g.x, g.z, g.w);
  if (f == 2) return make_int4(g.z, g.x, g.y, g.w);
  return g;
}

// floor(c / cs) clamped to [0, n-1] (reading Q13: out-of-box grains land in the boundary cells).
// |c| < 2^18 here, so the float quotient is within 1 of the truth and one correction step is exact.
__device__ __forceinline__ int emu_cell_axis(int c, int cs, float inv_cs, int n) {
  int q = __float2int_rd((float)c * inv_cs);
  int r = c - q * cs;
  q += (r >= cs) - (r < 0);
  return min(max(q, 0), n - 1);
}

__device__ __forceinline__ int emu_cell_of(const EmuDev& P, int x, int y, int z) {
  int cx = emu_cell_axis(x, P.cs[0], P.inv_cs[0], P.n[0]);
  int cy = emu_cell_axis(y, P.cs[1], P.inv_cs[1], P.n[1]);
  int cz = emu_cell_axis(z, P.cs[2], P.inv_cs[2], P.n[2]);
  return cx + P.n[0] * (cy + P.n[1] * cz);
}

// cell of a grain given in the coordinates of frame f
__device__ __forceinline__ int emu_cell_of_frame(const EmuDev& P, int f, int u, int v, int w) {
  const EmuFrame& F = P.fr[f];
  int cu = emu_cell_axis(u, P.cs[0], P.inv_cs[0], F.n[0]);
  int cv = emu_cell_axis(v, P.cs[1], P.inv_cs[1], F.n[1]);
  int cw = emu_cell_axis(w, P.cs[2], P.inv_cs[2], F.n[2]);
  return cu + F.n[0] * (cv + F.n[1] * cw);
}

// view that owns sorted position / row g: largest v in [v0, v1) with view_off[v] <= g
__device__ __forceinline__ int emu_find_view(const int* __restrict__ view_off, int v0, int v1, int g) {
  int lo = v0, hi = v1;              // invariant: view_off[lo] <= g < view_off[hi]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (__ldg(view_off + mid) <= g) lo = mid; else hi = mid;
  }
  return lo;
}

// Exact tube predicate ("the number of grains along the line"):
// P in tube <=> |(P-A) x d|^2 <= r2 * |d|^2.  |v| < 2^18, |d| < 2^11: every cross component fits
// int32 (< 2^30); the three squares are summed in 64 bits (< 2^62).
__device__ __forceinline__ bool emu_in_tube(int px, int py, int pz, int ax, int ay, int az,
                                            int dx, int dy, int dz, long long r2D2) {
  int vx = px - ax, vy = py - ay, vz = pz - az;
  int cx = vy * dz - vz * dy;
  int cy = vz * dx - vx * dz;
  int cz = vx * dy - vy * dx;
  long long s = (long long)cx * cx + (long long)cy * cy + (long long)cz * cz;
  return s <= r2D2;
}

// Bounded tube (tube_ext_q >= 0, Fig. 4(b) "along the seed"): along the line the grain must
// lie between the two seed grains or at most ext beyond either:  -ext |d| <= (P-A).d <= D2 + ext |d|, compared exactly
// through squares.  |s| < 2^31, ext <= 2^16, D2 < 2^22: every product below 2^62.  ext < 0: the whole line.
__device__ __forceinline__ bool emu_axial_ok(int ext, long long s, long long d2) {
  if (ext < 0) return true;
  const long long e2d2 = (long long)ext * ext * d2;
  if (s < 0 && s * s > e2d2) return false;
  const long long t = s - d2;
  if (t > 0 && t * t > e2d2) return false;
  return true;
}

__device__ __forceinline__ int emu_clampcell_f(float x, float inv_cs, int n) {
  return (int)fminf(fmaxf(floorf(x * inv_cs), 0.0f), (float)(n - 1));
}

struct EmuBox { int lo[3], hi[3]; };   // bounding box of one view's grains (q), computed on the device

// Walk every (cy,cz) row of cells the tube of the infinite line A + t*d can touch and call
// hit(j) for each sorted position j whose grain passes the exact integer test.  Rows are taken
// layer by layer in z, then in y; inside a row the cells cx0..cx1 are consecutive in memory, so a
// row costs two cell_start loads and one contiguous run of grains.
//
// The bounds are conservative float intervals: a grain in the tube is within R = ceil(sqrt(r2)) of
// its foot X(t*) on the line in every coordinate, so if the grain sits in row (cy,cz) then t* lies
// in the intersection of the two slab intervals widened by R, and the grain's x is within R of
// x(t*).  Rw = R + 2 absorbs the float rounding (|coord| < 2^18: errors are below 0.1 q).  The two
// boundary cells of every axis are open-ended because out-of-box grains are clamped into them
// (reading Q13); they reach as far as the data do, i.e. to the view's bounding box `bb`.
// Returns the number of point-line tests executed.
template <class Hit>
__device__ __forceinline__ int emu_walk_tube(const EmuDev& P, const EmuBox& bb, const int4* __restrict__ sorted,
                                             const int* __restrict__ cell_start, int vcell_base,
                                             int ax, int ay, int az, int dx, int dy, int dz,
                                             long long r2D2, Hit&& hit) {
  const float BIG = 1.0e9f;
  const float R = P.Rw;
  const float fax = (float)ax, fay = (float)ay, faz = (float)az;
  const float fdx = (float)dx, fdy = (float)dy;
  const float inv_dy = dy ? 1.0f / (float)dy : 0.0f;
  const float inv_dz = dz ? 1.0f / (float)dz : 0.0f;
  const int nx = P.n[0], ny = P.n[1], nz = P.n[2];
  int tests = 0;
  const long long d2 = (long long)dx * dx + (long long)dy * dy + (long long)dz * dz;
  int cz_lo = 0, cz_hi = nz - 1;
  if (dz == 0) {
    cz_lo = emu_clampcell_f(faz - R, P.inv_cs[2], nz);
    cz_hi = emu_clampcell_f(faz + R, P.inv_cs[2], nz);
  }
  for (int cz = cz_lo; cz <= cz_hi; ++cz) {
    float tz0 = -BIG, tz1 = BIG;
    if (dz != 0) {
      int lo = (cz == 0) ? bb.lo[2] : cz * P.cs[2];
      int hi = (cz == nz - 1) ? bb.hi[2] : (cz + 1) * P.cs[2] - 1;
      if (lo > hi) continue;
      float a = ((float)lo - R - faz) * inv_dz, b = ((float)hi + R - faz) * inv_dz;
      tz0 = fminf(a, b); tz1 = fmaxf(a, b);
    }
    float ya = fmaf(tz0, fdy, fay), yb = fmaf(tz1, fdy, fay);
    int cy0 = emu_clampcell_f(fminf(ya, yb) - R, P.inv_cs[1], ny);
    int cy1 = emu_clampcell_f(fmaxf(ya, yb) + R, P.inv_cs[1], ny);
    for (int cy = cy0; cy <= cy1; ++cy) {
      float t0 = tz0, t1 = tz1;
      if (dy != 0) {
        int lo = (cy == 0) ? bb.lo[1] : cy * P.cs[1];
        int hi = (cy == ny - 1) ? bb.hi[1] : (cy + 1) * P.cs[1] - 1;
        if (lo > hi) continue;
        float a = ((float)lo - R - fay) * inv_dy, b = ((float)hi + R - fay) * inv_dy;
        t0 = fmaxf(t0, fminf(a, b)); t1 = fminf(t1, fmaxf(a, b));
      }
      if (t0 > t1) continue;
      float xa = fmaf(t0, fdx, fax), xb = fmaf(t1, fdx, fax);
      int cx0 = emu_clampcell_f(fminf(xa, xb) - R, P.inv_cs[0], nx);
      int cx1 = emu_clampcell_f(fmaxf(xa, xb) + R, P.inv_cs[0], nx);
      int rb = vcell_base + (cz * ny + cy) * nx;
      int s = __ldg(cell_start + rb + cx0), e = __ldg(cell_start + rb + cx1 + 1);
      for (int j = s; j < e; ++j) {
        int4 p = __ldg(sorted + j);
        ++tests;
        if (emu_in_tube(p.x, p.y, p.z, ax, ay, az, dx, dy, dz, r2D2) &&
            emu_axial_ok(P.ext, (long long)(p.x - ax) * dx + (long long)(p.y - ay) * dy + (long long)(p.z - az) * dz, d2)) hit(j);
      }
    }
  }
  return tests;
}
