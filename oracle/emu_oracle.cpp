// emu_oracle.cpp - CPU ORACLE for the 4pi emulsion track-finding hot path.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
// It shares no code, header, table or helper with paper_1311_5334_b200/ (the ABI
// structs below are re-typed, not included), and it never reads anything the CUDA
// path produced.
//
// What it computes: the algorithm of Ariga & Ariga, arXiv 1311.5334, section 2
// (PAPER.md:72 and footnote PAPER.md:118, Fig. 4), step by step in the
// paper's order, with the readings of SURVEY.md 8(c) (listed in DESIGN.md) where the
// paper is silent.  Integer arithmetic throughout (int64_t), float64 only in the fit.
//
//   O1 bin        PAPER.md:118  every grain attributed to a 3D cell ("hash table")
//   O2 seeds      PAPER.md:72   "any grain pair whose distance is smaller than 25 um"
//   O3 count      PAPER.md:72   "a line is then defined connecting the two grains and the
//                               number of grains along the line is evaluated"
//   O4 threshold  PAPER.md:72   "above a preset threshold (e.g. 5) -> track"
//   O5 associate  PAPER.md:72   "each grain is exclusively associated with one track using
//                               that grain ... and again the threshold ... is applied"
//   O6 fit        BASELINE.json north_star (not in the paper): least-squares line
//   O7 order      SURVEY.md 8(c) O7: views ascending, tracks best-first
//   O5b angle cut SURVEY.md 8(f) NEXT-2, PAPER.md:144 (Fig. 8(c)): "a cut on the number of grains is applied
//                 according to the line drawn in the figure" - the line is not given numerically, so it is a table
//                 parameter: minimum members per bin of |cos theta| of the FITTED direction, applied after O5
//                 (reading Q17 in DESIGN.md).  All entries 0 (or <= min_grains): no effect.
//
// Two modes give the same result by construction (a test checks it):
//   mode 0 "brute": no cells at all - every seed is tested against every grain.
//   mode 1 "cells": the paper's 3D hash cells restrict both the pair search
//                   and the tube count to "the grains in the relevant cells".
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): hand-derived example E1 (tests/golden),
// exact-rational brute force over all grain triples on tiny inputs, exact recovery of
// noiseless tracks, permutation and x<->y invariance, cell-size independence,
// numpy.polyfit / Fraction for the fit, Poisson closed form for the efficiency.
// The paper's own 99.0 % / 1.4 % need real emulsion: PARITY UNPINNED.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

typedef struct emo_params {      // same field order as the library's params struct (re-typed)
  int32_t struct_size;
  int32_t view_size_q[3];
  int32_t cell_size_q[3];
  int32_t sep_min_q;
  int32_t sep_max_q;
  int32_t tube_r2_q;
  int32_t tube_ext_q;
  int32_t min_grains;
  int32_t max_tracks_per_view;
  int32_t reserved[4];
  int32_t angle_min_grains[8];   // NEXT-2: minimum members per bin of |cos theta|; 0 = no cut in the bin
} emo_params;

typedef struct emo_track {       // 32 B
  int32_t view, seed_a, seed_b;  // seed grains: rows of the input array, seed_a < seed_b
  int32_t n_tube, n_members;
  int32_t member_off;
  int32_t seed_d2, pad;
} emo_track;

typedef struct emo_fit {         // 48 B
  int32_t axis, n, u_min, u_max;
  double slope[2], icpt[2];
} emo_fit;

}  // extern "C"

namespace {

typedef int64_t i64;

struct Grain { int32_t x, y, z, row; };       // row = row in the caller's array (original index)

inline i64 floor_div(i64 a, i64 b) {          // b > 0
  i64 q = a / b, r = a % b;
  return (r != 0 && r < 0) ? q - 1 : q;
}
inline i64 clampi(i64 v, i64 lo, i64 hi) { return v < lo ? lo : (v > hi ? hi : v); }

struct Grid {
  i64 n[3], cs[3];
  double inv_cs[3];
  explicit Grid(const emo_params& p) {
    for (int i = 0; i < 3; ++i) {
      cs[i] = p.cell_size_q[i];
      inv_cs[i] = 1.0 / (double)cs[i];
      n[i] = (p.view_size_q[i] + cs[i] - 1) / cs[i];      // ceil(view_size / cell_size)
      if (n[i] < 1) n[i] = 1;
    }
  }
  i64 n_cells() const { return n[0] * n[1] * n[2]; }
  i64 ci(int axis, i64 coord) const { return clampi(floor_div(coord, cs[axis]), 0, n[axis] - 1); }
  i64 cell(i64 x, i64 y, i64 z) const { return ci(0, x) + n[0] * (ci(1, y) + n[1] * ci(2, z)); }
};

// O1 - SURVEY 8(c) O1 / PAPER.md:118.  Stable sort of one view's grains by cell id.
void bin_view(const Grid& g, const int32_t* grains, int32_t row0, int32_t n,
              std::vector<int32_t>& order /* local indices */, std::vector<int32_t>& cell_start) {
  std::vector<i64> cell(n);
  for (int32_t i = 0; i < n; ++i) {
    const int32_t* p = grains + 4 * (i64)(row0 + i);
    cell[i] = g.cell(p[0], p[1], p[2]);
  }
  order.resize(n);
  for (int32_t i = 0; i < n; ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return cell[a] < cell[b]; });
  cell_start.assign(g.n_cells() + 1, 0);
  for (int32_t i = 0; i < n; ++i) cell_start[cell[i] + 1] += 1;
  for (i64 c = 0; c < g.n_cells(); ++c) cell_start[c + 1] += cell_start[c];
}

// O3 predicate - SURVEY 8(c) O3: P in tube <=> |(P-A) x (B-A)|^2 <= r2 * |B-A|^2.
// Bounded tube (Fig. 4(b) "along the seed"): with ext = tube_ext_q >= 0 the grain
// must also lie, along the line, between the two seed grains or at most ext beyond either of them:
//   -ext |d| <= (P-A).d <= D2 + ext |d|,  compared exactly through squares (s < 0: s^2 <= ext^2 D2, and the same for
// s - D2 > 0).  Swapping A and B turns s into D2 - s, so the predicate stays orientation-free.  ext = -1: whole line.
// |s| < 3 * 2^18 * 2^11 < 2^31 and ext <= 2^16, D2 < 2^22: every product below 2^62.
inline bool in_tube(const Grain& A, i64 dx, i64 dy, i64 dz, i64 r2D2, const Grain& P, i64 d2, i64 ext) {
  i64 vx = (i64)P.x - A.x, vy = (i64)P.y - A.y, vz = (i64)P.z - A.z;
  i64 cx = vy * dz - vz * dy;
  i64 cy = vz * dx - vx * dz;
  i64 cz = vx * dy - vy * dx;
  if (cx * cx + cy * cy + cz * cz > r2D2) return false;
  if (ext < 0) return true;
  const i64 s = vx * dx + vy * dy + vz * dz, e2d2 = ext * ext * d2;
  if (s < 0 && s * s > e2d2) return false;
  if (s > d2 && (s - d2) * (s - d2) > e2d2) return false;
  return true;
}

// k(g) = (z, x+y, min(x,y), x, original index), compared lexicographically - SURVEY 8(c) O5.
struct Key5 { i64 v[5]; };
inline Key5 key5(const Grain& g) {
  Key5 k; k.v[0] = g.z; k.v[1] = (i64)g.x + g.y; k.v[2] = std::min(g.x, g.y); k.v[3] = g.x; k.v[4] = g.row;
  return k;
}
inline int cmp5(const Key5& a, const Key5& b) {
  for (int i = 0; i < 5; ++i) { if (a.v[i] < b.v[i]) return -1; if (a.v[i] > b.v[i]) return 1; }
  return 0;
}

struct Cand {
  int32_t a, b;          // local handles (positions in G) of the two seed grains
  int32_t n_tube;
  i64 d2;
  Key5 kmin, kmax;
  size_t mem_off;        // into the view's flat in-tube list (n_tube entries)
  int32_t n_members;
};

// C1 "better than" C2 - SURVEY 8(c) O5: larger n_tube; larger D2; smaller kmin; smaller kmax.
inline bool better(const Cand& c1, const Cand& c2) {
  if (c1.n_tube != c2.n_tube) return c1.n_tube > c2.n_tube;
  if (c1.d2 != c2.d2) return c1.d2 > c2.d2;
  int c = cmp5(c1.kmin, c2.kmin);
  if (c) return c < 0;
  return cmp5(c1.kmax, c2.kmax) < 0;
}

struct ViewResult {
  std::vector<emo_track> tracks;     // member_off relative to this view's member list
  std::vector<int32_t> members;      // rows
  std::vector<emo_fit> fits;
  std::vector<int32_t> seed_dump;    // 4 ints per seed: view, row_a, row_b, n_tube
  i64 cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};  // seeds, tube tests, candidates, tracks, members, status, pair tests, -
};

// O6 - SURVEY 8(c) O6 (BASELINE.json north_star; not in the paper).
emo_fit fit_members(const std::vector<Grain>& G, const int32_t* mem, int32_t n) {
  emo_fit f; std::memset(&f, 0, sizeof f);
  i64 mn[3], mx[3];
  for (int i = 0; i < n; ++i) {
    const Grain& g = G[mem[i]];
    i64 c[3] = {g.x, g.y, g.z};
    for (int a = 0; a < 3; ++a) {
      if (i == 0 || c[a] < mn[a]) mn[a] = c[a];
      if (i == 0 || c[a] > mx[a]) mx[a] = c[a];
    }
  }
  i64 ex = mx[0] - mn[0], ey = mx[1] - mn[1], ez = mx[2] - mn[2];
  int u, v, w;
  if (ez >= ex && ez >= ey) { u = 2; v = 0; w = 1; }
  else if (ex >= ey)        { u = 0; v = 1; w = 2; }
  else                      { u = 1; v = 0; w = 2; }
  i64 Su = 0, Sv = 0, Sw = 0, Suu = 0, Suv = 0, Suw = 0;
  for (int i = 0; i < n; ++i) {
    const Grain& g = G[mem[i]];
    i64 c[3] = {g.x, g.y, g.z};
    Su += c[u]; Sv += c[v]; Sw += c[w];
    Suu += c[u] * c[u]; Suv += c[u] * c[v]; Suw += c[u] * c[w];
  }
  i64 N = n, den = N * Suu - Su * Su;
  f.axis = u; f.n = n; f.u_min = (int32_t)mn[u]; f.u_max = (int32_t)mx[u];
  if (den == 0) {
    f.axis |= 0x100;
    f.slope[0] = 0.0; f.slope[1] = 0.0;
    f.icpt[0] = (double)Sv / (double)N; f.icpt[1] = (double)Sw / (double)N;
  } else {
    f.slope[0] = (double)(N * Suv - Su * Sv) / (double)den;
    f.icpt[0] = ((double)Sv - f.slope[0] * (double)Su) / (double)N;
    f.slope[1] = (double)(N * Suw - Su * Sw) / (double)den;
    f.icpt[1] = ((double)Sw - f.slope[1] * (double)Su) / (double)N;
  }
  return f;
}

// O5b - SURVEY 8(f) NEXT-2 / PAPER.md:144.  Bin of |cos theta| of the fitted line, theta = angle to the z axis
// (the normal of the emulsion layer).  The fitted direction is (1, slope_v, slope_w) along (u, v, w), i.e. proportional
// to the exact integers (den, num_v, num_w) of O6; cos^2 = c_z^2 / (den^2 + num_v^2 + num_w^2) with c_z the z component
// (den for u = z, else num_w: z is the second minor axis of u = x and of u = y).  bin = largest k in 0..7 with
// (k/8)^2 <= cos^2, decided exactly: k^2 S <= 64 c_z^2 in 128-bit integers (|den|, |num| <= 2^60: n < 2^13, |coord| <
// 2^17, so S < 3 * 2^120 and 49 S < 2^128).  den = 0 (all members coincide): no direction, bin -1 = never cut.
int angle_bin(const std::vector<Grain>& G, const int32_t* mem, int32_t n) {
  i64 mn[3], mx[3];
  for (int i = 0; i < n; ++i) {
    const Grain& g = G[mem[i]];
    i64 c[3] = {g.x, g.y, g.z};
    for (int a = 0; a < 3; ++a) {
      if (i == 0 || c[a] < mn[a]) mn[a] = c[a];
      if (i == 0 || c[a] > mx[a]) mx[a] = c[a];
    }
  }
  i64 ex = mx[0] - mn[0], ey = mx[1] - mn[1], ez = mx[2] - mn[2];
  int u, v, w;
  if (ez >= ex && ez >= ey) { u = 2; v = 0; w = 1; }
  else if (ex >= ey)        { u = 0; v = 1; w = 2; }
  else                      { u = 1; v = 0; w = 2; }
  i64 Su = 0, Sv = 0, Sw = 0, Suu = 0, Suv = 0, Suw = 0;
  for (int i = 0; i < n; ++i) {
    const Grain& g = G[mem[i]];
    i64 c[3] = {g.x, g.y, g.z};
    Su += c[u]; Sv += c[v]; Sw += c[w];
    Suu += c[u] * c[u]; Suv += c[u] * c[v]; Suw += c[u] * c[w];
  }
  const i64 N = n, den = N * Suu - Su * Su, nv = N * Suv - Su * Sv, nw = N * Suw - Su * Sw;
  if (den == 0) return -1;
  typedef unsigned __int128 u128;
  auto sq = [](i64 a) { u128 m = (u128)(a < 0 ? -a : a); return m * m; };
  const u128 S = sq(den) + sq(nv) + sq(nw);
  const u128 cz2 = (u == 2) ? sq(den) : sq(nw);
  int bin = 0;
  for (int k = 1; k <= 7; ++k) if ((u128)(k * k) * S <= (u128)64 * cz2) bin = k;
  return bin;
}

void track_view(const emo_params& P, const int32_t* grains, int32_t row0, int32_t n, int32_t view,
                int mode, bool want_dump, ViewResult& R) {
  std::vector<Grain> G(n);
  for (int32_t i = 0; i < n; ++i) {
    const int32_t* p = grains + 4 * (i64)(row0 + i);
    G[i].x = p[0]; G[i].y = p[1]; G[i].z = p[2]; G[i].row = row0 + i;
    // |coord| < 2^17 keeps every product below 2^62
    if (std::abs(G[i].x) >= (1 << 17) || std::abs(G[i].y) >= (1 << 17) || std::abs(G[i].z) >= (1 << 17)) {
      R.cnt[5] = -1; return;
    }
  }
  const i64 smin2 = (i64)P.sep_min_q * P.sep_min_q, smax2 = (i64)P.sep_max_q * P.sep_max_q;
  const i64 r2 = P.tube_r2_q;
  i64 R_up = 0; while (R_up * R_up < r2) ++R_up;          // integer radius >= sqrt(r2)

  Grid grid(P);
  std::vector<int32_t> order, cell_start;
  i64 bbmin[3] = {0, 0, 0}, bbmax[3] = {0, 0, 0};
  if (mode == 1) {
    // the "hash table": keep the view's grains in cell order, so that "the grains in the relevant
    // cells" are contiguous.  From here on a local handle is a position in G;
    // everything that leaves this function is expressed in rows, so the order of G is immaterial.
    bin_view(grid, grains, row0, n, order, cell_start);
    std::vector<Grain> S(n);
    for (int32_t k = 0; k < n; ++k) S[k] = G[order[k]];
    G.swap(S);
    for (int32_t i = 0; i < n; ++i) {
      i64 c[3] = {G[i].x, G[i].y, G[i].z};
      for (int a = 0; a < 3; ++a) {
        if (i == 0 || c[a] < bbmin[a]) bbmin[a] = c[a];
        if (i == 0 || c[a] > bbmax[a]) bbmax[a] = c[a];
      }
    }
  }

  // what the pair loop produces; in the brute mode several threads each fill one of their own and the parts are
  // joined afterwards (every later step is a max / count / sort over a total order, so the order of `cands` is
  // immaterial - and the seed dump is compared as a set)
  struct Part {
    std::vector<Cand> cands;
    std::vector<int32_t> tube;      // flat in-tube lists of the candidates (local indices)
    std::vector<int32_t> cur;
    std::vector<int32_t> seed_dump;
    i64 seeds = 0, tests = 0, pairs = 0;
  };

  // O3 for one seed (a < b local indices): fills `cur` with the grains in the tube.
  auto count_seed = [&](Part& W, int32_t a, int32_t b, i64 d2) {
    std::vector<int32_t>& cur = W.cur;
    const Grain& A = G[a];
    const i64 d[3] = {(i64)G[b].x - A.x, (i64)G[b].y - A.y, (i64)G[b].z - A.z};
    const i64 r2D2 = r2 * d2;
    cur.clear();
    if (mode == 0) {
      for (int32_t p = 0; p < n; ++p) {
        W.tests += 1;
        if (in_tube(A, d[0], d[1], d[2], r2D2, G[p], d2, P.tube_ext_q)) cur.push_back(p);
      }
      return;
    }
    // mode 1: walk the cells the tube can touch, slab by slab along the major axis u.
    // The walk only has to be a SUPERSET of the tube (every visited grain still takes the exact
    // integer test above), so its bounds are computed in double with 1 q of slack: every
    // magnitude here is below 2^31 and a double carries 53 bits, so the rounding error of these
    // few operations is far below the slack.
    int u = 0;
    if (std::llabs(d[1]) > std::llabs(d[u])) u = 1;
    if (std::llabs(d[2]) > std::llabs(d[u])) u = 2;
    const int minor[2] = {(u + 1) % 3, (u + 2) % 3};
    const i64 Ac[3] = {A.x, A.y, A.z};
    const double inv_du = 1.0 / (double)d[u];
    for (i64 s = 0; s < grid.n[u]; ++s) {
      // grains whose cell index along u is s have coordinate in [lo,hi]; the two boundary
      // cells are open-ended because out-of-box grains are clamped into them (reading Q13),
      // so they reach as far as the data do (bounding box of the view).
      i64 lo = (s == 0) ? bbmin[u] : std::max(bbmin[u], s * grid.cs[u]);
      i64 hi = (s == grid.n[u] - 1) ? bbmax[u] : std::min(bbmax[u], (s + 1) * grid.cs[u] - 1);
      if (lo > hi) continue;
      // the foot of such a grain on the line is within R_up of it, so the foot's u-coordinate
      // is in [lo-R, hi+R]; line parameter t (X = A + t d) at those two ends:
      const double t0 = (double)(lo - R_up - Ac[u]) * inv_du, t1 = (double)(hi + R_up - Ac[u]) * inv_du;
      i64 rng[3][2];
      rng[u][0] = s; rng[u][1] = s;
      for (int k = 0; k < 2; ++k) {
        const int m = minor[k];
        // the line's other coordinates are linear in t: extremes at the two ends; the grain is
        // within R_up of its foot in every coordinate.
        const double x0 = (double)Ac[m] + t0 * (double)d[m], x1 = (double)Ac[m] + t1 * (double)d[m];
        const double lo_m = std::min(x0, x1) - (double)R_up - 1.0, hi_m = std::max(x0, x1) + (double)R_up + 1.0;
        rng[m][0] = clampi((i64)std::floor(lo_m * grid.inv_cs[m]), 0, grid.n[m] - 1);
        rng[m][1] = clampi((i64)std::floor(hi_m * grid.inv_cs[m]), 0, grid.n[m] - 1);
      }
      for (i64 cz = rng[2][0]; cz <= rng[2][1]; ++cz)
        for (i64 cy = rng[1][0]; cy <= rng[1][1]; ++cy) {
          // cells cx0..cx1 of one (cy,cz) row are consecutive, and so are their grains
          i64 c0 = rng[0][0] + grid.n[0] * (cy + grid.n[1] * cz), c1 = c0 + (rng[0][1] - rng[0][0]);
          for (int32_t j = cell_start[c0]; j < cell_start[c1 + 1]; ++j) {
            W.tests += 1;
            if (in_tube(A, d[0], d[1], d[2], r2D2, G[j], d2, P.tube_ext_q)) cur.push_back(j);
          }
        }
    }
  };

  // O2 + O3 + O4 for the unordered pair {i,j}, i < j.
  auto try_pair = [&](Part& W, int32_t i, int32_t j) {
    W.pairs += 1;
    i64 dx = (i64)G[j].x - G[i].x, dy = (i64)G[j].y - G[i].y, dz = (i64)G[j].z - G[i].z;
    i64 d2 = dx * dx + dy * dy + dz * dz;
    if (d2 < smin2 || d2 >= smax2) return;                 // reading Q1: smin2 <= D2 < smax2
    W.seeds += 1;
    count_seed(W, i, j, d2);
    int32_t n_tube = (int32_t)W.cur.size();
    if (want_dump) {
      W.seed_dump.push_back(view); W.seed_dump.push_back(std::min(G[i].row, G[j].row));
      W.seed_dump.push_back(std::max(G[i].row, G[j].row)); W.seed_dump.push_back(n_tube);
    }
    if (n_tube < P.min_grains) return;                     // O4 (reading Q6: >=)
    Cand c; c.a = i; c.b = j; c.n_tube = n_tube; c.d2 = d2; c.n_members = 0;
    Key5 ka = key5(G[i]), kb = key5(G[j]);
    if (cmp5(ka, kb) <= 0) { c.kmin = ka; c.kmax = kb; } else { c.kmin = kb; c.kmax = ka; }
    c.mem_off = W.tube.size();
    W.tube.insert(W.tube.end(), W.cur.begin(), W.cur.end());
    W.cands.push_back(c);
  };

  std::vector<Cand> cands;
  std::vector<int32_t> tube;
  auto join = [&](Part& W) {                               // append a part to the view's lists
    for (Cand c : W.cands) { c.mem_off += tube.size(); cands.push_back(c); }
    tube.insert(tube.end(), W.tube.begin(), W.tube.end());
    R.seed_dump.insert(R.seed_dump.end(), W.seed_dump.begin(), W.seed_dump.end());
    R.cnt[0] += W.seeds; R.cnt[1] += W.tests; R.cnt[6] += W.pairs;
  };

  if (mode == 0) {
    // every pair against every grain.  When this view is the only one in flight (emo_track_views runs a single view
    // without an outer team) the rows of the pair loop are shared among the threads; each thread fills its own Part.
    int nt = 1;
#ifdef _OPENMP
    nt = omp_in_parallel() ? 1 : omp_get_max_threads();
#endif
    std::vector<Part> parts(nt);
#pragma omp parallel num_threads(nt) if (nt > 1)
    {
      int me = 0;
#ifdef _OPENMP
      me = omp_get_thread_num();
#endif
      Part& W = parts[me];
#pragma omp for schedule(dynamic, 8)
      for (int32_t i = 0; i < n; ++i)
        for (int32_t j = i + 1; j < n; ++j) try_pair(W, i, j);
    }
    for (Part& W : parts) join(W);
  } else {
    Part W;
    // PAPER.md:80 Fig. 4(a): "for each grain ... looping for grains within a given distance",
    // restricted to the cells that can hold them.  Cell index is monotone in
    // the coordinate (also under clamping), so |delta coord| < sep_max bounds the index range.
    for (int32_t i = 0; i < n; ++i) {
      i64 lo[3], hi[3];
      const i64 c[3] = {G[i].x, G[i].y, G[i].z};
      for (int a = 0; a < 3; ++a) { lo[a] = grid.ci(a, c[a] - P.sep_max_q); hi[a] = grid.ci(a, c[a] + P.sep_max_q); }
      for (i64 cz = lo[2]; cz <= hi[2]; ++cz)
        for (i64 cy = lo[1]; cy <= hi[1]; ++cy)
          for (i64 cx = lo[0]; cx <= hi[0]; ++cx) {
            i64 cc = cx + grid.n[0] * (cy + grid.n[1] * cz);
            for (int32_t j = cell_start[cc]; j < cell_start[cc + 1]; ++j)
              if (j > i) try_pair(W, i, j);                // reading Q2: each unordered pair once
          }
    }
    join(W);
  }
  R.cnt[2] = (i64)cands.size();

  // O5: every grain goes to the best candidate whose tube holds it; one round.
  std::vector<int32_t> owner(n, -1);
  for (size_t ci = 0; ci < cands.size(); ++ci) {
    const Cand& c = cands[ci];
    for (int32_t k = 0; k < c.n_tube; ++k) {
      int32_t g = tube[c.mem_off + k];
      if (owner[g] < 0 || better(c, cands[owner[g]])) owner[g] = (int32_t)ci;
    }
  }
  for (int32_t g = 0; g < n; ++g) if (owner[g] >= 0) cands[owner[g]].n_members += 1;
  std::vector<int32_t> trk;
  for (size_t ci = 0; ci < cands.size(); ++ci)
    if (cands[ci].n_members >= P.min_grains) trk.push_back((int32_t)ci);   // threshold again
  // O5b (NEXT-2): angle-dependent cut on the number of grains; a track that fails it is dropped and its
  // grains stay unassigned (as for the re-threshold, reading Q8).
  {
    bool any = false;
    for (int k = 0; k < 8; ++k) any = any || P.angle_min_grains[k] > 0;
    if (any) {
      std::vector<int32_t> kept;
      for (int32_t ci : trk) {
        std::vector<int32_t> mem;
        for (int32_t g = 0; g < n; ++g) if (owner[g] == ci) mem.push_back(g);
        const int bin = angle_bin(G, mem.data(), (int32_t)mem.size());
        if (bin >= 0 && cands[ci].n_members < P.angle_min_grains[bin]) continue;
        kept.push_back(ci);
      }
      trk.swap(kept);
    }
  }
  // O7: best first.
  std::sort(trk.begin(), trk.end(), [&](int32_t x, int32_t y) { return better(cands[x], cands[y]); });

  for (size_t t = 0; t < trk.size(); ++t) {
    const Cand& c = cands[trk[t]];
    emo_track T; std::memset(&T, 0, sizeof T);
    T.view = view; T.seed_a = std::min(G[c.a].row, G[c.b].row); T.seed_b = std::max(G[c.a].row, G[c.b].row);
    T.n_tube = c.n_tube; T.n_members = c.n_members;
    T.member_off = (int32_t)R.members.size(); T.seed_d2 = (int32_t)c.d2;
    std::vector<int32_t> mem;                               // local handles, by ascending row
    for (int32_t g = 0; g < n; ++g) if (owner[g] == trk[t]) mem.push_back(g);
    std::sort(mem.begin(), mem.end(), [&](int32_t x, int32_t y) { return G[x].row < G[y].row; });
    if (c.n_members >= (1 << 13)) { R.cnt[5] = -1; return; }   // n < 2^13
    R.fits.push_back(fit_members(G, mem.data(), (int32_t)mem.size()));
    for (int32_t g : mem) R.members.push_back(G[g].row);
    R.tracks.push_back(T);
  }
  R.cnt[3] = (i64)R.tracks.size();
  R.cnt[4] = (i64)R.members.size();
}

struct Result {
  std::vector<emo_track> tracks;
  std::vector<int32_t> track_off;
  std::vector<int32_t> members;
  std::vector<emo_fit> fits;
  std::vector<int32_t> seed_dump;
  i64 cnt[8];
};

bool params_ok(const emo_params* p) {
  if (!p || p->struct_size != (int32_t)sizeof(emo_params)) return false;
  for (int i = 0; i < 3; ++i)
    if (p->view_size_q[i] <= 0 || p->view_size_q[i] > 65536 || p->cell_size_q[i] <= 0) return false;
  if (p->sep_min_q < 1 || p->sep_max_q <= p->sep_min_q || p->sep_max_q > 2048) return false;
  if (p->tube_r2_q < 0 || p->tube_r2_q >= (1 << 20)) return false;
  if (p->tube_ext_q < -1 || p->tube_ext_q > 65536) return false;   // -1 = whole line; >= 0 = bounded tube (NEXT-1)
  if (p->min_grains < 2) return false;
  for (int k = 0; k < 8; ++k) if (p->angle_min_grains[k] < 0) return false;
  return true;
}

}  // namespace

extern "C" {

// O1 over a batch.  sorted[N][4] = x,y,z,row ordered by (view, cell, row); cell_start[n_views*n_cells+1].
int emo_bin(const emo_params* p, const int32_t* grains, const int32_t* view_off, int32_t n_views,
            int32_t* sorted, int32_t* cell_start) {
  if (!params_ok(p)) return -1;
  Grid g(*p);
  const i64 nc = g.n_cells();
  for (int32_t v = 0; v < n_views; ++v) {
    std::vector<int32_t> order, cs;
    int32_t row0 = view_off[v], n = view_off[v + 1] - view_off[v];
    bin_view(g, grains, row0, n, order, cs);
    for (int32_t i = 0; i < n; ++i) {
      const int32_t* s = grains + 4 * (i64)(row0 + order[i]);
      int32_t* d = sorted + 4 * (i64)(row0 + i);
      d[0] = s[0]; d[1] = s[1]; d[2] = s[2]; d[3] = row0 + order[i];
    }
    for (i64 c = 0; c < nc; ++c) cell_start[v * nc + c] = row0 + cs[c];
  }
  cell_start[(i64)n_views * nc] = view_off[n_views];
  return 0;
}

int64_t emo_n_cells(const emo_params* p) { return params_ok(p) ? Grid(*p).n_cells() : -1; }
void emo_grid_dims(const emo_params* p, int64_t* out3) { Grid g(*p); out3[0] = g.n[0]; out3[1] = g.n[1]; out3[2] = g.n[2]; }

// O2..O7 over a batch of independent views (one OpenMP task per view: the paper's own
// "each thread is responsible for processing a view").
void* emo_track_views(const emo_params* p, const int32_t* grains, const int32_t* view_off, int32_t n_views,
                      int32_t mode, int32_t n_threads, int32_t want_seed_dump) {
  if (!params_ok(p) || n_views < 0) return nullptr;
  std::vector<ViewResult> vr(n_views);
#ifdef _OPENMP
  omp_set_num_threads(n_threads > 0 ? n_threads : omp_get_num_procs());   // 0 = all cores (the setting persists between calls)
#endif
  // (a single view runs without an outer team, so that the brute mode can share its pair loop among the threads)
#pragma omp parallel for schedule(dynamic, 1) if (n_views > 1)
  for (int32_t v = 0; v < n_views; ++v)
    track_view(*p, grains, view_off[v], view_off[v + 1] - view_off[v], v, mode, want_seed_dump != 0, vr[v]);
  Result* R = new Result();
  std::memset(R->cnt, 0, sizeof R->cnt);
  R->track_off.push_back(0);
  for (int32_t v = 0; v < n_views; ++v) {
    int32_t moff = (int32_t)R->members.size();
    for (emo_track t : vr[v].tracks) { t.member_off += moff; R->tracks.push_back(t); }
    R->members.insert(R->members.end(), vr[v].members.begin(), vr[v].members.end());
    R->fits.insert(R->fits.end(), vr[v].fits.begin(), vr[v].fits.end());
    R->seed_dump.insert(R->seed_dump.end(), vr[v].seed_dump.begin(), vr[v].seed_dump.end());
    R->track_off.push_back((int32_t)R->tracks.size());
    for (int k = 0; k < 8; ++k) if (k != 5) R->cnt[k] += vr[v].cnt[k];
    if (vr[v].cnt[5] != 0) R->cnt[5] = vr[v].cnt[5];
  }
  return R;
}

int64_t emo_n_tracks(void* h) { return (int64_t)((Result*)h)->tracks.size(); }
int64_t emo_n_members(void* h) { return (int64_t)((Result*)h)->members.size(); }
int64_t emo_n_seed_dump(void* h) { return (int64_t)((Result*)h)->seed_dump.size() / 4; }
void emo_get(void* h, emo_track* tracks, int32_t* track_off, int32_t* members, emo_fit* fits, int64_t* cnt8) {
  Result* R = (Result*)h;
  if (tracks && !R->tracks.empty()) std::memcpy(tracks, R->tracks.data(), R->tracks.size() * sizeof(emo_track));
  if (track_off) std::memcpy(track_off, R->track_off.data(), R->track_off.size() * sizeof(int32_t));
  if (members && !R->members.empty()) std::memcpy(members, R->members.data(), R->members.size() * sizeof(int32_t));
  if (fits && !R->fits.empty()) std::memcpy(fits, R->fits.data(), R->fits.size() * sizeof(emo_fit));
  if (cnt8) std::memcpy(cnt8, R->cnt, sizeof R->cnt);
}
void emo_get_seed_dump(void* h, int32_t* out) {
  Result* R = (Result*)h;
  if (!R->seed_dump.empty()) std::memcpy(out, R->seed_dump.data(), R->seed_dump.size() * sizeof(int32_t));
}
void emo_free(void* h) { delete (Result*)h; }

// O6 alone, on caller-given member lists (rows of `grains`), for the fit pins.
int emo_fit_tracks(const int32_t* grains, const int32_t* members, const int32_t* member_off, int32_t n_tracks,
                   emo_fit* fits) {
  for (int32_t t = 0; t < n_tracks; ++t) {
    int32_t n = member_off[t + 1] - member_off[t];
    if (n < 1 || n >= (1 << 13)) return -1;
    std::vector<Grain> G(n); std::vector<int32_t> idx(n);
    for (int32_t i = 0; i < n; ++i) {
      const int32_t* p = grains + 4 * (i64)members[member_off[t] + i];
      G[i].x = p[0]; G[i].y = p[1]; G[i].z = p[2]; G[i].row = members[member_off[t] + i]; idx[i] = i;
    }
    fits[t] = fit_members(G, idx.data(), n);
  }
  return 0;
}

int emo_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
