// emu_find.cu - A2..A5 + A7: seeds, tube vote, threshold, exclusive association, threshold, order.
// (P:72 and Fig. 4; readings Q1-Q8, Q15 in DESIGN.md section 3.)
//
// FRAMES.  A seed line is walked in the frame whose first axis u is the line's dominant axis (emu_dev.cuh):
// rows of cells run along u, so a line with |dv|, |dw| <= |du| stays long in every row it enters and enters
// few of them.  Every view is therefore binned three times (frame 0 is the caller's A1 output, frames 1
// and 2 are binned here from it), the seeds of a view are split into three lists by dominant axis, and
// the brick kernels see three "virtual views" per view.  Grain-indexed state (priority keys, owners) is
// indexed by ROW (the caller's grain index), which every frame carries in w.
//
// Views are processed in chunks sized by the workspace.  Per chunk:
//   k_seed_pairs<0>   every grain A: number of seeds {A,B}, B behind A in cell order, per frame  (A2)
//   k_view_scan, k_chunk_offsets   per-grain / per-(view, frame) seed offsets
//   k_seed_pairs<1>   the seeds themselves: packed geometry (A, d) in frame coordinates, oriented so that
//                     du > 0, + the two sorted positions (frame 0)
//   k_plan            cut every (view, frame) into BRICKS (a tile of cell columns x a run of w layers) that
//                     fit shared memory
//   k_brick<kVote>    persistent blocks: stage one brick's grains + cell table in shared memory, stream
//                     all seeds of the (view, frame) past it; every lane walks its own seed's tube through
//                     the brick (uniform-grid ray traversal), counts with the exact test (float with an exact
//                     integer fallback inside its error band) and writes the grains it finds into the seed's
//                     hit record (A3)
//   k_cands<0/1>      n_tube >= min_grains -> candidate list grouped by (view, frame)            (A4)
//   k_assoc_hits      the candidates' hit records: atomicMax of a packed priority into each member grain (A5)
//   k_brick<kAssoc>   the same by a second walk, for the few candidates whose record overflowed
//   (both k_brick kernels also exist with kBounded = true for the bounded tube, tube_ext_q >= 0)
//   k_tie_detect, k_assoc_generic<1>   exact settlement of priority ties by (kmin, kmax)
//   k_wins, k_select  members won per candidate, threshold again
//   k_track_scan / k_track_emit / k_member_scan / k_member_scatter / k_member_sort: ordered output (A7)
// If a view cannot be cut into bricks (pathological density) the chunk falls back to the generic
// kernels k_vote_generic / k_assoc_generic<0> that walk the cells in global memory.
// Everything is a max / min / sum over a total order, so the result does not depend on the order in
// which threads run (reading Q7: "one-shot, order-free").
#include <math.h>
#include <stdlib.h>

#include "emu_dev.cuh"
#include "emu_host.h"

namespace {

constexpr int kVoteThreads = 128;                 // generic walkers and the pair kernels
constexpr int kCiBits = 29;                       // candidate index inside a chunk
constexpr unsigned kCiMask = (1u << kCiBits) - 1u;
constexpr unsigned kNone = 0xffffffffu;
constexpr int kMaxTube = 8191;                    // n_tube field of the packed priority: 13 bits

#ifndef EMU_BRICK_THREADS
#define EMU_BRICK_THREADS 1024
#endif
#ifndef EMU_CHUNK_GIB
#define EMU_CHUNK_GIB 96
#endif
#ifndef EMU_ITEMS_PER_SM
#define EMU_ITEMS_PER_SM 12
#endif
#ifndef EMU_BODY_REPS
#define EMU_BODY_REPS 2
#endif
#ifndef EMU_REFILL
#define EMU_REFILL 8
#endif
#ifndef EMU_REFILL_STOP
#define EMU_REFILL_STOP 4
#endif
constexpr int kBrickThreads = EMU_BRICK_THREADS;  // one persistent block per SM
constexpr int kPoolBytes = 222 * 1024;            // dynamic shared memory of a brick: grains | row table | cell table
#ifndef EMU_GRAB
#define EMU_GRAB 128
#endif
constexpr int kGrab = EMU_GRAB;                        // seeds a warp takes from the block's stream at a time
constexpr int kTieBits = 1 << 16;                 // bitmap of tied priorities

// shared-memory layout of a brick: n grains of 4 B, then one table row per row of cells: the brick slot
// of the first grain of each of its w cells, the end of the row, and (last two entries, as one 32-bit
// word) the sorted position of the row's first grain minus its slot.  Row stride in 16-bit entries:
__host__ __device__ inline int brick_row_stride(int w) { return (w + 4) & ~1; }
__host__ __device__ inline long long brick_bytes(long long n, long long rows, long long w) {
  return 4 * n + 2 * rows * (long long)brick_row_stride((int)w);
}

struct Cand {            // 16 B
  int a, b;              // sorted positions of the seed grains, a < b
  int n_tube_view;       // n_tube | (view - v0) << 16
  int d2;
};

struct Brick {           // 48 B: cells [cx0..cx1] x [cy0..cy1] x [cz0..cz1] (frame coordinates u, v, w) of one
  int view, cx0, cx1, cy0, cy1, cz0, cz1, n;   // (view, frame), n grains
  int frame;
  int ord;               // ordinal of the brick inside its (view, frame): selects the hit record of a seed
  int base;              // first entry of the brick in slot_row (brick slot -> row of the grain)
  int pad;
};

// Hit records.  While it counts, the voting pass also writes down WHICH grains it found: every (seed, brick)
// pair owns a record of kRecSlots 16-bit brick slots, and the 64-bit counter of the seed holds one 16-bit
// field per brick ordinal.  The association pass (k_assoc_hits) then reads the records of the candidates
// instead of walking their tubes again; a candidate with more than kRecSlots grains in one brick, or a
// (view, frame) cut into more than kRecBricks bricks, falls back to the walk (k_brick<kAssoc>).
constexpr int kRecBricks = 4;
constexpr int kRecSlots = 16;

struct Tiling { int tx, ty, w, h; };   // tiles per (view, frame) in u and v, tile width / height in cells
struct Tilings { Tiling t[3]; };

struct FramePtrs {       // the three binnings of the batch (frame 0 = the caller's arrays)
  const int4* sorted[3];
  const int* cell_start[3];
};

struct FindCtl {         // device scalars of one chunk
  unsigned cand_count;   // candidates of the chunk
  unsigned tie;          // 1 if some grain sees two top candidates with equal (n_tube, D2)
  unsigned seed_count;   // seeds of the chunk
  unsigned n_bricks;
  unsigned generic;      // 1: the brick plan failed, the generic kernels do the chunk
  unsigned skip;         // 1: capacity overflow, nothing more is done for the chunk
  unsigned work[2];      // work-item counters of the two brick passes
  unsigned slot_total;   // entries of slot_row handed out to bricks
  unsigned norecord;     // 1: a (view, frame) has more than kRecBricks bricks: no hit records, every candidate is walked
  unsigned ovf_count;    // candidates of the chunk that have to be walked (record overflow)
  unsigned prep_count;   // (seed, brick) records of the chunk (k_prep)
};

__device__ __forceinline__ unsigned long long cand_k1(int n_tube, int d2) {
  return ((unsigned long long)min(n_tube, kMaxTube) << 22) | (unsigned long long)(unsigned)d2;
}

// n_tube of a seed from its 64-bit counter: four 16-bit fields (one per brick ordinal) when the voting pass
// kept hit records, else one plain count.  A field holds one visit's count (<= 0xffff, clamped: such a seed
// is out of range anyway, EMU_ST_RANGE).
__device__ __forceinline__ unsigned tube_total(unsigned long long v, bool fields) {
  if (!fields) return (unsigned)min(v, 0xffffffffull);
  return (unsigned)(v & 0xffffu) + (unsigned)((v >> 16) & 0xffffu) + (unsigned)((v >> 32) & 0xffffu) + (unsigned)(v >> 48);
}
__device__ __forceinline__ bool tube_overflows(unsigned long long v) {   // some brick holds more grains than a record
  return (unsigned)(v & 0xffffu) > (unsigned)kRecSlots || (unsigned)((v >> 16) & 0xffffu) > (unsigned)kRecSlots ||
         (unsigned)((v >> 32) & 0xffffu) > (unsigned)kRecSlots || (unsigned)(v >> 48) > (unsigned)kRecSlots;
}

// k(g) = (z, x+y, min(x,y), x, row), lexicographic
__device__ __forceinline__ int cmp_k(const int4& p, const int4& q) {
  if (p.z != q.z) return p.z < q.z ? -1 : 1;
  int sp = p.x + p.y, sq = q.x + q.y;
  if (sp != sq) return sp < sq ? -1 : 1;
  int mp = min(p.x, p.y), mq = min(q.x, q.y);
  if (mp != mq) return mp < mq ? -1 : 1;
  if (p.x != q.x) return p.x < q.x ? -1 : 1;
  if (p.w != q.w) return p.w < q.w ? -1 : 1;
  return 0;
}

// (kmin, kmax) of candidate c smaller than that of candidate e?  (the last two keys of the order)
__device__ bool cand_kless(const int4* __restrict__ sorted, const Cand& c, const Cand& e) {
  int4 ca = sorted[c.a], cb = sorted[c.b], ea = sorted[e.a], eb = sorted[e.b];
  if (cmp_k(ca, cb) > 0) { int4 t = ca; ca = cb; cb = t; }
  if (cmp_k(ea, eb) > 0) { int4 t = ea; ea = eb; eb = t; }
  int r = cmp_k(ca, ea);
  if (r) return r < 0;
  return cmp_k(cb, eb) < 0;
}

// full order of SURVEY 8(c) O5: larger n_tube, larger D2, smaller kmin, smaller kmax
__device__ bool cand_better(const int4* __restrict__ sorted, const Cand& c, const Cand& e) {
  int nc = c.n_tube_view & 0xffff, ne = e.n_tube_view & 0xffff;
  if (nc != ne) return nc > ne;
  if (c.d2 != e.d2) return c.d2 > e.d2;
  return cand_kless(sorted, c, e);
}

// Packed seed geometry, 16 B: the line A + t*d and (for candidates) its n_tube.  Only views whose grains
// all lie inside the box take the brick path (k_plan), so A fits 16 bits per axis; |d| < 2^11.
//   x = Ax | Ay << 16      y = Az | n_tube << 16 (13 bits)
//   z = (dx + 2048) | (dy + 2048) << 16      w = dz + 2048
__device__ __forceinline__ int4 geo_pack(int ax, int ay, int az, int dx, int dy, int dz) {
  int4 g;
  g.x = (ax & 0xffff) | (ay << 16); g.y = az & 0xffff;
  g.z = ((dx + 2048) & 0xffff) | ((dy + 2048) << 16); g.w = (dz + 2048) & 0xffff;
  return g;
}
__device__ __forceinline__ void geo_d(const int4& g, int& dx, int& dy, int& dz) {
  dx = (g.z & 0xffff) - 2048; dy = (int)((unsigned)g.z >> 16) - 2048; dz = (g.w & 0xffff) - 2048;
}
// 16 bits of a word as a float WITHOUT a conversion instruction: the bytes are dropped into the mantissa
// of 2^23, so the result is 2^23 + value exactly ("magic" float).  sel picks the bytes (PRMT).
constexpr unsigned kMagic = 0x4B000000u;           // 2^23
constexpr float kMagicF = 8388608.0f;
__device__ __forceinline__ float magic_lo16(unsigned w) { return __uint_as_float(__byte_perm(w, kMagic, 0x7410)); }
__device__ __forceinline__ float magic_hi16(unsigned w) { return __uint_as_float(__byte_perm(w, kMagic, 0x7432)); }
__device__ __forceinline__ float magic_b2(unsigned w) { return __uint_as_float(__byte_perm(w, kMagic, 0x7442)); }
__device__ __forceinline__ float magic_b3(unsigned w) { return __uint_as_float(__byte_perm(w, kMagic, 0x7443)); }
// round-to-nearest float -> int and small int -> float through the 1.5 * 2^23 trick (|value| < 2^22)
__device__ __forceinline__ int rn_int(float y) { return __float_as_int(__fadd_rn(y, 12582912.0f)) - 0x4B400000; }
__device__ __forceinline__ float int_f(int i) { return __fadd_rn(__int_as_float(i + 0x4B400000), -12582912.0f); }
// round a float to the nearest integer, staying in float (|value| < 2^22)
__device__ __forceinline__ float rn_flt(float y) { return __fadd_rn(__fadd_rn(y, 12582912.0f), -12582912.0f); }
// a float that holds a small non-negative integer -> that integer
__device__ __forceinline__ int __float2int_rn_magic(float y) { return __float_as_int(__fadd_rn(y, 12582912.0f)) - 0x4B400000; }

// ---------------------------------------------------------------------------------------------
// per-view bounding boxes
__global__ void __launch_bounds__(256)
k_bbox_init(EmuBox* __restrict__ bb, int n_views) {
  int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v < n_views) {
    for (int a = 0; a < 3; ++a) { bb[v].lo[a] = 0x7fffffff; bb[v].hi[a] = (int)0x80000000; }
  }
}

__global__ void __launch_bounds__(256)
k_bbox(const int4* __restrict__ sorted, const int* __restrict__ view_off, int n_views, int n_grains,
       EmuBox* __restrict__ bb) {
  const int stride = gridDim.x * blockDim.x;
  const int lane = threadIdx.x & 31;
  for (int i0 = blockIdx.x * blockDim.x + (threadIdx.x & ~31); i0 < n_grains; i0 += stride) {
    const int i = i0 + lane;
    const bool on = i < n_grains;
    int4 g = on ? __ldg(sorted + i) : make_int4(0, 0, 0, 0);
    int v = on ? emu_find_view(view_off, 0, n_views, i) : -1;
    // 32 consecutive grains nearly always share a view: reduce in the warp, one set of atomics
    const int v_first = __shfl_sync(EMU_FULL, v, 0);
    const bool uniform = __all_sync(EMU_FULL, v == v_first || !on);
    if (uniform) {
      int lo[3] = {on ? g.x : 0x7fffffff, on ? g.y : 0x7fffffff, on ? g.z : 0x7fffffff};
      int hi[3] = {on ? g.x : (int)0x80000000, on ? g.y : (int)0x80000000, on ? g.z : (int)0x80000000};
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        lo[a] = __reduce_min_sync(EMU_FULL, lo[a]);
        hi[a] = __reduce_max_sync(EMU_FULL, hi[a]);
      }
      if (lane == 0) {
#pragma unroll
        for (int a = 0; a < 3; ++a) { atomicMin(&bb[v_first].lo[a], lo[a]); atomicMax(&bb[v_first].hi[a], hi[a]); }
      }
    } else if (on) {
      atomicMin(&bb[v].lo[0], g.x); atomicMax(&bb[v].hi[0], g.x);
      atomicMin(&bb[v].lo[1], g.y); atomicMax(&bb[v].hi[1], g.y);
      atomicMin(&bb[v].lo[2], g.z); atomicMax(&bb[v].hi[2], g.z);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// A2.  One warp per grain A.  The rows of cells (cy, cz) within sep_max of A are dealt to the lanes; a lane
// runs along its row and tests the partners B BEHIND A in sorted order (each unordered pair once, reading
// Q2) against the separation window (reading Q1).  A seed belongs to the frame of its dominant axis
// (largest |d| component, the lowest axis on a tie).
//   kFill = 0: seed_off[f * plane + a] = number of seeds of A in frame f
//   kFill = 1: the seeds are written at view_seed_off[(v - v0) * 3 + f] + seed_off[f * plane + a] + slot
//              (seed_off now holds the exclusive prefix inside the (view, frame)); the slot inside A's
//              group comes from a warp-private counter, so the order inside a group is arbitrary - nothing
//              downstream depends on the order of the seeds (every reduction is over a total order).
constexpr int kPairWarps = kVoteThreads / 32;

__device__ __forceinline__ int dominant_axis(int dx, int dy, int dz) {
  const int ax = abs(dx), ay = abs(dy), az = abs(dz);
  return (ax >= ay && ax >= az) ? 0 : (ay >= az ? 1 : 2);
}

template <int kFill>
__global__ void __launch_bounds__(kVoteThreads)
k_seed_pairs(EmuDev P, const int4* __restrict__ sorted, const int* __restrict__ cell_start,
             const int* __restrict__ view_off, int v0, int v1, unsigned* __restrict__ seed_off, size_t plane,
             const unsigned* __restrict__ view_seed_off, const FindCtl* __restrict__ ctl,
             int4* __restrict__ geo, int2* __restrict__ ab, unsigned long long* __restrict__ counts) {
  __shared__ unsigned cur_s[kPairWarps][4];
  if (kFill && ctl->skip) return;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int nwarps = gridDim.x * kPairWarps;
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  unsigned long long n_pairs = 0;
  for (int a = g0 + blockIdx.x * kPairWarps + wib; a < g1; a += nwarps) {
    const int v = emu_find_view(view_off, v0, v1, a);
    const int4 A = __ldg(sorted + a);
    const int vbase = v * P.ncell;
    const int cxa = emu_cell_axis(A.x - P.sep_max, P.cs[0], P.inv_cs[0], P.n[0]);
    const int cxb = emu_cell_axis(A.x + P.sep_max, P.cs[0], P.inv_cs[0], P.n[0]);
    const int cya = emu_cell_axis(A.y - P.sep_max, P.cs[1], P.inv_cs[1], P.n[1]);
    const int cyb = emu_cell_axis(A.y + P.sep_max, P.cs[1], P.inv_cs[1], P.n[1]);
    const int czA = emu_cell_axis(A.z, P.cs[2], P.inv_cs[2], P.n[2]);   // partners behind A: cell >= cell(A)
    const int czb = emu_cell_axis(A.z + P.sep_max, P.cs[2], P.inv_cs[2], P.n[2]);
    const int ny = cyb - cya + 1, n_rows = ny * (czb - czA + 1);
    const float inv_ny = 1.0f / (float)ny;
    // the rows of A's own layer that lie before A's row hold only grains before A in sorted order: not dealt out
    // (66 rows -> 61 on the bench grid: two rounds of 32 lanes instead of three)
    const int r_first = emu_cell_axis(A.y, P.cs[1], P.inv_cs[1], P.n[1]) - cya;
    unsigned n[3] = {0u, 0u, 0u};
    unsigned base[3] = {0u, 0u, 0u};
    if (kFill) {
#pragma unroll
      for (int f = 0; f < 3; ++f) base[f] = view_seed_off[(v - v0) * 3 + f] + seed_off[(size_t)f * plane + a];
      if (lane < 3) cur_s[wib][lane] = 0u;
      __syncwarp();
    }
    for (int r = r_first + lane; r < n_rows; r += 32) {
      const int lz = (int)(((float)r + 0.5f) * inv_ny);              // r / ny (small integers: exact)
      const int cz = czA + lz, cy = cya + (r - lz * ny);
      const int rb = vbase + (cz * P.n[1] + cy) * P.n[0];
      // Only the chord of the separation sphere in this row: a grain of row (cy, cz) is at least dy_min, dz_min away
      // from A in y and z (the outer side of a boundary row is open: grains outside the box are clamped into it), so a
      // partner has dx^2 < sep_max^2 - dy_min^2 - dz_min^2.  The box of rows holds about twice the pairs the sphere does.
      const int ylo = cy == 0 ? -0x40000000 : cy * P.cs[1], yhi = cy == P.n[1] - 1 ? 0x40000000 : (cy + 1) * P.cs[1] - 1;
      const int zlo = cz == 0 ? -0x40000000 : cz * P.cs[2], zhi = cz == P.n[2] - 1 ? 0x40000000 : (cz + 1) * P.cs[2] - 1;
      const float dym = (float)max(0, max(ylo - A.y, A.y - yhi)), dzm = (float)max(0, max(zlo - A.z, A.z - zhi));
      const float rx2 = (float)P.sep_max2 - dym * dym - dzm * dzm;     // exact: every term below 2^24
      if (rx2 <= 0.0f) continue;
      const int rx = (int)sqrtf(rx2) + 2;                              // (sqrt within 1 of the truth, one more for the strict <)
      const int cxa_r = emu_cell_axis(A.x - rx, P.cs[0], P.inv_cs[0], P.n[0]);
      const int cxb_r = emu_cell_axis(A.x + rx, P.cs[0], P.inv_cs[0], P.n[0]);
      int s = __ldg(cell_start + rb + cxa_r);
      const int e = __ldg(cell_start + rb + cxb_r + 1);
      s = max(s, a + 1);
      for (int j0 = s; j0 < e; j0 += 4) {
       int4 Bq[4];
#pragma unroll
       for (int q = 0; q < 4; ++q) Bq[q] = (j0 + q < e) ? __ldg(sorted + j0 + q) : make_int4(0, 0, 0, 0);   // four loads in flight
#pragma unroll
       for (int q = 0; q < 4; ++q) {
        const int j = j0 + q;
        if (j >= e) break;
        const int4 B = Bq[q];
        const int dx = B.x - A.x, dy = B.y - A.y, dz = B.z - A.z;
        // |d| can exceed 2^15 for far out-of-box grains: compare in 64 bits
        const long long d2 = (long long)dx * dx + (long long)dy * dy + (long long)dz * dz;
        ++n_pairs;
        if (d2 >= P.sep_min2 && d2 < P.sep_max2) {
          const int f = dominant_axis(dx, dy, dz);
          if (!kFill) {
            n[0] += (f == 0); n[1] += (f == 1); n[2] += (f == 2);
          } else {
            const unsigned idx = (f == 0 ? base[0] : (f == 1 ? base[1] : base[2])) + atomicAdd(&cur_s[wib][f], 1u);
            int4 Af = emu_to_frame(f, A);
            int4 df = emu_to_frame(f, make_int4(dx, dy, dz, 0));
            if (df.x < 0) { Af = emu_to_frame(f, B); df.x = -df.x; df.y = -df.y; df.z = -df.z; }   // du > 0
            geo[idx] = geo_pack(Af.x, Af.y, Af.z, df.x, df.y, df.z);
            ab[idx] = make_int2(a, j);
          }
        }
       }
      }
    }
    if (!kFill) {
#pragma unroll
      for (int f = 0; f < 3; ++f) {
        const unsigned t = __reduce_add_sync(EMU_FULL, n[f]);
        if (lane == 0) seed_off[(size_t)f * plane + a] = t;
      }
    } else {
      __syncwarp();
    }
  }
  if (!kFill) {
    for (int o = 16; o; o >>= 1) n_pairs += __shfl_xor_sync(EMU_FULL, n_pairs, o);
    if (lane == 0) atomicAdd(counts + EMU_CNT_PAIR_TESTS, n_pairs);
  }
}

// per-(view, frame) exclusive scan (in place) of the per-grain seed counts;
// view_tot[(v - v0) * 3 + f] = seeds of the view in frame f
__global__ void __launch_bounds__(1024)
k_view_scan(const int* __restrict__ view_off, int v0, int v1, unsigned* __restrict__ seed_off_all, size_t plane,
            unsigned* __restrict__ view_tot, unsigned long long* __restrict__ counts) {
  __shared__ unsigned warp_sum[32];
  __shared__ unsigned carry_s;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int vf = blockIdx.x; vf < (v1 - v0) * 3; vf += gridDim.x) {
    const int v = v0 + vf / 3;
    unsigned* seed_off = seed_off_all + (size_t)(vf % 3) * plane;
    const int g0 = __ldg(view_off + v), g1 = __ldg(view_off + v + 1);
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int b = g0; b < g1; b += blockDim.x) {
      const int g = b + threadIdx.x;
      unsigned x = (g < g1) ? seed_off[g] : 0u;
      unsigned incl = x;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { unsigned y = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += y; }
      if (lane == 31) warp_sum[wid] = incl;
      __syncthreads();
      if (wid == 0) {
        unsigned w = warp_sum[lane], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { unsigned y = __shfl_up_sync(EMU_FULL, wi, o); if (lane >= o) wi += y; }
        warp_sum[lane] = wi - w;
      }
      __syncthreads();
      const unsigned carry = carry_s;
      const unsigned long long mine64 = (unsigned long long)carry + warp_sum[wid] + incl;   // (a tile of 1 024 grains stays far below 2^32)
      const unsigned mine = (unsigned)mine64;
      if (g < g1) {
        if (mine64 > 0xffffffffull) atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)EMU_ST_SEED_OVERFLOW);  // >= 2^32 seeds in a (view, frame)
        seed_off[g] = mine - x;
      }
      __syncthreads();
      if (threadIdx.x == blockDim.x - 1) carry_s = mine;
      __syncthreads();
    }
    if (threadIdx.x == 0) view_tot[vf] = carry_s;
    __syncthreads();
  }
}

// exclusive scan over the views of a chunk (one block): off[0..nv], total -> *total_out; capacity check
__global__ void __launch_bounds__(1024)
k_chunk_offsets(int nv, const unsigned* __restrict__ tot, unsigned* __restrict__ off, unsigned* __restrict__ total_out,
                unsigned cap, unsigned status_bit, FindCtl* __restrict__ ctl, unsigned long long* __restrict__ counts,
                int count_slot, int need_slot, unsigned need_num, unsigned need_den) {
  __shared__ unsigned long long warp_sum[32];
  __shared__ unsigned long long carry_s;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int b = 0; b < nv; b += blockDim.x) {
    const int v = b + threadIdx.x;
    const unsigned long long x = (v < nv) ? tot[v] : 0ull;
    unsigned long long incl = x;                       // 64-bit throughout: 1 024 entries of up to 2^32 - 1 seeds
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { unsigned long long y = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += y; }
    if (lane == 31) warp_sum[wid] = incl;
    __syncthreads();
    if (wid == 0) {
      unsigned long long w = warp_sum[lane], wi = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { unsigned long long y = __shfl_up_sync(EMU_FULL, wi, o); if (lane >= o) wi += y; }
      warp_sum[lane] = wi - w;
    }
    __syncthreads();
    const unsigned long long carry = carry_s;
    const unsigned long long mine = carry + warp_sum[wid] + incl;
    if (v < nv) off[v] = (unsigned)min(mine - x, 0xffffffffull);
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry_s = mine;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const unsigned long long total = carry_s;
    off[nv] = (unsigned)min(total, 0xffffffffull);
    if (count_slot >= 0) atomicAdd(counts + count_slot, total);
    // what the chunk needed, in units of the seed capacity (a list that is sized as need_den / need_num entries per seed
    // reports the seed capacity that would have held it)
    if (need_slot >= 0) atomicMax(counts + need_slot, (total * need_num + need_den - 1) / need_den);
    if (total > cap) {
      atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)status_bit);
      ctl->skip = 1;
      *total_out = 0;
    } else {
      *total_out = (unsigned)total;
    }
  }
}

// the 64-bit counters of the seeds this chunk has (the count is on the device)
__global__ void __launch_bounds__(256)
k_clear_seed_cnt(const FindCtl* __restrict__ ctl, unsigned long long* __restrict__ seed_cnt) {
  const size_t n = ctl->seed_count;
  ulonglong2* p2 = reinterpret_cast<ulonglong2*>(seed_cnt);
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; 2 * i + 1 < n; i += stride) p2[i] = make_ulonglong2(0ull, 0ull);
  if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) seed_cnt[n - 1] = 0ull;
}

// ---------------------------------------------------------------------------------------------
// Brick plan: one warp per (view, frame).  Every tile (tx, ty) of cell columns is cut into runs of w layers
// whose grains, row table and cell table fit the shared-memory pool; empty bricks are dropped.
// The brick kernels keep a grain in 4 bytes (u in 16 bits, v and w relative to the cell in 8 bits),
// which needs every grain of the view inside the box: a view with out-of-box grains (legal, reading
// Q13), or a grid the format cannot hold, sends the chunk to the generic kernels.
__global__ void __launch_bounds__(128)
k_plan(EmuDev P, Tilings TT, FramePtrs F, const EmuBox* __restrict__ bbox, int v0, int v1,
       Brick* __restrict__ bricks, unsigned brick_cap, int* __restrict__ vf_brick_base, int2* __restrict__ vf_bricks,
       FindCtl* __restrict__ ctl) {
  const int lane = threadIdx.x & 31;
  const int vf = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (vf >= (v1 - v0) * 3 || ctl->skip) return;
  if (lane == 0) vf_bricks[vf] = make_int2(0, 0);
  const int v = v0 + vf / 3, f = vf % 3;
  const Tiling T = TT.t[f];
  const int* __restrict__ cell_start = F.cell_start[f];
  const int nx = P.fr[f].n[0], ny = P.fr[f].n[1], nz = P.fr[f].n[2];
  const int vbase = v * P.fr[f].ncell;
  if (cell_start[vbase + P.fr[f].ncell] == cell_start[vbase]) return;          // empty view: no bricks
  {
    const EmuBox bb = bbox[v];                                               // lab coordinates
    bool in_box = P.packed_ok != 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) in_box = in_box && bb.lo[a] >= 0 && bb.hi[a] < P.n[a] * P.cs[a];
#pragma unroll
    for (int i = 0; i < 3; ++i) {                                            // ... and inside every frame's grid
      const int a = emu_frame_axis(f, i);
      in_box = in_box && bb.hi[a] < P.fr[f].n[i] * P.cs[i];
    }
    if (!in_box) { if (lane == 0) ctl->generic = 1; return; }
  }
  // two sweeps over the same cuts: the first counts the bricks, so that the (view, frame) gets ONE contiguous range of
  // the brick array (k_prep walks it), the second writes them
  unsigned first = 0;
  for (int sweep = 0; sweep < 2; ++sweep) {
    int ord = 0;
    for (int t = 0; t < T.tx * T.ty; ++t) {
      const int cx0 = (t % T.tx) * T.w, cy0 = (t / T.tx) * T.h;
      const int cx1 = min(nx, cx0 + T.w) - 1, cy1 = min(ny, cy0 + T.h) - 1;
      if (cx0 > cx1 || cy0 > cy1) continue;
      const int W = cx1 - cx0 + 1, H = cy1 - cy0 + 1;
      int z_first = 0, acc = 0;
      int batch = 0;                                        // grains of layer (cz & ~31) + lane, 32 layers at a time
      for (int cz = 0; cz <= nz; ++cz) {
        if ((cz & 31) == 0) {
          // the counts of the next 32 layers, one per lane (a layer at a time made every step wait for its own loads:
          // 0.2 ms for the 75 layers of frame 2 when a single view is processed)
          const int mz = cz + lane;
          batch = 0;
          if (mz < nz) {
            if (W == nx) {                                  // full rows: the cells of rows cy0..cy1 are consecutive
              batch = __ldg(cell_start + vbase + (mz * ny + cy1) * nx + nx) - __ldg(cell_start + vbase + (mz * ny + cy0) * nx);
            } else {
              for (int cy = cy0; cy <= cy1; ++cy) {
                const int rb = vbase + (mz * ny + cy) * nx;
                batch += __ldg(cell_start + rb + cx1 + 1) - __ldg(cell_start + rb + cx0);
              }
            }
          }
        }
        int cnt = 0;
        if (cz < nz) {
          cnt = __shfl_sync(EMU_FULL, batch, cz & 31);
          if (brick_bytes(cnt, H, W) > kPoolBytes) { if (lane == 0) ctl->generic = 1; return; }
        }
        const bool flush = (cz == nz) || brick_bytes(acc + cnt, (long long)(cz - z_first + 1) * H, W) > kPoolBytes;
        if (flush) {
          if (acc > 0) {
            if (sweep == 1 && lane == 0) {
              const unsigned slot = first + (unsigned)ord;
              if (slot < brick_cap) {
                Brick b; b.view = v; b.cx0 = cx0; b.cx1 = cx1; b.cy0 = cy0; b.cy1 = cy1; b.cz0 = z_first; b.cz1 = cz - 1; b.n = acc;
                b.frame = f; b.ord = ord; b.base = (int)atomicAdd(&ctl->slot_total, (unsigned)acc); b.pad = 0;
                bricks[slot] = b;
                if (ord < kRecBricks) vf_brick_base[vf * kRecBricks + ord] = b.base;
                else ctl->norecord = 1;
              }
            }
            ++ord;
          }
          z_first = cz; acc = 0;
        }
        acc += cnt;
      }
    }
    if (sweep == 0) {
      if (lane == 0) first = atomicAdd(&ctl->n_bricks, (unsigned)ord);
      first = __shfl_sync(EMU_FULL, first, 0);
      if (lane == 0 && first + (unsigned)ord <= brick_cap) vf_bricks[vf] = make_int2((int)first, ord);
    }
  }
}

__global__ void k_plan_finish(FindCtl* ctl, unsigned brick_cap) {
  if (ctl->n_bricks > brick_cap) ctl->generic = 1;
  if (ctl->generic) ctl->n_bricks = 0;
}

// ---------------------------------------------------------------------------------------------
// Per-brick seed lists.  One thread per seed of a (view, frame): the line is clipped against every brick of the
// (view, frame) - the brick's extent widened by the walk radius, and for the bounded tube the part of the line the
// tube covers - and every HIT leaves a 32-byte record in that brick's list: the packed line, the seed's index, the u
// interval [t0, t1] of the line inside the brick and the first / last w layer it can touch there.  The brick kernel
// then streams its own list: no seed is fetched by a brick it misses (38 % of the visits on the bench), and the clip
// runs here with full warps instead of inside the walk.  kFill = 0 counts (one atomic per warp and brick), a scan over
// the bricks gives the list offsets, kFill = 1 writes.  The order inside a list is arbitrary (nothing depends on it).
// 1 / x for |x| >= 1 (a component of d): one MUFU.RCP, no range handling (relative error 2^-23: the traversal
// bounds only have to be a superset and carry 2 q of slack)
__device__ __forceinline__ float rcp_fast(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

struct PrepRec { int4 geo; unsigned sidx; float t0, t1; unsigned layers; };   // 32 B; layers = first | last << 16
constexpr int kPrepSubMin = 32, kPrepSubMax = 512;   // sub-lists per brick = blocks per (view, frame) of k_prep: more when
                                                     // the chunk holds few views, so that a single view still fills the GPU

// the line of a seed as the clip needs it (computed once per seed, used for every brick of its (view, frame))
struct ClipLine { float ax, ay, az, dx, a, bz, y0, z0, inv_a, inv_b, eu; bool has_y, has_z; };

template <bool kBounded>
__device__ __forceinline__ ClipLine clip_line(const EmuDev& P, const int4& q) {
  ClipLine L;
  L.ax = (float)(q.x & 0xffff); L.ay = (float)((unsigned)q.x >> 16); L.az = (float)(q.y & 0xffff);
  int idx, idy, idz;
  geo_d(q, idx, idy, idz);
  const float dx = (float)idx, dy = (float)idy, dz = (float)idz;
  const float inv_dx = rcp_fast(dx);                                  // du >= 1
  L.dx = dx;
  L.a = dy * inv_dx; L.bz = dz * inv_dx;
  L.y0 = __fmaf_rn(-L.a, L.ax, L.ay); L.z0 = __fmaf_rn(-L.bz, L.ax, L.az);
  L.has_y = dy != 0.f; L.has_z = dz != 0.f;
  L.inv_a = L.has_y ? dx * rcp_fast(dy) : 0.0f;
  L.inv_b = L.has_z ? dx * rcp_fast(dz) : 0.0f;
  // bounded tube: the feet of the grains that can count lie between u(A) - E du/|d| and u(B) + E du/|d| (2 q of slack)
  L.eu = kBounded ? __fmaf_rn((float)P.ext * dx, rsqrtf(__fmaf_rn(dx, dx, __fmaf_rn(dy, dy, dz * dz))) * 1.0001f, 2.0f) : 0.0f;
  return L;
}

template <bool kBounded>
__device__ __forceinline__ bool clip_to_brick(const EmuDev& P, const Brick& B, const ClipLine& L, float& t0, float& t1,
                                              unsigned& layers) {
  const float R = P.Rw;
  const float blo0 = (float)(B.cx0 * P.cs[0]) - R, bhi0 = (float)((B.cx1 + 1) * P.cs[0] - 1) + R;
  const float blo1 = (float)(B.cy0 * P.cs[1]) - R, bhi1 = (float)((B.cy1 + 1) * P.cs[1] - 1) + R;
  const float blo2 = (float)(B.cz0 * P.cs[2]) - R, bhi2 = (float)((B.cz1 + 1) * P.cs[2] - 1) + R;
  t0 = blo0; t1 = bhi0;
  bool hit = true;
  if (L.has_y) { const float p = (blo1 - L.y0) * L.inv_a, r = (bhi1 - L.y0) * L.inv_a; t0 = fmaxf(t0, fminf(p, r)); t1 = fminf(t1, fmaxf(p, r)); }
  else hit = hit && (L.ay >= blo1) && (L.ay <= bhi1);
  if (L.has_z) { const float p = (blo2 - L.z0) * L.inv_b, r = (bhi2 - L.z0) * L.inv_b; t0 = fmaxf(t0, fminf(p, r)); t1 = fminf(t1, fmaxf(p, r)); }
  else hit = hit && (L.az >= blo2) && (L.az <= bhi2);
  if (kBounded) { t0 = fmaxf(t0, L.ax - L.eu); t1 = fminf(t1, L.ax + L.dx + L.eu); }
  if (!(hit && t0 <= t1)) return false;
  const float za = __fmaf_rn(L.bz, t0, L.z0), zb = __fmaf_rn(L.bz, t1, L.z0);
  const int c_lo = max(B.cz0, rn_int(__fmaf_rn(fminf(za, zb), P.inv_cs[2], P.klo[2])));
  const int c_hi = min(B.cz1, rn_int(__fmaf_rn(fmaxf(za, zb), P.inv_cs[2], P.khi[2])));
  if (c_lo > c_hi) return false;
  layers = (unsigned)c_lo | ((unsigned)c_hi << 16);
  return true;
}

template <int kFill, bool kBounded>
__global__ void __launch_bounds__(256)
k_prep(EmuDev P, const FindCtl* __restrict__ ctl, const unsigned* __restrict__ view_seed_off, const int4* __restrict__ geo,
       const Brick* __restrict__ bricks, const int2* __restrict__ vf_bricks, unsigned* __restrict__ brick_cnt,
       const unsigned* __restrict__ brick_off, PrepRec* __restrict__ prec) {
  if (ctl->skip || ctl->generic) return;
  const int vf = blockIdx.y, lane = threadIdx.x & 31;
  const unsigned lo = view_seed_off[vf], hi = view_seed_off[vf + 1];
  const int2 vb = vf_bricks[vf];
  for (unsigned i0 = lo + blockIdx.x * blockDim.x + (threadIdx.x & ~31u); i0 < hi; i0 += gridDim.x * blockDim.x) {
    const unsigned i = i0 + (unsigned)lane;
    const bool on = i < hi;
    const int4 q = on ? __ldg(geo + i) : make_int4(0, 0, 0x08010801, 0x0800);   // (an idle lane: d = (1, 1, 0))
    const ClipLine L = clip_line<kBounded>(P, q);
    for (int k = 0; k < vb.y; ++k) {
      const Brick B = bricks[vb.x + k];
      float t0, t1;
      unsigned layers = 0;
      const bool hit = on && clip_to_brick<kBounded>(P, B, L, t0, t1, layers);
      const unsigned m = __ballot_sync(EMU_FULL, hit);
      if (!m) continue;
      // every brick's list is cut into gridDim.x sub-lists, one per blockIdx.x, each with its own counter: the eight
      // warps of a block are all that ever meet on one address (a single counter per brick cost 0.9 ms per view)
      const unsigned slot = (unsigned)(vb.x + k) * gridDim.x + blockIdx.x;
      unsigned base = 0;
      if (lane == 0) base = atomicAdd(brick_cnt + slot, (unsigned)__popc(m));
      if (!kFill) continue;
      base = __shfl_sync(EMU_FULL, base, 0) + brick_off[slot];
      if (hit) {
        PrepRec r; r.geo = q; r.sidx = i; r.t0 = t0; r.t1 = t1; r.layers = layers;
        const unsigned at = base + (unsigned)__popc(m & ((1u << lane) - 1u));
        reinterpret_cast<int4*>(prec + at)[0] = r.geo;
        reinterpret_cast<int4*>(prec + at)[1] = make_int4((int)r.sidx, __float_as_int(r.t0), __float_as_int(r.t1), (int)r.layers);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// A3 / A5 on shared-memory bricks.
//
// A persistent block takes work items (brick, slice of the seed list of the brick's (view, frame)).  It
// stages the brick in shared memory - every grain in 4 bytes (u | v-in-cell << 16 | w-in-cell << 24) in
// (cw, cv, cu) order, a 16-bit cell table, and per row of cells the sorted position of its first grain - and
// streams the seeds of the slice past it.  Each LANE owns one seed at a time; the loop body is fused:
//   SEED  idle lanes are refilled in batches from the block's seed stream: unpack, clip against the brick
//   ROW   lanes whose run of grains is used up advance: next row of cells (cv) of the current w layer, else
//         the next layer, giving a run [j, e) of consecutive grains of the cells cu0..cu1 the tube can touch
//   TEST  up to two point-line tests of the grains j, j+1; VOTE counts, ASSOC joins the priority maximum
//
// Traversal.  In its frame the line has du > 0 and |dv|, |dw| <= du, so it is a function of u:
//   v(u) = v0 + a u,  w(u) = w0 + b u,  a = dv/du, b = dw/du, |a|, |b| <= 1.
// A grain in the tube is within R of its foot on the line in every coordinate, so a grain in row (cv, cw)
// has its foot's u inside the intersection of the two slab intervals {u : v(u) in [cv cs - Rw, (cv+1) cs - 1 + Rw]}
// and likewise for w, Rw = R + 2 q, and its own u within Rw of that interval.  The bounds are float (errors
// far below the 2 q of slack, measured in v / w: an error in an interval end is the error of v(u) there divided
// by a, so it does not grow in v) and only have to be a superset: the test decides.
//
// Test: v = P - A and d are exact in float (|v| < 2^16, |d| < 2^11).  c = v x d is formed as
// fma(v1, d2, -rn(v2 d1)): the products stay below 2^27, so |c_f - c| <= 4 + 2^-24 |c| per component, and
// s_f = |c_f|^2 carries a relative error below 2^-22.  With m_up = R_up (|dx| + |dy| + |dz|) >= sqrt(T),
// T = r2 D2, delta = 16 + 2^-21 m_up and band = 1.01 (2 m_up delta + delta^2) + 2^-20 T:
//   s_f < T - band  =>  in the tube;   s_f > T + band  =>  outside;   |s_f - T| <= band: the exact 64-bit
// integer predicate (emu_in_tube) decides.  The result is therefore the exact one in every case
// (DESIGN.md section 6 has the derivation).
enum { kVote = 0, kAssoc = 1 };
constexpr int kRefill = EMU_REFILL;                        // idle lanes of a warp that trigger a refill from the seed stream
constexpr int kRefillStop = EMU_REFILL_STOP;                    // the refill goes on while at least this many lanes are still idle
constexpr int kPairs = 1;                         // pairs of grains a lane tests at most per iteration (the run of a row)

__device__ __forceinline__ unsigned lds_u32(unsigned addr) {
  unsigned v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ unsigned lds_u32_off4(unsigned addr) {
  unsigned v;
  asm volatile("ld.shared.u32 %0, [%1+4];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ unsigned lds_u16(unsigned addr) {
  unsigned short v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
  return (unsigned)v;
}

struct BrickShared {
  int row_gs[kBrickThreads];
  unsigned warp_sum[kBrickThreads / 32];
  unsigned work;
  unsigned next, end;
  int carry;
};

// kBounded: the bounded tube (tube_ext_q >= 0).  The walk is clipped to the part of the line between the seed grains
// plus the extension, and the test adds the axial condition -E |d| <= (P-A).d <= D2 + E |d| in float, as
// |s_f - D2/2| <= D2/2 + E |d|, with its own error band (|s_f - s| <= 16: three products below 2^27; E |d| through
// sqrtf: relative 2^-22 of at most 2^27) and the exact predicate emu_axial_ok inside the band.
template <int kMode, bool kBounded>
__global__ void __launch_bounds__(kBrickThreads, 1)
k_brick(EmuDev P, FramePtrs F, int v0, const Brick* __restrict__ bricks, FindCtl* __restrict__ ctl,
        int slices, const int4* __restrict__ geo, const unsigned* __restrict__ item_ci,
        const unsigned* __restrict__ view_item_off, const PrepRec* __restrict__ prec, const unsigned* __restrict__ brick_off, int prep_sub, unsigned long long* __restrict__ seed_cnt, unsigned short* __restrict__ recs, int* __restrict__ slot_row,
        unsigned long long* __restrict__ keyA, unsigned long long* __restrict__ keyB,
        unsigned long long* __restrict__ counts) {
  extern __shared__ __align__(16) unsigned char pool[];
  __shared__ BrickShared sh;

  if (ctl->skip || ctl->generic) return;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const unsigned n_items = ctl->n_bricks * (unsigned)slices;
  const bool record = (kMode == kVote) && recs != nullptr && ctl->norecord == 0;
  const float R = P.Rw;
  const float r2f = (float)P.r2;
  const float BIG = 1.0e9f;
  unsigned pool_a;                                  // shared-window address of the pool (volatile: computed once)
  asm volatile("mov.u32 %0, %1;" : "=r"(pool_a) : "r"((unsigned)__cvta_generic_to_shared(pool)));
  unsigned long long n_tests = 0;
  int cur_brick = -1;
  Brick B;
  B.view = 0; B.cx0 = B.cx1 = B.cy0 = B.cy1 = B.cz0 = B.cz1 = B.n = 0; B.frame = 0;
  int W = 1, H = 1, S = 4;
  float blo[3] = {0.f, 0.f, 0.f}, bhi[3] = {0.f, 0.f, 0.f};   // brick extent widened by R
  const int4* __restrict__ sorted = F.sorted[0];

  for (;;) {
    __syncthreads();                                  // everyone is done with the previous item
    if (tid == 0) sh.work = atomicAdd(&ctl->work[kMode], 1u);
    __syncthreads();
    const unsigned w = sh.work;
    if (w >= n_items) break;
    const int b = (int)(w / (unsigned)slices), sl = (int)(w % (unsigned)slices);
    if (kMode == kVote) {                                // an item whose slice of the brick's list is empty: nothing to stage
      const unsigned lo = brick_off[b * prep_sub], hi = brick_off[(b + 1) * prep_sub];
      const unsigned per = (hi - lo + (unsigned)slices - 1u) / (unsigned)slices;
      if (min(hi, lo + per * (unsigned)sl) >= hi) continue;
    }

    if (b != cur_brick) {
      // ---- stage brick b ----
      cur_brick = b;
      B = bricks[b];
      sorted = F.sorted[B.frame];
      const int* __restrict__ cell_start = F.cell_start[B.frame];
      const int gnx = P.fr[B.frame].n[0], gny = P.fr[B.frame].n[1];
      W = B.cx1 - B.cx0 + 1; H = B.cy1 - B.cy0 + 1; S = brick_row_stride(W);
      const int rows = H * (B.cz1 - B.cz0 + 1);
      const int vbase = B.view * P.fr[B.frame].ncell;
      unsigned* sgw = reinterpret_cast<unsigned*>(pool);
      unsigned short* tab = reinterpret_cast<unsigned short*>(pool + 4 * (size_t)B.n);
      {
        const int c0[3] = {B.cx0, B.cy0, B.cz0}, c1[3] = {B.cx1, B.cy1, B.cz1};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          blo[a] = (float)(c0[a] * P.cs[a]) - R; bhi[a] = (float)((c1[a] + 1) * P.cs[a] - 1) + R;
        }
      }
      if (tid == 0) sh.carry = 0;
      __syncthreads();
      for (int r0 = 0; r0 < rows; r0 += kBrickThreads) {
        const int r = r0 + tid;
        int gs = 0, len = 0;
        if (r < rows) {
          const int cz = B.cz0 + r / H, cy = B.cy0 + r % H;
          const int rb = vbase + (cz * gny + cy) * gnx;
          gs = __ldg(cell_start + rb + B.cx0);
          len = __ldg(cell_start + rb + B.cx1 + 1) - gs;
        }
        int incl = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += y; }
        if (lane == 31) sh.warp_sum[wid] = (unsigned)incl;
        __syncthreads();
        if (wid == 0) {
          unsigned x = (lane < kBrickThreads / 32) ? sh.warp_sum[lane] : 0u, xi = x;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) { unsigned y = __shfl_up_sync(EMU_FULL, xi, o); if (lane >= o) xi += y; }
          if (lane < kBrickThreads / 32) sh.warp_sum[lane] = xi - x;
        }
        __syncthreads();
        const int carry = sh.carry;
        const int off = carry + (int)sh.warp_sum[wid] + incl - len;     // slot of the first grain of row r
        sh.row_gs[tid] = gs;
        if (r < rows) *reinterpret_cast<int*>(tab + (size_t)r * S + (S - 2)) = gs - off;
        __syncthreads();
        if (tid == kBrickThreads - 1) sh.carry = off + len;
        const int nr = min(kBrickThreads, rows - r0);
        for (int k = wid; k < nr; k += kBrickThreads / 32) {
          const int rr = r0 + k;
          const int rgs = sh.row_gs[k], roff = rgs - *reinterpret_cast<const int*>(tab + (size_t)rr * S + (S - 2));
          const int cz = B.cz0 + rr / H, cy = B.cy0 + rr % H;
          const int rb = vbase + (cz * gny + cy) * gnx + B.cx0;
          for (int i = lane; i <= W; i += 32) tab[(size_t)rr * S + i] = (unsigned short)(roff + (__ldg(cell_start + rb + i) - rgs));
          const int rlen = __ldg(cell_start + rb + W) - rgs;
          const int y0 = cy * P.cs[1], z0 = cz * P.cs[2];
          for (int i = lane; i < rlen; i += 32) {
            const int4 g = __ldg(sorted + rgs + i);
            sgw[roff + i] = (unsigned)g.x | ((unsigned)(g.y - y0) << 16) | ((unsigned)(g.z - z0) << 24);
            if (record && sl == 0) slot_row[B.base + roff + i] = g.w;      // the first item of a brick publishes its rows
          }
        }
        __syncthreads();
      }
    }
    // ---- the slice of the (view, frame)'s items ----
    {
      // VOTE: the brick's own list of prepared seeds (k_prep); ASSOC: the walk list of the brick's (view, frame)
      const int vf = (B.view - v0) * 3 + B.frame;
      const unsigned lo = kMode == kVote ? brick_off[b * prep_sub] : view_item_off[vf];
      const unsigned hi = kMode == kVote ? brick_off[(b + 1) * prep_sub] : view_item_off[vf + 1];
      const unsigned per = (hi - lo + (unsigned)slices - 1u) / (unsigned)slices;
      const unsigned s0 = min(hi, lo + per * (unsigned)sl), s1 = min(hi, s0 + per);
      if (tid == 0) { sh.next = s0; sh.end = s1; }
    }
    __syncthreads();
    const unsigned s_end = sh.end;
    // table address of row (cy = 0, cz = cz0 - 1) of the brick's numbering moved back by cx0 cells, so that
    // cell cx of row cy of the current layer sits at layp + cy * row_b + 2 cx
    const unsigned row_b = 2u * (unsigned)S, lay_b = row_b * (unsigned)H;   // table bytes per row / per w layer
    const unsigned tab0 = pool_a + 4u * (unsigned)B.n - 2u * (unsigned)B.cx0 - (unsigned)B.cy0 * row_b - lay_b;
    const unsigned delta_o = 2u * (unsigned)(B.cx0 + S - 2);               // from a row address to its position word
    const float cz1f = (float)B.cz1, cy1f = (float)B.cy1, cy0f = (float)B.cy0;
    const int ord_shift = record ? 16 * (B.ord & (kRecBricks - 1)) : 0;   // without records: one plain counter
    const size_t rec_ord = (size_t)(B.ord & (kRecBricks - 1)) * kRecSlots;

    // ---- per-lane state: one seed per lane ----
    bool idle = true;                                // no seed (waiting for the next refill)
    float ay = 0.f, dx = 1.f, dy = 0.f, dz = 0.f;
    float a = 0.f, y0 = 0.f;                         // v(u) = y0 + a u
    float oxm = 0.f, oym = 0.f, ozm = 0.f;           // magic-biased origin of v = P - A for the current row
    float T = 0.f, band = 0.f;                       // r2 D2 and the half-width of the float test's error band
    float amid = 0.f, ahalf = 0.f, aband = 0.f;      // bounded tube: |(P-A).d - amid| <= ahalf, error band aband
    unsigned short* rec = nullptr;                   // hit record of the lane's seed in this brick
    float t0 = 0.f, t1 = 0.f;                        // u interval of the line inside the brick
    float pk0 = 0.f, pk1 = 0.f;                      // two values parked between the stages of the refill
    float dty = 0.f, tyl = 0.f, tyh = 0.f, dtz = 0.f, tzl = 0.f, tzh = 0.f;
    float cyf = 1.f, cyhf = 0.f, czf = 0.f, czhf = -1.f;   // current / last row of the layer, current / last layer
    unsigned rowp = 0, layp = 0;                     // table address of the current row / of row 0 of the current layer
    unsigned j = 0, e = 0;                           // shared-memory addresses of the pending run of grains
    unsigned sidx = 0;
    int count = 0;
    unsigned long long ka = 0, kb = 0;
    unsigned wcur = 0, wend = 0;
    bool exhausted = false;
    unsigned item_tests = 0;

    // |(P - A) x d|^2 in float for the grain word g (see the header comment for the error band)
    auto tube_s = [&](unsigned g, float& vx, float& vy, float& vz) {
      vx = __fsub_rn(magic_lo16(g), oxm); vy = __fsub_rn(magic_b2(g), oym); vz = __fsub_rn(magic_b3(g), ozm);
      const float cx = __fmaf_rn(vy, dz, -__fmul_rn(vz, dy));
      const float cyy = __fmaf_rn(vz, dx, -__fmul_rn(vx, dz));
      const float czz = __fmaf_rn(vx, dy, -__fmul_rn(vy, dx));
      return __fmaf_rn(cx, cx, __fmaf_rn(cyy, cyy, __fmul_rn(czz, czz)));
    };
    auto exact_in = [&](float vx, float vy, float vz) {
      const int idx = __float2int_rn(dx), idy = __float2int_rn(dy), idz = __float2int_rn(dz);
      const int ivx = __float2int_rn(vx), ivy = __float2int_rn(vy), ivz = __float2int_rn(vz);
      const long long id2 = (long long)(idx * idx + idy * idy + idz * idz);
      if (!emu_in_tube(ivx, ivy, ivz, 0, 0, 0, idx, idy, idz, (long long)P.r2 * id2)) return false;
      return !kBounded || emu_axial_ok(P.ext, (long long)ivx * idx + (long long)ivy * idy + (long long)ivz * idz, id2);
    };
    // bounded tube: distance of the axial coordinate (P-A).d from the middle of the allowed interval, in float
    auto axial = [&](float vx, float vy, float vz) {
      return fabsf(__fmaf_rn(vx, dx, __fmaf_rn(vy, dy, __fmul_rn(vz, dz))) - amid);
    };

    for (;;) {
      // ---------------- SEED: refill the idle lanes once enough of them wait ----------------
      // Stage 1 (repeated until few lanes are left idle): fetch a seed, unpack it, clip the line against the
      // brick; a seed that misses the brick is dropped at once.  Stage 2 (once per refill, for all the lanes
      // that got a seed): the constants of the traversal and of the test.  Between the stages the values
      // stage 2 needs wait in registers that it overwrites anyway (ozm, tl0, tl1, dty, dtz, count).
      unsigned mS = __ballot_sync(EMU_FULL, idle);
      if (!exhausted && __popc(mS) >= kRefill) {
        bool fresh = false;
        // the counts of the lanes that finished since the last refill leave together (count != 0: not yet flushed)
        if (kMode == kVote && idle && count) { atomicAdd(seed_cnt + sidx, (unsigned long long)min(count, 0xffff) << ord_shift); count = 0; }
        if (kMode == kVote) {
          // the brick's own list: every record is a hit with its clip stored (k_prep), one pass serves the idle lanes
          if (wcur == wend) {
            unsigned base = 0;
            if (lane == 0) base = atomicAdd(&sh.next, (unsigned)kGrab);
            base = __shfl_sync(EMU_FULL, base, 0);
            if (base >= s_end) exhausted = true;
            else { wcur = base; wend = min(base + (unsigned)kGrab, s_end); }
          }
          if (!exhausted) {
            const unsigned idx = wcur + (unsigned)__popc(mS & ((1u << lane) - 1u));
            const bool take = idle && (idx < wend);
            wcur = min(wend, wcur + (unsigned)__popc(mS));
            if (take) {
              const int4 q = __ldg(reinterpret_cast<const int4*>(prec + idx));
              const int4 x = __ldg(reinterpret_cast<const int4*>(prec + idx) + 1);
              oxm = magic_lo16((unsigned)q.x);
              const float ax = oxm - kMagicF;
              ay = magic_hi16((unsigned)q.x) - kMagicF;
              const float az = magic_lo16((unsigned)q.y) - kMagicF;
              dx = magic_lo16((unsigned)q.z) - (kMagicF + 2048.0f); dy = magic_hi16((unsigned)q.z) - (kMagicF + 2048.0f);
              dz = magic_lo16((unsigned)q.w) - (kMagicF + 2048.0f);
              const float inv_dx = rcp_fast(dx);
              a = dy * inv_dx;
              const float bz = dz * inv_dx;
              y0 = __fmaf_rn(-a, ax, ay);
              sidx = (unsigned)x.x; t0 = __int_as_float(x.y); t1 = __int_as_float(x.z);
              ozm = az; pk0 = __int_as_float(x.w); pk1 = __fmaf_rn(-bz, ax, az);       // parked for stage 2
              dty = dy != 0.f ? dx * rcp_fast(dy) : 0.0f; dtz = dz != 0.f ? dx * rcp_fast(dz) : 0.0f;
              fresh = true;
              idle = false;
            }
          }
        } else
        for (;;) {
          if (wcur == wend) {
            unsigned base = 0;
            if (lane == 0) base = atomicAdd(&sh.next, (unsigned)kGrab);
            base = __shfl_sync(EMU_FULL, base, 0);
            if (base >= s_end) { exhausted = true; break; }
            wcur = base; wend = min(base + (unsigned)kGrab, s_end);
          }
          const unsigned idx = wcur + (unsigned)__popc(mS & ((1u << lane) - 1u));
          const bool take = idle && (idx < wend);
          wcur = min(wend, wcur + (unsigned)__popc(mS));
          if (take) {
            const int4 q = __ldg(geo + idx);
            oxm = magic_lo16((unsigned)q.x);
            const float ax = oxm - kMagicF;
            ay = magic_hi16((unsigned)q.x) - kMagicF;
            const float az = magic_lo16((unsigned)q.y) - kMagicF;
            dx = magic_lo16((unsigned)q.z) - (kMagicF + 2048.0f); dy = magic_hi16((unsigned)q.z) - (kMagicF + 2048.0f);
            dz = magic_lo16((unsigned)q.w) - (kMagicF + 2048.0f);
            // du >= 1 (the seed is oriented along +u and u is its dominant axis)
            const float inv_dx = rcp_fast(dx);
            a = dy * inv_dx;
            const float bz = dz * inv_dx;
            y0 = __fmaf_rn(-a, ax, ay);
            const float z0 = __fmaf_rn(-bz, ax, az);
            const float inv_a = dy != 0.f ? dx * rcp_fast(dy) : 0.0f;
            const float inv_b = dz != 0.f ? dx * rcp_fast(dz) : 0.0f;
            // clip the line against the brick's extent (already widened by R): an interval of u
            t0 = blo[0]; t1 = bhi[0];
            bool hit = true;
            if (dy != 0.f) { const float p = (blo[1] - y0) * inv_a, r = (bhi[1] - y0) * inv_a; t0 = fmaxf(t0, fminf(p, r)); t1 = fminf(t1, fmaxf(p, r)); }
            else hit = hit && (ay >= blo[1]) && (ay <= bhi[1]);
            if (dz != 0.f) { const float p = (blo[2] - z0) * inv_b, r = (bhi[2] - z0) * inv_b; t0 = fmaxf(t0, fminf(p, r)); t1 = fminf(t1, fmaxf(p, r)); }
            else hit = hit && (az >= blo[2]) && (az <= bhi[2]);
            if (kBounded) {
              // the feet of the grains that can count lie between u(A) - E du/|d| and u(B) + E du/|d| (2 q of slack)
              const float eu = __fmaf_rn((float)P.ext * dx, rsqrtf(__fmaf_rn(dx, dx, __fmaf_rn(dy, dy, dz * dz))) * 1.0001f, 2.0f);
              t0 = fmaxf(t0, ax - eu); t1 = fminf(t1, ax + dx + eu);
            }
            if (hit && t0 <= t1) {
              sidx = idx;
              ozm = az; pk0 = bz; pk1 = z0; dty = inv_a; dtz = inv_b;       // parked for stage 2
              if (kMode == kAssoc) count = (int)((unsigned)q.y >> 16);        // n_tube of the candidate, parked
              fresh = true;
              idle = false;
            }
          }
          mS = __ballot_sync(EMU_FULL, idle);
          if (__popc(mS) < kRefillStop) break;
        }
        if (fresh) {
          const float az = ozm, bz = pk0, z0 = pk1, inv_a = dty, inv_b = dtz;
          const float D2 = __fmaf_rn(dx, dx, __fmaf_rn(dy, dy, dz * dz));        // exact: < 2^22
          {
            T = r2f * D2;
            const float m_up = P.Rup * (dx + fabsf(dy) + fabsf(dz));
            const float delta = __fmaf_rn(m_up, 4.76837158203125e-7f, 16.0f);   // 16 + 2^-21 m_up
            band = __fmaf_rn(1.01f * delta, __fmaf_rn(2.0f, m_up, delta), T * 9.5367431640625e-7f);
          }
          if (kBounded) {
            const float L = (float)P.ext * sqrtf(D2);
            amid = 0.5f * D2; ahalf = amid + L; aband = __fmaf_rn(L, 1.9073486328125e-6f, 160.0f);   // 160 + 2^-19 E |d|
          }
          if (record) rec = recs + ((size_t)sidx * (kRecBricks * kRecSlots) + rec_ord);
          if (kMode == kAssoc) {
            const unsigned long long k1 = cand_k1(count, __float2int_rn(D2));
            const unsigned ci = __ldg(item_ci + sidx);               // the streamed list is the "walk" list
            ka = (k1 << kCiBits) | (unsigned long long)(kCiMask - ci);
            kb = (k1 << kCiBits) | (unsigned long long)ci;
          }
          count = 0;
          // slab k of an axis covers [k cs - R, (k+1) cs - 1 + R]: its u interval is the one of slab 0 moved by k cs / slope
          dty = P.csf[1] * inv_a; dtz = P.csf[2] * inv_b;
          tyl = -BIG; tyh = BIG; tzl = -BIG; tzh = BIG;
          if (dy != 0.f) { const float p = (-R - y0) * inv_a, r = (P.csf[1] - 1.0f + R - y0) * inv_a; tyl = fminf(p, r); tyh = fmaxf(p, r); }
          if (dz != 0.f) { const float p = (-R - z0) * inv_b, r = (P.csf[2] - 1.0f + R - z0) * inv_b; tzl = fminf(p, r); tzh = fmaxf(p, r); }
          int czi;                                       // the layer before the first
          if (kMode == kVote) {                          // first | last << 16 from the record (k_prep)
            const unsigned lay = __float_as_uint(bz);
            czi = (int)(lay & 0xffffu) - 1;
            czhf = int_f((int)(lay >> 16));
          } else {
            const float za = __fmaf_rn(bz, t0, z0), zb = __fmaf_rn(bz, t1, z0);
            czi = max(B.cz0, rn_int(__fmaf_rn(fminf(za, zb), P.inv_cs[2], P.klo[2]))) - 1;
            czhf = fminf(cz1f, rn_flt(__fmaf_rn(fmaxf(za, zb), P.inv_cs[2], P.khi[2])));
          }
          czf = int_f(czi);
          ozm = __fmaf_rn(-czf, P.csf[2], az + kMagicF);
          layp = tab0 + (unsigned)(czi - B.cz0 + 1) * lay_b;
          cyf = 1.f; cyhf = 0.f;                        // forces a layer step first
          j = 0; e = 0;
        }
      } else if (mS == EMU_FULL) {
        break;                                              // the slice is exhausted and every lane is done
      }

#pragma unroll
      for (int body = 0; body < EMU_BODY_REPS; ++body) {    // advance + test rounds between two looks at the idle lanes
      // ---------------- ADVANCE: lanes whose run is used up move to the next row of cells; a lane whose layer has no
      //                  row left takes the next w layer in the same breath.  ONE instruction sequence serves both
      //                  cases: the layer's u interval and row range are functions of the layer index and are simply
      //                  derived again on every step (it costs less than a second, thinly populated code path) ----
      if (!idle && j >= e) {
        const bool nl = cyf >= cyhf;                        // the rows of the layer are used up
        if (nl) { czf += 1.0f; ozm -= P.csf[2]; layp += lay_b; }
        if (czf > czhf) {                                   // the seed is finished (its count is flushed by the next refill)
          idle = true;
        } else {
          const float tl0 = fmaxf(t0, __fmaf_rn(czf, dtz, tzl)), tl1 = fminf(t1, __fmaf_rn(czf, dtz, tzh));
          const float ya = __fmaf_rn(a, tl0, y0), yb = __fmaf_rn(a, tl1, y0);
          const float cyl = fmaxf(cy0f, rn_flt(__fmaf_rn(fminf(ya, yb), P.inv_cs[1], P.klo[1])));
          const float cyh = fminf(cy1f, rn_flt(__fmaf_rn(fmaxf(ya, yb), P.inv_cs[1], P.khi[1])));
          cyf = nl ? cyl : cyf + 1.0f;
          cyhf = tl0 <= tl1 ? cyh : cyf;                    // an empty layer has no further row
          rowp = layp + (unsigned)rn_int(cyf) * row_b;
          oym = __fmaf_rn(-cyf, P.csf[1], ay + kMagicF);
          const float ta = fmaxf(tl0, __fmaf_rn(cyf, dty, tyl)), tb = fminf(tl1, __fmaf_rn(cyf, dty, tyh));
          if (ta <= tb && cyf <= cyh) {
            const int c0 = max(B.cx0, rn_int(__fmaf_rn(ta, P.inv_cs[0], P.klo[0])));
            const int c1 = min(B.cx1, rn_int(__fmaf_rn(tb, P.inv_cs[0], P.khi[0])));
            if (c0 <= c1) {
              const unsigned sj = lds_u16(rowp + 2u * (unsigned)c0), se = lds_u16(rowp + 2u * (unsigned)c1 + 2u);
              j = pool_a + 4u * sj;
              e = pool_a + 4u * se;
              item_tests += se - sj;
            }
          }
        }
      }
      // ---------------- TEST: up to kPairs pairs of grains of the pending run ----------------
      {
#pragma unroll 1
        for (int pr = 0; pr < kPairs; ++pr) {
          if (j >= e) break;
          {
            const unsigned g0 = lds_u32(j), g1 = lds_u32_off4(j);   // g1 may lie beyond the run (still inside the pool)
            float v0x, v0y, v0z, v1x, v1y, v1z;
            const float s0 = tube_s(g0, v0x, v0y, v0z), s1 = tube_s(g1, v1x, v1y, v1z);
            // what a pair of decisions does: VOTE counts and writes the brick slots of the grains found into the hit
            // record (the first kRecSlots of this seed in this brick), ASSOC joins the priority maximum of the grains
            auto commit = [&](bool in0, bool in1) {
              if (kMode == kVote) {
                if (record) {
                  const unsigned slot = (j - pool_a) >> 2;
                  if (in0) rec[min(count, kRecSlots - 1)] = (unsigned short)slot;
                  count += (int)in0;
                  if (in1) rec[min(count, kRecSlots - 1)] = (unsigned short)(slot + 1u);
                  count += (int)in1;
                } else {
                  count += (int)in0 + (int)in1;
                }
              } else if (in0 || in1) {
                // slot of the grain in the brick + (sorted position - slot) of the first grain of its row -> row of the grain
                const int pos = (int)((j - pool_a) >> 2) + (int)lds_u32(rowp + delta_o);
                if (in0) { const int row = __ldg(&sorted[pos].w); atomicMax(keyA + row, ka); atomicMax(keyB + row, kb); }
                if (in1) { const int row = __ldg(&sorted[pos + 1].w); atomicMax(keyA + row, ka); atomicMax(keyB + row, kb); }
              }
            };
            const bool two = j + 4u < e;
            if (kBounded) {
              const float a0 = axial(v0x, v0y, v0z), a1 = axial(v1x, v1y, v1z);
              if (fminf(fabsf(s0 - T), fabsf(s1 - T)) > band && fminf(fabsf(a0 - ahalf), fabsf(a1 - ahalf)) > aband) {
                commit(s0 <= T && a0 <= ahalf, (s1 <= T && a1 <= ahalf) && two);
              } else {                                             // inside one of the error bands: the exact predicates
                commit(exact_in(v0x, v0y, v0z), exact_in(v1x, v1y, v1z) && two);
              }
            } else if (fminf(fabsf(s0 - T), fabsf(s1 - T)) > band) {   // the common case: the float test decides both
              commit(s0 <= T, (s1 <= T) && two);
            } else {                                               // inside the error band: the exact predicate
              const bool in0 = fabsf(s0 - T) <= band ? exact_in(v0x, v0y, v0z) : (s0 <= T);
              const bool in1 = fabsf(s1 - T) <= band ? exact_in(v1x, v1y, v1z) : (s1 <= T);
              commit(in0, in1 && two);
            }
            j += 8u;
          }
        }
      }
      }   // body
    }
    if (kMode == kVote && count) atomicAdd(seed_cnt + sidx, (unsigned long long)min(count, 0xffff) << ord_shift);
    n_tests += item_tests;
  }

  for (int o = 16; o; o >>= 1) n_tests += __shfl_xor_sync(EMU_FULL, n_tests, o);
  if (lane == 0 && n_tests) atomicAdd(counts + EMU_CNT_TESTS, n_tests);
}

// ---------------------------------------------------------------------------------------------
// A4: candidates = seeds with n_tube >= min_grains, grouped by (view, frame).  grid = (blocks, groups of
// the chunk).  A warp takes 1024 consecutive seeds at a time, counts its candidates with ballots (keeping
// every lane's 32 flags in a register) and makes ONE atomicAdd on the group's counter per 1024 seeds.
// Candidates whose hit records are incomplete (more than kRecSlots grains in one brick, or no records at
// all) also go to the "walk" list (packed geometry + candidate index), which k_brick<kAssoc> streams.
template <int kFill>
__global__ void __launch_bounds__(256)
k_cands(EmuDev P, int v0, const FindCtl* __restrict__ ctl, const unsigned* __restrict__ view_seed_off,
        const unsigned long long* __restrict__ seed_cnt, const int4* __restrict__ geo, const int2* __restrict__ ab,
        unsigned* __restrict__ view_cand_cnt, const unsigned* __restrict__ view_cand_off,
        unsigned* __restrict__ view_ovf_cnt, const unsigned* __restrict__ view_ovf_off,
        Cand* __restrict__ cands, unsigned* __restrict__ cand_seed, int4* __restrict__ ovf_geo,
        unsigned* __restrict__ ovf_ci, unsigned long long* __restrict__ counts) {
  if (ctl->skip || ctl->generic) return;
  const bool fields = ctl->norecord == 0;
  const int vf = blockIdx.y, lane = threadIdx.x & 31;
  const unsigned lo = view_seed_off[vf], hi = view_seed_off[vf + 1];
  const unsigned wpb = blockDim.x >> 5;
  const unsigned span = gridDim.x * wpb * 1024u;
  unsigned status = 0;
  for (unsigned c0 = lo + (blockIdx.x * wpb + (threadIdx.x >> 5)) * 1024u; c0 < hi; c0 += span) {
    unsigned flags = 0, oflags = 0, total = 0, ototal = 0;
#pragma unroll 4
    for (int it = 0; it < 32; ++it) {
      const unsigned i = c0 + (unsigned)it * 32u + (unsigned)lane;
      bool is = false, ov = false;
      if (i < hi) {
        const unsigned long long v = seed_cnt[i];
        is = tube_total(v, fields) >= (unsigned)P.min_grains;
        ov = is && (!fields || tube_overflows(v));
      }
      flags |= (unsigned)is << it; oflags |= (unsigned)ov << it;
      total += __popc(__ballot_sync(EMU_FULL, is));
      ototal += __popc(__ballot_sync(EMU_FULL, ov));
    }
    if (!total) continue;
    unsigned base = 0, obase = 0;
    if (lane == 0) {
      base = atomicAdd(view_cand_cnt + vf, total);
      if (ototal) obase = atomicAdd(view_ovf_cnt + vf, ototal);
    }
    if (!kFill) continue;
    base = __shfl_sync(EMU_FULL, base, 0) + view_cand_off[vf];
    obase = __shfl_sync(EMU_FULL, obase, 0) + view_ovf_off[vf];
    for (int it = 0; it < 32; ++it) {
      const bool is = (flags >> it) & 1u, ov = (oflags >> it) & 1u;
      const unsigned m = __ballot_sync(EMU_FULL, is), mo = __ballot_sync(EMU_FULL, ov);
      if (is) {
        const unsigned i = c0 + (unsigned)it * 32u + (unsigned)lane;
        const unsigned ci = base + (unsigned)__popc(m & ((1u << lane) - 1u));
        const unsigned n = tube_total(seed_cnt[i], fields);
        int4 g = geo[i];
        const int2 p = ab[i];
        int dx, dy, dz;
        geo_d(g, dx, dy, dz);
        if (n > (unsigned)kMaxTube) status |= EMU_ST_RANGE;
        Cand c; c.a = p.x; c.b = p.y; c.n_tube_view = (int)min(n, 0xffffu) | ((vf / 3) << 16); c.d2 = dx * dx + dy * dy + dz * dz;
        cands[ci] = c;
        cand_seed[ci] = i;
        if (ov) {
          const unsigned oi = obase + (unsigned)__popc(mo & ((1u << lane) - 1u));
          g.y = (int)(((unsigned)g.y & 0xffffu) | (min(n, (unsigned)kMaxTube) << 16));
          ovf_geo[oi] = g;
          ovf_ci[oi] = ci;
        }
      }
      base += __popc(m); obase += __popc(mo);
    }
  }
  if (kFill && __any_sync(EMU_FULL, status != 0) && lane == 0) atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)EMU_ST_RANGE);
}

// A5 from the hit records: every candidate whose records are complete gives its packed priority to the
// grains written down by the voting pass (brick slot -> row through slot_row).  grid = (blocks, groups).
__global__ void __launch_bounds__(256)
k_assoc_hits(int v0, const FindCtl* __restrict__ ctl, const unsigned* __restrict__ view_cand_off,
             const Cand* __restrict__ cands, const unsigned* __restrict__ cand_seed,
             const unsigned long long* __restrict__ seed_cnt, const unsigned short* __restrict__ recs,
             const int* __restrict__ slot_row, const int* __restrict__ vf_brick_base,
             unsigned long long* __restrict__ keyA, unsigned long long* __restrict__ keyB) {
  if (ctl->skip || ctl->generic || ctl->norecord) return;
  const int vf = blockIdx.y;
  const unsigned lo = view_cand_off[vf], hi = view_cand_off[vf + 1];
  // one thread per (candidate, brick ordinal): the record is read with two 16-byte loads, the rows of its grains
  // with independent loads, and the priorities leave as fire-and-forget atomics (no thread waits on one)
  const unsigned n4 = (hi - lo) * (unsigned)kRecBricks;
  for (unsigned t = blockIdx.x * blockDim.x + threadIdx.x; t < n4; t += gridDim.x * blockDim.x) {
    const unsigned ci = lo + t / (unsigned)kRecBricks;
    const int ord = (int)(t % (unsigned)kRecBricks);
    const unsigned i = cand_seed[ci];
    const unsigned long long v = seed_cnt[i];
    if (tube_overflows(v)) continue;                        // walked by k_brick<kAssoc>
    const int cnt = (int)((v >> (16 * ord)) & 0xffffu);
    if (!cnt) continue;
    const Cand c = cands[ci];
    const unsigned long long k1 = cand_k1(c.n_tube_view & 0xffff, c.d2);
    const unsigned long long ka = (k1 << kCiBits) | (unsigned long long)(kCiMask - ci);
    const unsigned long long kb = (k1 << kCiBits) | (unsigned long long)ci;
    const int base = vf_brick_base[vf * kRecBricks + ord];
    const uint4* rec = reinterpret_cast<const uint4*>(recs + ((size_t)i * (kRecBricks * kRecSlots) + (size_t)ord * kRecSlots));
    const uint4 r0 = __ldg(rec);
    const uint4 r1 = cnt > 8 ? __ldg(rec + 1) : make_uint4(0u, 0u, 0u, 0u);
    const unsigned w[8] = {r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, r1.z, r1.w};
    int rows[kRecSlots];
#pragma unroll
    for (int k = 0; k < kRecSlots; ++k) {
      const int slot = (int)((w[k >> 1] >> (16 * (k & 1))) & 0xffffu);
      rows[k] = k < cnt ? slot_row[base + slot] : -1;
    }
    // A grain is hit by hundreds of candidates and only the few that raise its maximum matter: look first (a plain
    // load that may be stale - the keys only grow, so an old value can cause a needless atomic, never a missing one) and
    // join the maximum only if this candidate's (n_tube, D2) is not already beaten.  Equal (n_tube, D2) must go on:
    // that is the tie the two keys exist to detect.
    unsigned long long seen[kRecSlots];
#pragma unroll
    for (int k = 0; k < kRecSlots; ++k) seen[k] = rows[k] >= 0 ? __ldcg(keyA + rows[k]) : ~0ull;
#pragma unroll
    for (int k = 0; k < kRecSlots; ++k) {
      if (rows[k] >= 0 && (seen[k] >> kCiBits) <= k1) { atomicMax(keyA + rows[k], ka); atomicMax(keyB + rows[k], kb); }
    }
  }
}

// seed dump for emu_count_seeds: (view, row_a, row_b, n_tube), rows ordered
__global__ void __launch_bounds__(256)
k_seed_dump(int v0, const FindCtl* __restrict__ ctl, const int4* __restrict__ sorted,
            const unsigned* __restrict__ view_seed_off, const unsigned long long* __restrict__ seed_cnt,
            const int2* __restrict__ ab, int4* __restrict__ dump, long long dump_cap) {
  if (ctl->skip || ctl->generic) return;
  const bool fields = ctl->norecord == 0;
  const int vf = blockIdx.y;
  const unsigned lo = view_seed_off[vf], hi = view_seed_off[vf + 1];
  for (unsigned i = lo + blockIdx.x * blockDim.x + threadIdx.x; i < hi; i += gridDim.x * blockDim.x) {
    if ((long long)i >= dump_cap) continue;
    const int2 p = ab[i];
    const int ra = sorted[p.x].w, rb = sorted[p.y].w;
    dump[i] = make_int4(v0 + vf / 3, min(ra, rb), max(ra, rb), (int)tube_total(seed_cnt[i], fields));
  }
}

// ---------------------------------------------------------------------------------------------
// Generic fallback (global-memory walker): A2 + A3 + A4 in one kernel, one warp per grain A.
template <bool kDump>
__global__ void __launch_bounds__(kVoteThreads)
k_vote_generic(EmuDev P, const int4* __restrict__ sorted, const int* __restrict__ cell_start,
               const int* __restrict__ view_off, const EmuBox* __restrict__ bbox, int v0, int v1,
               Cand* __restrict__ cands, unsigned cand_cap, FindCtl* __restrict__ ctl,
               int4* __restrict__ dump, long long dump_cap, unsigned long long* __restrict__ dump_cursor,
               unsigned long long* __restrict__ counts) {
  __shared__ int queue_s[kVoteThreads / 32][64];
  if (ctl->skip || !ctl->generic) return;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  int* queue = queue_s[wib];
  const int nwarps = gridDim.x * (kVoteThreads / 32);
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  unsigned long long n_tests = 0, n_cands = 0;
  unsigned status = 0;

  for (int a = g0 + blockIdx.x * (kVoteThreads / 32) + wib; a < g1; a += nwarps) {
    const int v = emu_find_view(view_off, v0, v1, a);
    const int4 A = __ldg(sorted + a);
    const int vbase = v * P.ncell;
    EmuBox bb = bbox[v];
    const int cxa = emu_cell_axis(A.x - P.sep_max, P.cs[0], P.inv_cs[0], P.n[0]);
    const int cxb = emu_cell_axis(A.x + P.sep_max, P.cs[0], P.inv_cs[0], P.n[0]);
    const int cya = emu_cell_axis(A.y - P.sep_max, P.cs[1], P.inv_cs[1], P.n[1]);
    const int cyb = emu_cell_axis(A.y + P.sep_max, P.cs[1], P.inv_cs[1], P.n[1]);
    const int czA = emu_cell_axis(A.z, P.cs[2], P.inv_cs[2], P.n[2]);
    const int czb = emu_cell_axis(A.z + P.sep_max, P.cs[2], P.inv_cs[2], P.n[2]);
    int qhead = 0, qn = 0;

    auto process = [&](int cnt) {
      int b = (lane < cnt) ? queue[(qhead + lane) & 63] : -1;
      int n_tube = 0, d2 = 0;
      int4 B = make_int4(0, 0, 0, 0);
      if (b >= 0) {
        B = __ldg(sorted + b);
        int dx = B.x - A.x, dy = B.y - A.y, dz = B.z - A.z;
        d2 = dx * dx + dy * dy + dz * dz;
        long long r2D2 = (long long)P.r2 * d2;
        n_tests += emu_walk_tube(P, bb, sorted, cell_start, vbase, A.x, A.y, A.z, dx, dy, dz, r2D2,
                                 [&](int) { ++n_tube; });
      }
      if (kDump) {
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(dump_cursor, (unsigned long long)cnt);
        base = __shfl_sync(EMU_FULL, base, 0);
        if (b >= 0 && (long long)(base + lane) < dump_cap)
          dump[base + lane] = make_int4(v, min(A.w, B.w), max(A.w, B.w), n_tube);
      }
      bool is_cand = (b >= 0) && (n_tube >= P.min_grains);
      unsigned m = __ballot_sync(EMU_FULL, is_cand);
      if (m && !kDump) {
        unsigned base = 0;
        if (lane == 0) base = atomicAdd(&ctl->cand_count, (unsigned)__popc(m));
        base = __shfl_sync(EMU_FULL, base, 0);
        if (is_cand) {
          unsigned idx = base + __popc(m & ((1u << lane) - 1u));
          if (n_tube > kMaxTube) status |= EMU_ST_RANGE;
          if (idx < cand_cap) {
            Cand c; c.a = a; c.b = b; c.n_tube_view = min(n_tube, 0xffff) | ((v - v0) << 16); c.d2 = d2;
            cands[idx] = c;
          }
        }
      }
      n_cands += is_cand;
    };

    for (int cz = czA; cz <= czb; ++cz) {
      for (int cy = cya; cy <= cyb; ++cy) {
        const int rb = vbase + (cz * P.n[1] + cy) * P.n[0];
        int s = __ldg(cell_start + rb + cxa);
        const int e = __ldg(cell_start + rb + cxb + 1);
        s = max(s, a + 1);
        for (int j0 = s; j0 < e; j0 += 32) {
          const int j = j0 + lane;
          bool ok = false;
          if (j < e) {
            int4 B = __ldg(sorted + j);
            int dx = B.x - A.x, dy = B.y - A.y, dz = B.z - A.z;
            long long d2 = (long long)dx * dx + (long long)dy * dy + (long long)dz * dz;
            ok = (d2 >= P.sep_min2) && (d2 < P.sep_max2);
          }
          unsigned m = __ballot_sync(EMU_FULL, ok);
          if (ok) queue[(qhead + qn + __popc(m & ((1u << lane) - 1u))) & 63] = j;
          qn += __popc(m);
          __syncwarp();
          if (qn >= 32) { process(32); qhead = (qhead + 32) & 63; qn -= 32; __syncwarp(); }
        }
      }
    }
    if (qn) { process(qn); __syncwarp(); }
  }
  for (int o = 16; o; o >>= 1) {
    n_tests += __shfl_xor_sync(EMU_FULL, n_tests, o);
    n_cands += __shfl_xor_sync(EMU_FULL, n_cands, o);
    status |= __shfl_xor_sync(EMU_FULL, status, o);
  }
  if (lane == 0) {
    atomicAdd(counts + EMU_CNT_TESTS, n_tests);
    if (!kDump) atomicAdd(counts + EMU_CNT_CANDIDATES, n_cands);
    if (status) atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)status);
  }
}

// after the candidates of a chunk are known: capacity check, reset of the tie flag
__global__ void k_cands_finish(FindCtl* ctl, unsigned cand_cap, unsigned long long* counts) {
  unsigned n = ctl->cand_count;
  if (n > cand_cap) { atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)EMU_ST_CAND_OVERFLOW); ctl->cand_count = 0; ctl->skip = 1; }
  ctl->tie = 0;
}

// ---------------------------------------------------------------------------------------------
// A5 with the generic walker.  kPass 0: priority maximum (only when the chunk runs generic).
// kPass 1: settlement of ties - every candidate whose (n_tube, D2) is flagged in the tie bitmap walks
// its tube again and competes for the tied grains by (kmin, kmax) with a CAS-min.
//   keyA = K1 << 29 | (mask - ci)   keyB = K1 << 29 | ci,   K1 = n_tube << 22 | D2, both indexed by ROW.
// The top K1 of a grain is unique; keyA and keyB then name the same candidate unless several
// candidates tie on K1 for that grain.
__device__ __forceinline__ unsigned tie_hash(unsigned long long k1, int vl) {
  unsigned long long h = (k1 ^ ((unsigned long long)vl << 40)) * 0x9E3779B97F4A7C15ull;
  return (unsigned)(h >> 48) & (kTieBits - 1);
}

template <int kPass>
__global__ void __launch_bounds__(kVoteThreads)
k_assoc_generic(EmuDev P, const int4* __restrict__ sorted, const int* __restrict__ cell_start,
                const EmuBox* __restrict__ bbox, int v0, const Cand* __restrict__ cands, const FindCtl* __restrict__ ctl,
                const unsigned* __restrict__ tie_bits, unsigned long long* __restrict__ keyA,
                unsigned long long* __restrict__ keyB, unsigned* __restrict__ owner) {
  if (ctl->skip) return;
  if (kPass == 0 && !ctl->generic) return;
  if (kPass == 1 && ctl->tie == 0) return;
  const unsigned n = ctl->cand_count;
  const unsigned stride = gridDim.x * blockDim.x;
  for (unsigned ci = blockIdx.x * blockDim.x + threadIdx.x; ci < n; ci += stride) {
    const Cand c = cands[ci];
    const int vl = c.n_tube_view >> 16;
    const unsigned long long k1 = cand_k1(c.n_tube_view & 0xffff, c.d2);
    if (kPass == 1) {
      const unsigned h = tie_hash(k1, vl);
      if (!((tie_bits[h >> 5] >> (h & 31)) & 1u)) continue;
    }
    const int v = v0 + vl;
    const int4 A = __ldg(sorted + c.a), B = __ldg(sorted + c.b);
    const int dx = B.x - A.x, dy = B.y - A.y, dz = B.z - A.z;
    const EmuBox bb = bbox[v];
    if (kPass == 0) {
      const unsigned long long ka = (k1 << kCiBits) | (unsigned long long)(kCiMask - ci);
      const unsigned long long kb = (k1 << kCiBits) | (unsigned long long)ci;
      emu_walk_tube(P, bb, sorted, cell_start, v * P.ncell, A.x, A.y, A.z, dx, dy, dz, (long long)P.r2 * c.d2,
                    [&](int j) { const int g = sorted[j].w; atomicMax(keyA + g, ka); atomicMax(keyB + g, kb); });
    } else {
      emu_walk_tube(P, bb, sorted, cell_start, v * P.ncell, A.x, A.y, A.z, dx, dy, dz, (long long)P.r2 * c.d2,
                    [&](int j) {
                      const int g = sorted[j].w;                 // keys and owners are indexed by row
                      if ((keyA[g] >> kCiBits) != k1) return;
                      unsigned cur = owner[g];
                      while (cur == kNone || (cur != ci && cand_kless(sorted, c, cands[cur]))) {
                        unsigned old = atomicCAS(owner + g, cur, ci);
                        if (old == cur) break;
                        cur = old;
                      }
                    });
    }
  }
}

// a grain whose keyA and keyB name different candidates has a tie at its top priority: flag that
// priority in the bitmap (the settlement pass re-walks only candidates with a flagged priority)
__global__ void __launch_bounds__(256)
k_tie_detect(const int* __restrict__ view_off, int v0, int v1, const unsigned long long* __restrict__ keyA,
             const unsigned long long* __restrict__ keyB, FindCtl* __restrict__ ctl, unsigned* __restrict__ tie_bits) {
  if (ctl->skip) return;
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  bool tie = false;
  for (int g = g0 + blockIdx.x * blockDim.x + threadIdx.x; g < g1; g += gridDim.x * blockDim.x) {
    unsigned long long ka = keyA[g], kb = keyB[g];
    if (ka && (kCiMask - (unsigned)(ka & kCiMask)) != (unsigned)(kb & kCiMask)) {
      tie = true;
      const int vl = emu_find_view(view_off, v0, v1, g) - v0;
      const unsigned h = tie_hash(ka >> kCiBits, vl);
      atomicOr(tie_bits + (h >> 5), 1u << (h & 31));
    }
  }
  if (__any_sync(EMU_FULL, tie) && (threadIdx.x & 31) == 0) ctl->tie = 1;
}

__device__ __forceinline__ unsigned owner_of(int g, const FindCtl* ctl, const unsigned long long* keyA,
                                             const unsigned long long* keyB, const unsigned* owner) {
  const unsigned long long ka = keyA[g];
  if (!ka) return kNone;
  const unsigned ca = kCiMask - (unsigned)(ka & kCiMask);
  if (ctl->tie && ca != (unsigned)(keyB[g] & kCiMask)) return owner[g];
  return ca;
}

// A5 part 2: members won per candidate
__global__ void __launch_bounds__(256)
k_wins(const int* __restrict__ view_off, int v0, int v1, const FindCtl* __restrict__ ctl,
       const unsigned long long* __restrict__ keyA, const unsigned long long* __restrict__ keyB,
       const unsigned* __restrict__ owner, int* __restrict__ wins) {
  if (ctl->skip) return;
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  for (int g = g0 + blockIdx.x * blockDim.x + threadIdx.x; g < g1; g += gridDim.x * blockDim.x) {
    unsigned ci = owner_of(g, ctl, keyA, keyB, owner);
    if (ci != kNone) atomicAdd(wins + ci, 1);
  }
}

// A5 part 3: "again the threshold on number of grains is applied to all tracks"
__global__ void __launch_bounds__(256)
k_select(EmuDev P, const Cand* __restrict__ cands, const FindCtl* __restrict__ ctl, const int* __restrict__ wins,
         int* __restrict__ view_ntracks, unsigned* __restrict__ view_tracks, unsigned* __restrict__ cand_slot,
         unsigned long long* __restrict__ counts) {
  if (ctl->skip) return;
  const unsigned n = ctl->cand_count;
  for (unsigned ci = blockIdx.x * blockDim.x + threadIdx.x; ci < n; ci += gridDim.x * blockDim.x) {
    if (wins[ci] >= P.min_grains) {
      int vl = cands[ci].n_tube_view >> 16;
      int slot = atomicAdd(view_ntracks + vl, 1);
      if (slot < P.max_tracks) {
        view_tracks[(size_t)vl * P.max_tracks + slot] = ci;
        if (P.angle_cut) cand_slot[ci] = (unsigned)slot;           // for k_cut_acc (cand_track is free until k_track_emit)
      } else {
        atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)EMU_ST_TRACK_OVERFLOW);
      }
    }
  }
}

// ---- A5b: angle-dependent cut on the number of grains (Fig. 8(c); emu.h angle_min_grains; reading Q17) ----
// The members of the surviving candidates are not listed yet, so every grain adds itself to the moment sums of its
// owner (slot = place of the owner in its view's track list): extents and the nine sums S(x), S(y), S(z), S(xx), ...,
// from which the direction of the least-squares line of emu_fit follows exactly: it is proportional to the integers
// (den, num_v, num_w) along (u, v, w).  bin = largest k with (k/8)^2 <= cos^2 = c_z^2 / (den^2 + num_v^2 + num_w^2),
// decided in 128-bit integers (|den|, |num| <= 2^60: n < 2^13, |coord| < 2^17).  A track with fewer members than
// angle_min[bin] leaves the list; its grains stay unassigned.
struct CutAcc { int lo[3], hi[3]; long long s[9]; };   // 96 B: sums x, y, z, xx, yy, zz, xy, xz, yz

__global__ void __launch_bounds__(256)
k_cut_init(EmuDev P, int nv, const FindCtl* __restrict__ ctl, const int* __restrict__ view_ntracks, CutAcc* __restrict__ acc) {
  if (ctl->skip) return;
  const int vl = blockIdx.y;
  if (vl >= nv) return;
  const int nt = min(view_ntracks[vl], P.max_tracks);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nt; i += gridDim.x * blockDim.x) {
    CutAcc a;
    for (int k = 0; k < 3; ++k) { a.lo[k] = 0x7fffffff; a.hi[k] = (int)0x80000000; }
    for (int k = 0; k < 9; ++k) a.s[k] = 0;
    acc[(size_t)vl * P.max_tracks + i] = a;
  }
}

__global__ void __launch_bounds__(256)
k_cut_acc(EmuDev P, const int4* __restrict__ sorted, const int* __restrict__ view_off, int v0, int v1,
          const FindCtl* __restrict__ ctl, const unsigned long long* __restrict__ keyA,
          const unsigned long long* __restrict__ keyB, const unsigned* __restrict__ owner, const Cand* __restrict__ cands,
          const unsigned* __restrict__ cand_slot, CutAcc* __restrict__ acc) {
  if (ctl->skip) return;
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  for (int j = g0 + blockIdx.x * blockDim.x + threadIdx.x; j < g1; j += gridDim.x * blockDim.x) {
    const int4 g = __ldg(sorted + j);
    const unsigned ci = owner_of(g.w, ctl, keyA, keyB, owner);
    if (ci == kNone) continue;
    const unsigned slot = cand_slot[ci];
    if (slot == kNone) continue;
    CutAcc* a = acc + ((size_t)(cands[ci].n_tube_view >> 16) * P.max_tracks + slot);
    const int c[3] = {g.x, g.y, g.z};
#pragma unroll
    for (int k = 0; k < 3; ++k) { atomicMin(&a->lo[k], c[k]); atomicMax(&a->hi[k], c[k]); }
    const long long x = g.x, y = g.y, z = g.z;
    const long long v[9] = {x, y, z, x * x, y * y, z * z, x * y, x * z, y * z};
#pragma unroll
    for (int k = 0; k < 9; ++k) atomicAdd(reinterpret_cast<unsigned long long*>(&a->s[k]), (unsigned long long)v[k]);
  }
}

__device__ __forceinline__ unsigned __int128 sq128(long long a) {
  const unsigned __int128 m = (unsigned __int128)(unsigned long long)(a < 0 ? -a : a);
  return m * m;
}

__global__ void __launch_bounds__(256)
k_cut_decide(EmuDev P, int nv, const FindCtl* __restrict__ ctl, const int* __restrict__ view_ntracks,
             unsigned* __restrict__ view_tracks, const int* __restrict__ wins, const CutAcc* __restrict__ acc,
             unsigned* __restrict__ cand_slot) {
  if (ctl->skip) return;
  const int vl = blockIdx.y;
  if (vl >= nv) return;
  const int nt = min(view_ntracks[vl], P.max_tracks);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nt; i += gridDim.x * blockDim.x) {
    const size_t at = (size_t)vl * P.max_tracks + i;
    const unsigned ci = view_tracks[at];
    cand_slot[ci] = kNone;                                     // back to "no track yet" for k_track_emit
    const CutAcc a = acc[at];
    const long long ex = (long long)a.hi[0] - a.lo[0], ey = (long long)a.hi[1] - a.lo[1], ez = (long long)a.hi[2] - a.lo[2];
    // dominant axis by member extent, ties z, x, y (emu_fit); s: 0 x, 1 y, 2 z, 3 xx, 4 yy, 5 zz, 6 xy, 7 xz, 8 yz
    long long Su, Sv, Sw, Suu, Suv, Suw;
    bool u_is_z = false;
    if (ez >= ex && ez >= ey) { u_is_z = true; Su = a.s[2]; Sv = a.s[0]; Sw = a.s[1]; Suu = a.s[5]; Suv = a.s[7]; Suw = a.s[8]; }
    else if (ex >= ey)        { Su = a.s[0]; Sv = a.s[1]; Sw = a.s[2]; Suu = a.s[3]; Suv = a.s[6]; Suw = a.s[7]; }
    else                      { Su = a.s[1]; Sv = a.s[0]; Sw = a.s[2]; Suu = a.s[4]; Suv = a.s[6]; Suw = a.s[8]; }
    const long long N = wins[ci];
    const long long den = N * Suu - Su * Su, nvv = N * Suv - Su * Sv, nww = N * Suw - Su * Sw;
    if (den == 0) continue;                                    // all members coincide: no direction, never cut
    const unsigned __int128 S = sq128(den) + sq128(nvv) + sq128(nww);
    const unsigned __int128 cz2 = u_is_z ? sq128(den) : sq128(nww);
    int bin = 0;
#pragma unroll
    for (int k = 1; k <= 7; ++k) if ((unsigned __int128)(k * k) * S <= (unsigned __int128)64 * cz2) bin = k;
    if ((int)N < P.angle_min[bin]) view_tracks[at] = kNone;
  }
}

// the per-view track lists without the tracks the cut removed (one block per view; in place: a tile is read, the
// block synchronises, and its survivors land at or before the places just read)
__global__ void __launch_bounds__(256)
k_cut_compact(EmuDev P, int nv, const FindCtl* __restrict__ ctl, int* __restrict__ view_ntracks, unsigned* __restrict__ view_tracks) {
  __shared__ int warp_sum[8];
  __shared__ int base_s;
  if (ctl->skip) return;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int vl = blockIdx.x; vl < nv; vl += gridDim.x) {
    const int nt = min(view_ntracks[vl], P.max_tracks);
    unsigned* list = view_tracks + (size_t)vl * P.max_tracks;
    if (threadIdx.x == 0) base_s = 0;
    __syncthreads();
    for (int i0 = 0; i0 < nt; i0 += blockDim.x) {
      const int i = i0 + threadIdx.x;
      const unsigned ci = i < nt ? list[i] : kNone;
      const bool keep = ci != kNone;
      const unsigned m = __ballot_sync(EMU_FULL, keep);
      if (lane == 0) warp_sum[wid] = __popc(m);
      __syncthreads();
      int before = 0, total = 0;
      for (int w = 0; w < 8; ++w) { if (w < wid) before += warp_sum[w]; total += warp_sum[w]; }
      const int base = base_s;
      __syncthreads();
      if (keep) list[base + before + __popc(m & ((1u << lane) - 1u))] = ci;
      if (threadIdx.x == 0) base_s = base + total;
      __syncthreads();
    }
    if (threadIdx.x == 0) view_ntracks[vl] = base_s;    // (<= max_tracks: k_track_scan's clamp changes nothing)
    __syncthreads();
  }
}

// A7: track_off over the chunk's views (one block; continues from the previous chunk's total)
__global__ void __launch_bounds__(1024)
k_track_scan(EmuDev P, int v0, int v1, int* __restrict__ view_ntracks, int* __restrict__ track_off) {
  __shared__ int warp_sum[32];
  __shared__ int carry_s;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x == 0) { if (v0 == 0) track_off[0] = 0; carry_s = (v0 == 0) ? 0 : track_off[v0]; }
  __syncthreads();
  for (int b = v0; b < v1; b += blockDim.x) {
    int v = b + threadIdx.x;
    int x = 0;
    if (v < v1) { x = min(view_ntracks[v - v0], P.max_tracks); view_ntracks[v - v0] = x; }
    int incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += y; }
    if (lane == 31) warp_sum[wid] = incl;
    __syncthreads();
    if (wid == 0) {
      int w = warp_sum[lane], wi = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(EMU_FULL, wi, o); if (lane >= o) wi += y; }
      warp_sum[lane] = wi - w;
    }
    __syncthreads();
    int carry = carry_s;
    if (v < v1) track_off[v + 1] = carry + warp_sum[wid] + incl;
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry_s = carry + warp_sum[wid] + incl;
    __syncthreads();
  }
}

// A7: inside a view, best first.  rank = number of better tracks (the order is total, reading Q15).
__global__ void __launch_bounds__(256)
k_track_emit(EmuDev P, const int4* __restrict__ sorted, int v0, int v1, const Cand* __restrict__ cands,
             const int* __restrict__ wins, const int* __restrict__ view_ntracks,
             const unsigned* __restrict__ view_tracks, const int* __restrict__ track_off,
             emu_track* __restrict__ tracks, unsigned* __restrict__ cand_track) {
  // grid = (parts, views): the tracks of a view are dealt to gridDim.x blocks (one view alone would otherwise rank its
  // 1 400 tracks against one another in a single block: 1.9 ms for a config-4 view)
  for (int v = v0 + blockIdx.y; v < v1; v += gridDim.y) {
    const int nt = view_ntracks[v - v0];
    const unsigned* list = view_tracks + (size_t)(v - v0) * P.max_tracks;
    const int t0 = track_off[v];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nt; i += gridDim.x * blockDim.x) {
      const unsigned ci = list[i];
      const Cand c = cands[ci];
      int rank = 0;
      for (int j = 0; j < nt; ++j) {
        if (j == i) continue;
        rank += cand_better(sorted, cands[list[j]], c);
      }
      const int4 A = sorted[c.a], B = sorted[c.b];
      emu_track t;
      t.view = v; t.seed_a = min(A.w, B.w); t.seed_b = max(A.w, B.w);
      t.n_tube = c.n_tube_view & 0xffff; t.n_members = wins[ci]; t.member_off = 0; t.seed_d2 = c.d2; t.pad = 0;
      tracks[t0 + rank] = t;
      cand_track[ci] = (unsigned)(t0 + rank);
    }
  }
}

// member_off = running sum of n_members over the chunk's tracks in final order (one block);
// also resets the per-track fill cursors and publishes the running totals.
__global__ void __launch_bounds__(1024)
k_member_scan(int v0, int v1, const int* __restrict__ track_off, emu_track* __restrict__ tracks,
              int* __restrict__ cursor, unsigned long long* __restrict__ counts, long long members_capacity) {
  __shared__ long long warp_sum[32];
  __shared__ long long carry_s;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int t0 = track_off[v0], t1 = track_off[v1];
  if (threadIdx.x == 0) carry_s = (long long)counts[EMU_CNT_MEMBERS];
  __syncthreads();
  for (int b = t0; b < t1; b += blockDim.x) {
    int t = b + threadIdx.x;
    long long x = (t < t1) ? tracks[t].n_members : 0;
    long long incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { long long y = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += y; }
    if (lane == 31) warp_sum[wid] = incl;
    __syncthreads();
    if (wid == 0) {
      long long w = warp_sum[lane], wi = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { long long y = __shfl_up_sync(EMU_FULL, wi, o); if (lane >= o) wi += y; }
      warp_sum[lane] = wi - w;
    }
    __syncthreads();
    long long carry = carry_s;
    if (t < t1) {
      long long off = carry + warp_sum[wid] + incl - x;
      tracks[t].member_off = (int)min(off, (long long)0x7fffffff);
      cursor[t - t0] = 0;
      if (off + x > members_capacity) {
        // the list does not fit: the track carries no members (emu_fit_tracks then reads nothing); the total needed
        // still goes to counts[EMU_CNT_MEMBERS]
        atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)EMU_ST_MEMBER_OVERFLOW);
        tracks[t].n_members = 0; tracks[t].member_off = 0;
      }
    }
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry_s = carry + warp_sum[wid] + incl;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    counts[EMU_CNT_MEMBERS] = (unsigned long long)carry_s;
    counts[EMU_CNT_TRACKS] = (unsigned long long)t1;
  }
}

__global__ void __launch_bounds__(256)
k_member_scatter(const int4* __restrict__ sorted, const int* __restrict__ view_off, int v0, int v1,
                 const FindCtl* __restrict__ ctl, const unsigned long long* __restrict__ keyA,
                 const unsigned long long* __restrict__ keyB, const unsigned* __restrict__ owner,
                 const unsigned* __restrict__ cand_track, const int* __restrict__ track_off,
                 const emu_track* __restrict__ tracks, int* __restrict__ cursor, int* __restrict__ members,
                 long long members_capacity) {
  if (ctl->skip) return;
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  const int t0 = track_off[v0];
  for (int g = g0 + blockIdx.x * blockDim.x + threadIdx.x; g < g1; g += gridDim.x * blockDim.x) {
    unsigned ci = owner_of(g, ctl, keyA, keyB, owner);
    if (ci == kNone) continue;
    unsigned t = cand_track[ci];
    if (t == kNone || tracks[t].n_members == 0) continue;     // (no members: the list did not fit, k_member_scan)
    int k = atomicAdd(cursor + (t - t0), 1);
    long long pos = (long long)tracks[t].member_off + k;
    if (pos < members_capacity) members[pos] = g;                // g is a row
  }
}

// members of a track in ascending row order: one warp per track, rank sort through shared memory
constexpr int kSortCap = 1024;
__global__ void __launch_bounds__(256)
k_member_sort(int v0, int v1, const int* __restrict__ track_off, const emu_track* __restrict__ tracks,
              int* __restrict__ members, long long members_capacity) {
  __shared__ int buf_s[8][kSortCap];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  int* buf = buf_s[wib];
  const int t0 = track_off[v0], t1 = track_off[v1];
  for (int t = t0 + blockIdx.x * 8 + wib; t < t1; t += gridDim.x * 8) {
    const int n = tracks[t].n_members;
    const long long off = tracks[t].member_off;
    if (off + n > members_capacity) continue;
    int* m = members + off;
    if (n <= kSortCap) {
      for (int i = lane; i < n; i += 32) buf[i] = m[i];
      __syncwarp();
      for (int i = lane; i < n; i += 32) {
        int x = buf[i], r = 0;
        for (int k = 0; k < n; ++k) r += (buf[k] < x);
        m[r] = x;                                   // rows are distinct: ranks are a permutation
      }
      __syncwarp();
    } else {
      // rare (a track with more than 1024 grains): odd-even transposition in place
      for (int pass = 0; pass < n; ++pass) {
        for (int i = (pass & 1) + 2 * lane; i + 1 < n; i += 64) {
          int x = m[i], y = m[i + 1];
          if (x > y) { m[i] = y; m[i + 1] = x; }
        }
        __syncwarp();
      }
    }
  }
}

// arrays sized by the chunk's candidate count (read on the device)
__global__ void k_reset_cand_arrays(const FindCtl* ctl, int* wins, unsigned* cand_track) {
  const unsigned n = ctl->cand_count;
  for (unsigned i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) { wins[i] = 0; cand_track[i] = kNone; }
}

// ---------------------------------------------------------------------------------------------
// workspace
struct FindWs {
  EmuBox* bbox; unsigned long long* keyA; unsigned long long* keyB; unsigned* owner; unsigned* seed_off;
  FindCtl* ctl; unsigned* tie_bits; unsigned long long* dump_cursor;
  unsigned* view_seed_tot; unsigned* view_seed_off; unsigned* view_cand_cnt; unsigned* view_cand_off;
  int* view_ntracks; unsigned* view_tracks; Brick* bricks;
  int4* sortedF[3]; int* cell_startF[3]; void* bin_ws; size_t bin_ws_bytes;     // frames 1, 2 (0 = the caller's)
  int* slot_row; int* vf_brick_base; unsigned* view_ovf_cnt; unsigned* view_ovf_off;
  int4* geo; int2* ab; unsigned long long* seed_cnt; unsigned short* recs;
  PrepRec* prec; size_t prep_cap; int2* vf_bricks; unsigned* brick_cnt; unsigned* brick_off; int prep_sub;
  Cand* cands; unsigned* cand_seed; int4* ovf_geo; unsigned* ovf_ci; int* wins; unsigned* cand_track;
  CutAcc* cut_acc;                                                                // only with the angle cut
  size_t seed_cap, cand_cap, brick_cap; int views_per_chunk;
};

constexpr size_t kRecBytes = (size_t)kRecBricks * kRecSlots * sizeof(unsigned short);             // 128 per seed
constexpr size_t kPrepPerSeed8 = 20;    // (seed, brick) records reserved per seed, in eighths: 2.5 (1.9 on the bench)
constexpr size_t kSeedBytes = sizeof(int4) + sizeof(int2) + sizeof(unsigned long long) + kRecBytes + kPrepPerSeed8 * sizeof(PrepRec) / 8;   // 240
constexpr size_t kCandBytes = sizeof(Cand) + sizeof(unsigned) + sizeof(int4) + sizeof(unsigned) + sizeof(int) + sizeof(unsigned);  // 48
constexpr size_t kMinSeedCap = 1u << 20, kMinCandCap = 1u << 16;

size_t bricks_per_view(const EmuDev& P, const Tilings& TT) {
  size_t n = 0;
  for (int f = 0; f < 3; ++f) n += (size_t)TT.t[f].tx * TT.t[f].ty * (size_t)P.fr[f].n[2];
  return n;
}

// sub-lists per brick for chunks of up to vpc views: about 8 blocks of k_prep per SM of a 148-SM part
int prep_sub_for(int vpc) {
  const int s = (8 * 148 + 3 * vpc - 1) / (3 * (vpc > 0 ? vpc : 1));
  return s < kPrepSubMin ? kPrepSubMin : (s > kPrepSubMax ? kPrepSubMax : s);
}

size_t fixed_bytes(const EmuDev& P, const Tilings& TT, int64_t n_grains, int32_t n_views, int vpc) {
  size_t b = 0;
  b += emu_align256((size_t)n_views * sizeof(EmuBox));
  b += 2 * emu_align256((size_t)n_grains * sizeof(unsigned long long));
  b += emu_align256((size_t)n_grains * sizeof(unsigned));                   // owner
  b += emu_align256(3 * (size_t)n_grains * sizeof(unsigned));               // seed_off, one plane per frame
  b += emu_align256(sizeof(FindCtl)) + emu_align256(kTieBits / 8) + 256;
  b += 6 * emu_align256((3 * (size_t)vpc + 1) * sizeof(unsigned));
  b += emu_align256(3 * (size_t)vpc * kRecBricks * sizeof(int));            // vf_brick_base
  b += emu_align256(3 * (size_t)n_grains * sizeof(int));                    // slot_row: every grain once per frame
  b += emu_align256((size_t)vpc * sizeof(int));
  b += emu_align256((size_t)vpc * P.max_tracks * sizeof(unsigned));
  if (P.angle_cut) b += emu_align256((size_t)vpc * P.max_tracks * sizeof(CutAcc));
  b += emu_align256((size_t)vpc * bricks_per_view(P, TT) * sizeof(Brick));
  b += emu_align256(3 * (size_t)vpc * sizeof(int2));                        // vf_bricks
  b += 2 * emu_align256(((size_t)vpc * bricks_per_view(P, TT) * prep_sub_for(vpc) + 1) * sizeof(unsigned));   // brick_cnt, brick_off
  for (int f = 1; f < 3; ++f) {                                             // the binnings of frames 1 and 2
    b += emu_align256((size_t)n_grains * sizeof(int4));
    b += emu_align256(((size_t)n_views * P.fr[f].ncell + 1) * sizeof(int));
  }
  b += emu_align256(emu_bin_ws_bytes(P, n_grains, n_views));
  return b + 256;
}

// Tiles per (view, frame): the fewest tiles (every seed is streamed past every brick of its view and frame)
// for which an average tile - 1.35 x its share of the grains, its rows and its cells over the whole w extent -
// fits the shared-memory pool; among the factorisations of that count the squarest in physical size.
// k_plan cuts a tile that turns out too full into runs of w layers.
Tiling choose_tiling(const EmuDev& P, int f, int64_t n_grains, int32_t n_views) {
  const int* n = P.fr[f].n;
  const double avg = n_views > 0 ? (double)n_grains / n_views : 0.0;
  Tiling fallback; fallback.tx = n[0]; fallback.ty = n[1]; fallback.w = 1; fallback.h = 1;   // one column per tile
  const int64_t max_t = emu_min64((int64_t)n[0] * n[1], 8192);
  {   // frames 0 and 1 (w = z, the thin axis of a view): one tile, cut by k_plan into runs of w layers, whenever a
      // single layer fits - a long line is nearly level and stays inside one or two such slabs (measured: 2 % faster)
    const double grains = 1.35 * avg / (double)n[2] + 64.0;
    if (f != 2 && brick_bytes((long long)grains, (long long)n[1], n[0]) <= kPoolBytes) {
      Tiling one; one.tx = 1; one.ty = 1; one.w = n[0]; one.h = n[1];
      return one;
    }
  }
  for (int64_t t = 1; t <= max_t; ++t) {
    Tiling best; best.tx = best.ty = best.w = best.h = 0;
    double best_score = -1.0;
    for (int64_t tx = 1; tx <= t; ++tx) {
      if (t % tx) continue;
      const int64_t ty = t / tx;
      if (tx > n[0] || ty > n[1]) continue;
      const int w = (int)((n[0] + tx - 1) / tx), h = (int)((n[1] + ty - 1) / ty);
      const double grains = 1.35 * avg * ((double)w * h) / ((double)n[0] * n[1]) + 64.0;
      if (brick_bytes((long long)grains, (long long)h * n[2], w) > kPoolBytes) continue;
      const double sx = (double)w * P.cs[0], sy = (double)h * P.cs[1];
      const double score = sx < sy ? sx / sy : sy / sx;
      if (score > best_score) { best_score = score; best.tx = (int)tx; best.ty = (int)ty; best.w = w; best.h = h; }
    }
    if (best_score >= 0.0) return best;
  }
  return fallback;
}

Tilings choose_tilings(const EmuDev& P, int64_t n_grains, int32_t n_views) {
  Tilings TT;
  for (int f = 0; f < 3; ++f) TT.t[f] = choose_tiling(P, f, n_grains, n_views);
  return TT;
}

struct Hints { int seeds_per_grain, cand_per_grain; };

}  // namespace

size_t emu_find_ws_min_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views) {
  Tilings TT = choose_tilings(P, n_grains, n_views);
  return fixed_bytes(P, TT, n_grains, n_views, 1) + kMinSeedCap * kSeedBytes + kMinCandCap * kCandBytes + 8 * 256;
}

size_t emu_find_ws_recommended_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views, int seeds_per_grain,
                                     int cand_per_grain) {
  Tilings TT = choose_tilings(P, n_grains, n_views);
  const int64_t per_view_g = emu_max64(1, (n_grains + emu_max64(1, n_views) - 1) / emu_max64(1, n_views));
  const int64_t spv = per_view_g * seeds_per_grain, cpv = per_view_g * cand_per_grain;
  const int64_t per_view_bytes = spv * (int64_t)kSeedBytes + cpv * (int64_t)kCandBytes;
  // as many views per chunk as fit EMU_CHUNK_GIB (96) GiB of seed / candidate storage (at least one)
  int64_t vpc = emu_max64(1, emu_min64(emu_max64(1, n_views), ((int64_t)EMU_CHUNK_GIB << 30) / emu_max64(1, per_view_bytes)));
  vpc = emu_min64(vpc, 21000);
  const size_t seed_cap = (size_t)emu_max64((int64_t)kMinSeedCap, spv * vpc);
  const size_t cand_cap = (size_t)emu_max64((int64_t)kMinCandCap, cpv * vpc);
  return fixed_bytes(P, TT, n_grains, n_views, (int)vpc) + seed_cap * kSeedBytes + cand_cap * kCandBytes + 16 * 256;
}

static int carve(const EmuDev& P, const Tilings& TT, Hints hints, int64_t n_grains, int32_t n_views, void* d_ws,
                 size_t ws_bytes, FindWs& W) {
  if (ws_bytes < emu_find_ws_min_bytes(P, n_grains, n_views)) return EMU_ERR_CAPACITY;
  const int64_t per_view_g = emu_max64(1, (n_grains + emu_max64(1, n_views) - 1) / emu_max64(1, n_views));
  const int64_t spv = per_view_g * hints.seeds_per_grain, cpv = per_view_g * hints.cand_per_grain;
  // views per chunk: the most whose expected seeds and candidates fit what is left after the fixed part
  // (3 groups per view must fit the 65 535 blocks of grid.y)
  size_t seed_cap = 0, cand_cap = 0;
  auto fits = [&](int vpc, bool relaxed) {
    const size_t fx = fixed_bytes(P, TT, n_grains, n_views, vpc) + 16 * 256;
    if (fx + kMinSeedCap * kSeedBytes + kMinCandCap * kCandBytes > ws_bytes) return false;
    const size_t avail = ws_bytes - fx;
    // what is available is split between seeds and candidates in the proportion of the hints
    const double ws_seed = (double)spv * kSeedBytes, ws_cand = (double)cpv * kCandBytes;
    seed_cap = (size_t)((double)avail * ws_seed / (ws_seed + ws_cand) / kSeedBytes);
    const size_t seed_max = (avail - kMinCandCap * kCandBytes) / kSeedBytes;     // leave the candidates their minimum
    if (seed_cap > seed_max) seed_cap = seed_max;
    if (seed_cap < kMinSeedCap) seed_cap = kMinSeedCap;
    cand_cap = (avail - seed_cap * kSeedBytes) / kCandBytes;
    return cand_cap >= kMinCandCap && ((int64_t)seed_cap >= spv * vpc || relaxed);
  };
  int lo = 1, hi = n_views > 0 ? (int)emu_min64(n_views, 21000) : 1;
  if (!fits(1, true)) return EMU_ERR_CAPACITY;
  while (lo < hi) {                                   // the largest chunk that fits (the predicate is monotone)
    const int mid = lo + (hi - lo + 1) / 2;
    if (fits(mid, false)) lo = mid; else hi = mid - 1;
  }
  const int vpc = lo;
  fits(vpc, vpc == 1);                                // sets seed_cap / cand_cap for the chunk size chosen
  if (cand_cap > (size_t)kCiMask) cand_cap = kCiMask;
  if (seed_cap > (size_t)0x7fffffff) seed_cap = 0x7fffffff;
  char* p = (char*)emu_align_ptr(d_ws);
  auto take = [&](size_t bytes) { char* r = p; p += emu_align256(bytes); return r; };
  W.bbox = (EmuBox*)take((size_t)n_views * sizeof(EmuBox));
  W.keyA = (unsigned long long*)take((size_t)n_grains * sizeof(unsigned long long));
  W.keyB = (unsigned long long*)take((size_t)n_grains * sizeof(unsigned long long));
  W.owner = (unsigned*)take((size_t)n_grains * sizeof(unsigned));
  W.seed_off = (unsigned*)take(3 * (size_t)n_grains * sizeof(unsigned));
  W.ctl = (FindCtl*)take(sizeof(FindCtl));
  W.tie_bits = (unsigned*)take(kTieBits / 8);
  W.dump_cursor = (unsigned long long*)take(256);
  W.view_seed_tot = (unsigned*)take((3 * (size_t)vpc + 1) * sizeof(unsigned));
  W.view_seed_off = (unsigned*)take((3 * (size_t)vpc + 1) * sizeof(unsigned));
  W.view_cand_cnt = (unsigned*)take((3 * (size_t)vpc + 1) * sizeof(unsigned));
  W.view_cand_off = (unsigned*)take((3 * (size_t)vpc + 1) * sizeof(unsigned));
  W.view_ovf_cnt = (unsigned*)take((3 * (size_t)vpc + 1) * sizeof(unsigned));
  W.view_ovf_off = (unsigned*)take((3 * (size_t)vpc + 1) * sizeof(unsigned));
  W.vf_brick_base = (int*)take(3 * (size_t)vpc * kRecBricks * sizeof(int));
  W.slot_row = (int*)take(3 * (size_t)n_grains * sizeof(int));
  W.view_ntracks = (int*)take((size_t)vpc * sizeof(int));
  W.view_tracks = (unsigned*)take((size_t)vpc * P.max_tracks * sizeof(unsigned));
  W.cut_acc = P.angle_cut ? (CutAcc*)take((size_t)vpc * P.max_tracks * sizeof(CutAcc)) : nullptr;
  W.brick_cap = (size_t)vpc * bricks_per_view(P, TT);
  W.bricks = (Brick*)take(W.brick_cap * sizeof(Brick));
  W.vf_bricks = (int2*)take(3 * (size_t)vpc * sizeof(int2));
  W.prep_sub = prep_sub_for(vpc);
  W.brick_cnt = (unsigned*)take((W.brick_cap * W.prep_sub + 1) * sizeof(unsigned));
  W.brick_off = (unsigned*)take((W.brick_cap * W.prep_sub + 1) * sizeof(unsigned));
  W.sortedF[0] = nullptr; W.cell_startF[0] = nullptr;
  for (int f = 1; f < 3; ++f) {
    W.sortedF[f] = (int4*)take((size_t)n_grains * sizeof(int4));
    W.cell_startF[f] = (int*)take(((size_t)n_views * P.fr[f].ncell + 1) * sizeof(int));
  }
  W.bin_ws_bytes = emu_bin_ws_bytes(P, n_grains, n_views);
  W.bin_ws = take(W.bin_ws_bytes);
  W.geo = (int4*)take(seed_cap * sizeof(int4));
  W.ab = (int2*)take(seed_cap * sizeof(int2));
  W.seed_cnt = (unsigned long long*)take(seed_cap * sizeof(unsigned long long));
  W.recs = (unsigned short*)take(seed_cap * kRecBytes);
  W.prep_cap = (size_t)emu_min64((int64_t)(seed_cap * kPrepPerSeed8 / 8), 0xfffffff0ll);
  W.prec = (PrepRec*)take(W.prep_cap * sizeof(PrepRec));
  W.cands = (Cand*)take(cand_cap * sizeof(Cand));
  W.cand_seed = (unsigned*)take(cand_cap * sizeof(unsigned));
  W.ovf_geo = (int4*)take(cand_cap * sizeof(int4));
  W.ovf_ci = (unsigned*)take(cand_cap * sizeof(unsigned));
  W.wins = (int*)take(cand_cap * sizeof(int));
  W.cand_track = (unsigned*)take(cand_cap * sizeof(unsigned));
  W.seed_cap = seed_cap; W.cand_cap = cand_cap; W.views_per_chunk = vpc;
  return EMU_OK;
}

static int grid_for(int64_t n, int threads, int max_blocks) {
  int64_t b = (n + threads - 1) / threads;
  if (b < 1) b = 1;
  return (int)emu_min64(b, max_blocks);
}


#define EMU_CK(x) do { if ((x) != cudaSuccess) return EMU_ERR_CUDA; } while (0)

static int choose_slices(const Tilings& TT, int nv, int n_sm, int per_sm, int64_t chunk_grains, int entries_per_grain,
                         int min_entries = 2048) {
  // Work items = bricks x slices of a brick's list.  A big chunk wants fine items (per_sm of them per SM: short tail);
  // a small one must not be cut finer than its work pays for - an item stages its brick and drains its lanes once:
  // at least one item per SM if that leaves about min_entries list entries per item, items of 16 Ki entries beyond
  // that.  (A single config-1 view: 768 items of 1 900 seeds took 1.02 ms, 150 items of 10 k take 0.52; config 0:
  // 0.31 -> 0.09 ms.)  The lists are counted on the device; the host plans with entries_per_grain per grain.
  int64_t bricks = 0;
  for (int f = 0; f < 3; ++f) bricks += (int64_t)nv * TT.t[f].tx * TT.t[f].ty;
  bricks = emu_max64(1, bricks);
  const int64_t fine = (per_sm * (int64_t)n_sm + bricks - 1) / bricks;
  const int64_t wave = ((int64_t)n_sm + bricks - 1) / bricks;
  const int64_t per_brick = chunk_grains * entries_per_grain / bricks;
  int64_t s = emu_min64(fine, emu_max64(wave, per_brick / 16384));
  s = emu_min64(s, emu_max64(1, per_brick / min_entries));
  if (s < 1) s = 1;
  if (s > 256) s = 256;
  return (int)s;
}

// once per call: bounding boxes, and the binnings of frames 1 and 2 from frame 0's (the caller's) output
static int prepare_frames(const EmuDev& P, FindWs& W, FramePtrs& F, const int32_t* d_sorted, const int32_t* d_cell_start,
                          const int32_t* d_view_off, int64_t n_grains, int32_t n_views, int kSM, cudaStream_t st) {
  const int n = (int)n_grains;
  EMU_LAUNCH(EMU_STAGE_PREP, st, k_bbox_init<<<grid_for(n_views, 256, 1 << 20), 256, 0, st>>>(W.bbox, n_views));
  EMU_LAUNCH(EMU_STAGE_PREP, st, k_bbox<<<grid_for(n, 256, kSM * 8), 256, 0, st>>>((const int4*)d_sorted, d_view_off, n_views, n, W.bbox));
  F.sorted[0] = (const int4*)d_sorted; F.cell_start[0] = d_cell_start;
  for (int f = 1; f < 3; ++f) {
    F.sorted[f] = W.sortedF[f]; F.cell_start[f] = W.cell_startF[f];
    if (!P.packed_ok) continue;                        // every chunk will take the generic kernels (frame 0 only)
    int rc = emu_bin_launch(P, f, d_sorted, d_view_off, n_grains, n_views, (int32_t*)W.sortedF[f], W.cell_startF[f],
                            nullptr, W.bin_ws, W.bin_ws_bytes, st);
    if (rc != EMU_OK) return rc;
  }
  return EMU_OK;
}

// seeds + votes of the chunk [v0, v1): leaves geo / ab / seed_cnt / view_seed_off filled (brick path), or
// ctl->generic set
static int vote_chunk(const EmuDev& P, const Tilings& TT, FindWs& W, const FramePtrs& F, const int32_t* d_view_off,
                      int64_t n_grains, int v0, int v1, int slices, int kSM, unsigned long long* counts, cudaStream_t st) {
  const int nv = v1 - v0;
  const int4* sorted = F.sorted[0];
  const int* d_cell_start = F.cell_start[0];
  const size_t plane = (size_t)n_grains;
  EMU_CK(cudaMemsetAsync(W.ctl, 0, sizeof(FindCtl), st));
  EMU_CK(cudaMemsetAsync(W.view_cand_cnt, 0, (3 * (size_t)nv + 1) * sizeof(unsigned), st));
  EMU_LAUNCH(EMU_STAGE_SEEDS, st, k_seed_pairs<0><<<kSM * 16, kVoteThreads, 0, st>>>(
      P, sorted, d_cell_start, d_view_off, v0, v1, W.seed_off, plane, nullptr, W.ctl, nullptr, nullptr, counts));
  EMU_LAUNCH(EMU_STAGE_SEEDS, st, k_view_scan<<<grid_for(3 * nv, 1, kSM * 2), 1024, 0, st>>>(
      d_view_off, v0, v1, W.seed_off, plane, W.view_seed_tot, counts));
  EMU_LAUNCH(EMU_STAGE_SEEDS, st, k_chunk_offsets<<<1, 1024, 0, st>>>(
      3 * nv, W.view_seed_tot, W.view_seed_off, &W.ctl->seed_count, (unsigned)W.seed_cap, (unsigned)EMU_ST_SEED_OVERFLOW,
      W.ctl, counts, EMU_CNT_SEEDS, EMU_CNT_NEED, 1u, 1u));
  EMU_LAUNCH(EMU_STAGE_SEEDS, st, k_seed_pairs<1><<<kSM * 16, kVoteThreads, 0, st>>>(
      P, sorted, d_cell_start, d_view_off, v0, v1, W.seed_off, plane, W.view_seed_off, W.ctl, W.geo, W.ab, counts));
  // only the counters of the seeds this chunk has are cleared (the count is on the device)
  EMU_LAUNCH(EMU_STAGE_PREP, st, k_clear_seed_cnt<<<kSM * 8, 256, 0, st>>>(W.ctl, W.seed_cnt));
  EMU_LAUNCH(EMU_STAGE_PREP, st, k_plan<<<grid_for(3 * nv, 4, 1 << 20), 128, 0, st>>>(
      P, TT, F, W.bbox, v0, v1, W.bricks, (unsigned)W.brick_cap, W.vf_brick_base, W.vf_bricks, W.ctl));
  EMU_LAUNCH(EMU_STAGE_PREP, st, k_plan_finish<<<1, 1, 0, st>>>(W.ctl, (unsigned)W.brick_cap));
  // per-brick lists of prepared seeds: count, scan over the bricks, fill
  const dim3 gp(W.prep_sub, 3 * nv);
  EMU_CK(cudaMemsetAsync(W.brick_cnt, 0, (W.brick_cap * W.prep_sub + 1) * sizeof(unsigned), st));
  if (P.ext >= 0) EMU_LAUNCH(EMU_STAGE_SEEDS, st, k_prep<0, true><<<gp, 256, 0, st>>>(P, W.ctl, W.view_seed_off, W.geo, W.bricks, W.vf_bricks, W.brick_cnt, nullptr, nullptr));
  else EMU_LAUNCH(EMU_STAGE_SEEDS, st, k_prep<0, false><<<gp, 256, 0, st>>>(P, W.ctl, W.view_seed_off, W.geo, W.bricks, W.vf_bricks, W.brick_cnt, nullptr, nullptr));
  EMU_LAUNCH(EMU_STAGE_SEEDS, st, k_chunk_offsets<<<1, 1024, 0, st>>>(
      (int)(W.brick_cap * W.prep_sub), W.brick_cnt, W.brick_off, &W.ctl->prep_count, (unsigned)W.prep_cap, (unsigned)EMU_ST_SEED_OVERFLOW,
      W.ctl, counts, -1, EMU_CNT_NEED, 8u, (unsigned)kPrepPerSeed8));      // prep_cap = seed_cap * kPrepPerSeed8 / 8: NEED is in seeds
  EMU_CK(cudaMemsetAsync(W.brick_cnt, 0, (W.brick_cap * W.prep_sub + 1) * sizeof(unsigned), st));
  if (P.ext >= 0) EMU_LAUNCH(EMU_STAGE_SEEDS, st, k_prep<1, true><<<gp, 256, 0, st>>>(P, W.ctl, W.view_seed_off, W.geo, W.bricks, W.vf_bricks, W.brick_cnt, W.brick_off, W.prec));
  else EMU_LAUNCH(EMU_STAGE_SEEDS, st, k_prep<1, false><<<gp, 256, 0, st>>>(P, W.ctl, W.view_seed_off, W.geo, W.bricks, W.vf_bricks, W.brick_cnt, W.brick_off, W.prec));
  auto vote_kernel = P.ext >= 0 ? k_brick<kVote, true> : k_brick<kVote, false>;
  EMU_CK(cudaFuncSetAttribute(vote_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kPoolBytes));
  EMU_LAUNCH(EMU_STAGE_VOTE, st, vote_kernel<<<kSM, kBrickThreads, kPoolBytes, st>>>(
      P, F, v0, W.bricks, W.ctl, slices, W.geo, nullptr, W.view_seed_off, W.prec, W.brick_off, W.prep_sub, W.seed_cnt, W.recs, W.slot_row, nullptr,
      nullptr, counts));
  return EMU_OK;
}

int emu_find_launch(const EmuDev& P, int seeds_per_grain, int cand_per_grain, const int32_t* d_sorted,
                    const int32_t* d_cell_start, const int32_t* d_view_off, int64_t n_grains, int32_t n_views,
                    emu_track* d_tracks, int32_t* d_track_off, int32_t* d_members, int64_t members_capacity,
                    int64_t* d_counts, void* d_ws, size_t ws_bytes, cudaStream_t st) {
  FindWs W;
  const Tilings TT = choose_tilings(P, n_grains, n_views);
  Hints hints; hints.seeds_per_grain = seeds_per_grain; hints.cand_per_grain = cand_per_grain;
  int rc = carve(P, TT, hints, n_grains, n_views, d_ws, ws_bytes, W);
  if (rc != EMU_OK) return rc;
  const int4* sorted = (const int4*)d_sorted;
  unsigned long long* counts = (unsigned long long*)d_counts;
  const int kSM = emu_sm_count();
  EMU_CK(cudaMemsetAsync(d_counts, 0, 8 * sizeof(int64_t), st));
  EMU_CK(cudaMemsetAsync(d_track_off, 0, ((size_t)n_views + 1) * sizeof(int32_t), st));
  EMU_CK(cudaMemsetAsync(W.keyA, 0, (size_t)n_grains * sizeof(unsigned long long), st));
  EMU_CK(cudaMemsetAsync(W.keyB, 0, (size_t)n_grains * sizeof(unsigned long long), st));
  EMU_CK(cudaMemsetAsync(W.owner, 0xff, (size_t)n_grains * sizeof(unsigned), st));
  FramePtrs F;
  rc = prepare_frames(P, W, F, d_sorted, d_cell_start, d_view_off, n_grains, n_views, kSM, st);
  if (rc != EMU_OK) return rc;

  for (int v0 = 0; v0 < n_views; v0 += W.views_per_chunk) {
    const int v1 = (int)emu_min64(n_views, (int64_t)v0 + W.views_per_chunk);
    const int nv = v1 - v0;
    // (host copies of view_off are not available: the chunk's grains are taken as its share of the batch)
    const int64_t chunk_grains = n_views > 0 ? n_grains * nv / n_views : 0;
    const int slices = choose_slices(TT, nv, kSM, EMU_ITEMS_PER_SM, chunk_grains, 64);   // the voting pass: fine items, short tail
    const int slices_walk = choose_slices(TT, nv, kSM, 4, chunk_grains, 1);              // the walk list is short: staging would dominate
    EMU_CK(cudaMemsetAsync(W.view_ntracks, 0, (size_t)nv * sizeof(int), st));
    EMU_CK(cudaMemsetAsync(W.tie_bits, 0, kTieBits / 8, st));
    rc = vote_chunk(P, TT, W, F, d_view_off, n_grains, v0, v1, slices, kSM, counts, st);
    if (rc != EMU_OK) return rc;
    // A4: candidates grouped by (view, frame)
    EMU_CK(cudaMemsetAsync(W.view_ovf_cnt, 0, (3 * (size_t)nv + 1) * sizeof(unsigned), st));
    const int gx = (int)emu_max64(16, emu_min64(512, (4 * kSM + 3 * nv - 1) / (3 * nv)));   // blocks per (view, frame): few views still fill the GPU
    EMU_LAUNCH(EMU_STAGE_CANDS, st, k_cands<0><<<dim3(gx, 3 * nv), 256, 0, st>>>(
        P, v0, W.ctl, W.view_seed_off, W.seed_cnt, W.geo, W.ab, W.view_cand_cnt, nullptr, W.view_ovf_cnt, nullptr,
        nullptr, nullptr, nullptr, nullptr, counts));
    EMU_LAUNCH(EMU_STAGE_CANDS, st, k_chunk_offsets<<<1, 1024, 0, st>>>(
        3 * nv, W.view_cand_cnt, W.view_cand_off, &W.ctl->cand_count, (unsigned)W.cand_cap, (unsigned)EMU_ST_CAND_OVERFLOW,
        W.ctl, counts, EMU_CNT_CANDIDATES, -1, 1u, 1u));
    EMU_LAUNCH(EMU_STAGE_CANDS, st, k_chunk_offsets<<<1, 1024, 0, st>>>(
        3 * nv, W.view_ovf_cnt, W.view_ovf_off, &W.ctl->ovf_count, (unsigned)W.cand_cap, (unsigned)EMU_ST_CAND_OVERFLOW,
        W.ctl, counts, -1, -1, 1u, 1u));
    EMU_CK(cudaMemsetAsync(W.view_cand_cnt, 0, (3 * (size_t)nv + 1) * sizeof(unsigned), st));
    EMU_CK(cudaMemsetAsync(W.view_ovf_cnt, 0, (3 * (size_t)nv + 1) * sizeof(unsigned), st));
    EMU_LAUNCH(EMU_STAGE_CANDS, st, k_cands<1><<<dim3(gx, 3 * nv), 256, 0, st>>>(
        P, v0, W.ctl, W.view_seed_off, W.seed_cnt, W.geo, W.ab, W.view_cand_cnt, W.view_cand_off, W.view_ovf_cnt,
        W.view_ovf_off, W.cands, W.cand_seed, W.ovf_geo, W.ovf_ci, counts));
    // generic fallback for the whole chunk (returns at once unless the brick plan failed)
    EMU_LAUNCH(EMU_STAGE_GENERIC, st, k_vote_generic<false><<<kSM * 16, kVoteThreads, 0, st>>>(
        P, sorted, d_cell_start, d_view_off, W.bbox, v0, v1, W.cands, (unsigned)W.cand_cap, W.ctl, nullptr, 0, nullptr,
        counts));
    EMU_LAUNCH(EMU_STAGE_PREP, st, k_cands_finish<<<1, 1, 0, st>>>(W.ctl, (unsigned)W.cand_cap, counts));
    EMU_LAUNCH(EMU_STAGE_PREP, st, k_reset_cand_arrays<<<kSM * 8, 256, 0, st>>>(W.ctl, W.wins, W.cand_track));
    // A5
    auto walk_kernel = P.ext >= 0 ? k_brick<kAssoc, true> : k_brick<kAssoc, false>;
    EMU_CK(cudaFuncSetAttribute(walk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kPoolBytes));
    EMU_LAUNCH(EMU_STAGE_ASSOC, st, k_assoc_hits<<<dim3(emu_max64(48, gx), 3 * nv), 256, 0, st>>>(
        v0, W.ctl, W.view_cand_off, W.cands, W.cand_seed, W.seed_cnt, W.recs, W.slot_row, W.vf_brick_base, W.keyA, W.keyB));
    EMU_LAUNCH(EMU_STAGE_ASSOC, st, walk_kernel<<<kSM, kBrickThreads, kPoolBytes, st>>>(
        P, F, v0, W.bricks, W.ctl, slices_walk, W.ovf_geo, W.ovf_ci, W.view_ovf_off, nullptr, nullptr, 1, nullptr, nullptr, nullptr, W.keyA, W.keyB,
        counts));
    EMU_LAUNCH(EMU_STAGE_ASSOC, st, k_assoc_generic<0><<<kSM * 16, kVoteThreads, 0, st>>>(
        P, sorted, d_cell_start, W.bbox, v0, W.cands, W.ctl, W.tie_bits, W.keyA, W.keyB, W.owner));
    EMU_LAUNCH(EMU_STAGE_ASSOC, st, k_tie_detect<<<kSM * 4, 256, 0, st>>>(d_view_off, v0, v1, W.keyA, W.keyB, W.ctl, W.tie_bits));
    EMU_LAUNCH(EMU_STAGE_ASSOC, st, k_assoc_generic<1><<<kSM * 16, kVoteThreads, 0, st>>>(
        P, sorted, d_cell_start, W.bbox, v0, W.cands, W.ctl, W.tie_bits, W.keyA, W.keyB, W.owner));
    EMU_LAUNCH(EMU_STAGE_SELECT, st, k_wins<<<kSM * 4, 256, 0, st>>>(d_view_off, v0, v1, W.ctl, W.keyA, W.keyB, W.owner, W.wins));
    EMU_LAUNCH(EMU_STAGE_SELECT, st, k_select<<<kSM * 8, 256, 0, st>>>(P, W.cands, W.ctl, W.wins, W.view_ntracks, W.view_tracks, W.cand_track, counts));
    if (P.angle_cut) {                                           // A5b: angle-dependent cut on the number of grains
      const dim3 gv(4, nv);
      EMU_LAUNCH(EMU_STAGE_SELECT, st, k_cut_init<<<gv, 256, 0, st>>>(P, nv, W.ctl, W.view_ntracks, W.cut_acc));
      EMU_LAUNCH(EMU_STAGE_SELECT, st, k_cut_acc<<<kSM * 4, 256, 0, st>>>(
          P, sorted, d_view_off, v0, v1, W.ctl, W.keyA, W.keyB, W.owner, W.cands, W.cand_track, W.cut_acc));
      EMU_LAUNCH(EMU_STAGE_SELECT, st, k_cut_decide<<<gv, 256, 0, st>>>(P, nv, W.ctl, W.view_ntracks, W.view_tracks, W.wins, W.cut_acc, W.cand_track));
      EMU_LAUNCH(EMU_STAGE_SELECT, st, k_cut_compact<<<grid_for(nv, 1, kSM * 8), 256, 0, st>>>(P, nv, W.ctl, W.view_ntracks, W.view_tracks));
    }
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_track_scan<<<1, 1024, 0, st>>>(P, v0, v1, W.view_ntracks, d_track_off));
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_track_emit<<<dim3((unsigned)emu_max64(1, emu_min64(16, (2 * kSM + nv - 1) / nv)), (unsigned)emu_min64(nv, 65535)), 256, 0, st>>>(
        P, sorted, v0, v1, W.cands, W.wins, W.view_ntracks, W.view_tracks, d_track_off, d_tracks, W.cand_track));
    // the per-track fill cursors reuse view_tracks (its contents are dead after k_track_emit)
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_member_scan<<<1, 1024, 0, st>>>(v0, v1, d_track_off, d_tracks, (int*)W.view_tracks, counts, members_capacity));
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_member_scatter<<<kSM * 4, 256, 0, st>>>(
        sorted, d_view_off, v0, v1, W.ctl, W.keyA, W.keyB, W.owner, W.cand_track, d_track_off, d_tracks, (int*)W.view_tracks,
        d_members, members_capacity));
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_member_sort<<<kSM * 4, 256, 0, st>>>(v0, v1, d_track_off, d_tracks, d_members, members_capacity));
  }
  return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
}

int emu_count_seeds_launch(const EmuDev& P, int seeds_per_grain, int cand_per_grain, const int32_t* d_sorted,
                           const int32_t* d_cell_start, const int32_t* d_view_off, int64_t n_grains, int32_t n_views,
                           int32_t* d_seed_dump, int64_t dump_capacity, int64_t* d_counts, void* d_ws, size_t ws_bytes,
                           cudaStream_t st) {
  FindWs W;
  const Tilings TT = choose_tilings(P, n_grains, n_views);
  Hints hints; hints.seeds_per_grain = seeds_per_grain; hints.cand_per_grain = cand_per_grain;
  int rc = carve(P, TT, hints, n_grains, n_views, d_ws, ws_bytes, W);
  if (rc != EMU_OK) return rc;
  if (W.views_per_chunk < n_views) return EMU_ERR_CAPACITY;      // the per-seed dump is a one-chunk test aid
  const int4* sorted = (const int4*)d_sorted;
  unsigned long long* counts = (unsigned long long*)d_counts;
  const int kSM = emu_sm_count();
  EMU_CK(cudaMemsetAsync(d_counts, 0, 8 * sizeof(int64_t), st));
  EMU_CK(cudaMemsetAsync(W.dump_cursor, 0, 256, st));
  FramePtrs F;
  rc = prepare_frames(P, W, F, d_sorted, d_cell_start, d_view_off, n_grains, n_views, kSM, st);
  if (rc != EMU_OK) return rc;
  if (n_views > 0) {
    rc = vote_chunk(P, TT, W, F, d_view_off, n_grains, 0, n_views, choose_slices(TT, n_views, kSM, EMU_ITEMS_PER_SM, n_grains, 64), kSM, counts, st);
    if (rc != EMU_OK) return rc;
    EMU_LAUNCH(EMU_STAGE_CANDS, st, k_seed_dump<<<dim3(64, 3 * n_views), 256, 0, st>>>(
        0, W.ctl, sorted, W.view_seed_off, W.seed_cnt, W.ab, (int4*)d_seed_dump, dump_capacity));
    EMU_LAUNCH(EMU_STAGE_GENERIC, st, k_vote_generic<true><<<kSM * 16, kVoteThreads, 0, st>>>(
        P, sorted, d_cell_start, d_view_off, W.bbox, 0, n_views, nullptr, 0, W.ctl, (int4*)d_seed_dump, dump_capacity,
        W.dump_cursor, counts));
  }
  return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
}
