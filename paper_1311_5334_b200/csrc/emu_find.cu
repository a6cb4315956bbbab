// emu_find.cu - A2..A5 + A7: seeds, tube vote, threshold, exclusive association, threshold, order.
// (P:72 and Fig. 4; readings Q1-Q8, Q15 in DESIGN.md section 3.)
//
// Views are processed in chunks sized by the candidate workspace.  Per chunk:
//   k_vote        every seed of the chunk: walk its tube, count; n_tube >= min -> candidate list
//   k_assoc_max   every candidate: walk again, atomicMax a packed priority into each member grain
//   k_tie_detect  does any grain see two different top candidates with equal (n_tube, D2)?
//   k_assoc_tie   (only then) every candidate: walk, settle the ties by (kmin, kmax) with a CAS-min
//   k_wins        every grain: +1 for its owner
//   k_select      every candidate: wins >= min -> per-view track list
//   k_track_scan / k_track_emit / k_member_scan / k_member_scatter / k_member_sort: ordered output
// Everything is a max / min / sum over a total order, so the result does not depend on the order in
// which threads run (reading Q7: "one-shot, order-free").
#include "emu_dev.cuh"
#include "emu_host.h"

namespace {

constexpr int kVoteThreads = 128;
constexpr int kCiBits = 29;                       // candidate index inside a chunk
constexpr unsigned kCiMask = (1u << kCiBits) - 1u;
constexpr unsigned kNone = 0xffffffffu;
constexpr int kMaxTube = 8191;                    // n_tube field of the packed priority: 13 bits

struct Cand {            // 16 B
  int a, b;              // sorted positions of the seed grains, a < b
  int n_tube_view;       // n_tube | (view - v0) << 16
  int d2;
};

struct FindCtl {         // device scalars of one emu_find_tracks call
  unsigned cand_count;   // candidates of the current chunk
  unsigned tie;          // 1 if the current chunk has a priority tie on some grain
  unsigned pad[2];
};

__device__ __forceinline__ unsigned long long cand_k1(int n_tube, int d2) {
  return ((unsigned long long)min(n_tube, kMaxTube) << 22) | (unsigned long long)(unsigned)d2;
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
// A2 + A3 + A4.  One warp per grain A: the lanes scan the cells around A for partners B behind A in
// sorted order (each unordered pair once, reading Q2), queue the pairs inside the separation window
// (reading Q1), and then every lane walks the tube of one queued seed.
template <bool kDump>
__global__ void __launch_bounds__(kVoteThreads)
k_vote(EmuDev P, const int4* __restrict__ sorted, const int* __restrict__ cell_start,
       const int* __restrict__ view_off, const EmuBox* __restrict__ bbox, int v0, int v1,
       Cand* __restrict__ cands, unsigned cand_cap, FindCtl* __restrict__ ctl,
       int4* __restrict__ dump, long long dump_cap, unsigned long long* __restrict__ counts) {
  __shared__ int queue_s[kVoteThreads / 32][64];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  int* queue = queue_s[wib];
  const int nwarps = gridDim.x * (kVoteThreads / 32);
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  unsigned long long n_tests = 0, n_pairs = 0, n_seeds = 0, n_cands = 0;
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
    const int czA = emu_cell_axis(A.z, P.cs[2], P.inv_cs[2], P.n[2]);   // partners behind A: cell >= cell(A)
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
      n_seeds += (b >= 0);
      if (kDump) {
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(counts + EMU_CNT_NEED, (unsigned long long)cnt);   // dump cursor
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
            // |d| can exceed 2^15 for far out-of-box grains: compare in 64 bits
            long long d2 = (long long)dx * dx + (long long)dy * dy + (long long)dz * dz;
            ok = (d2 >= P.sep_min2) && (d2 < P.sep_max2);
            ++n_pairs;
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

  // one set of atomics per warp
  for (int o = 16; o; o >>= 1) {
    n_tests += __shfl_xor_sync(EMU_FULL, n_tests, o);
    n_pairs += __shfl_xor_sync(EMU_FULL, n_pairs, o);
    n_seeds += __shfl_xor_sync(EMU_FULL, n_seeds, o);
    n_cands += __shfl_xor_sync(EMU_FULL, n_cands, o);
    status |= __shfl_xor_sync(EMU_FULL, status, o);
  }
  if (lane == 0) {
    atomicAdd(counts + EMU_CNT_SEEDS, n_seeds);
    atomicAdd(counts + EMU_CNT_TESTS, n_tests);
    atomicAdd(counts + EMU_CNT_PAIR_TESTS, n_pairs);
    atomicAdd(counts + EMU_CNT_CANDIDATES, n_cands);
    if (status) atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)status);
  }
}

// after k_vote: clamp the candidate count to the capacity and record overflow / need
__global__ void k_vote_finish(FindCtl* ctl, unsigned cand_cap, unsigned long long* counts) {
  unsigned n = ctl->cand_count;
  atomicMax(counts + EMU_CNT_NEED, (unsigned long long)n);
  if (n > cand_cap) { atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)EMU_ST_CAND_OVERFLOW); ctl->cand_count = cand_cap; }
  ctl->tie = 0;
}

// ---------------------------------------------------------------------------------------------
// A5 part 1: every member grain of every candidate receives max over candidates of
//   keyA = K1 << 29 | (mask - ci)   and   keyB = K1 << 29 | ci,   K1 = n_tube << 22 | D2.
// The top K1 of a grain is unique; keyA and keyB then name the same candidate unless several
// candidates tie on K1 for that grain (settled exactly in k_assoc_tie).
template <int kPass>
__global__ void __launch_bounds__(kVoteThreads)
k_assoc(EmuDev P, const int4* __restrict__ sorted, const int* __restrict__ cell_start,
        const EmuBox* __restrict__ bbox, int v0, const Cand* __restrict__ cands, const FindCtl* __restrict__ ctl,
        unsigned long long* __restrict__ keyA, unsigned long long* __restrict__ keyB,
        unsigned* __restrict__ owner) {
  if (kPass == 1 && ctl->tie == 0) return;
  const unsigned n = ctl->cand_count;
  const unsigned stride = gridDim.x * blockDim.x;
  for (unsigned ci = blockIdx.x * blockDim.x + threadIdx.x; ci < n; ci += stride) {
    const Cand c = cands[ci];
    const int v = v0 + (c.n_tube_view >> 16);
    const int4 A = __ldg(sorted + c.a), B = __ldg(sorted + c.b);
    const int dx = B.x - A.x, dy = B.y - A.y, dz = B.z - A.z;
    const unsigned long long k1 = cand_k1(c.n_tube_view & 0xffff, c.d2);
    const EmuBox bb = bbox[v];
    if (kPass == 0) {
      const unsigned long long ka = (k1 << kCiBits) | (unsigned long long)(kCiMask - ci);
      const unsigned long long kb = (k1 << kCiBits) | (unsigned long long)ci;
      emu_walk_tube(P, bb, sorted, cell_start, v * P.ncell, A.x, A.y, A.z, dx, dy, dz, (long long)P.r2 * c.d2,
                    [&](int g) { atomicMax(keyA + g, ka); atomicMax(keyB + g, kb); });
    } else {
      emu_walk_tube(P, bb, sorted, cell_start, v * P.ncell, A.x, A.y, A.z, dx, dy, dz, (long long)P.r2 * c.d2,
                    [&](int g) {
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

__global__ void __launch_bounds__(256)
k_tie_detect(const int* __restrict__ view_off, int v0, int v1, const unsigned long long* __restrict__ keyA,
             const unsigned long long* __restrict__ keyB, FindCtl* __restrict__ ctl) {
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  bool tie = false;
  for (int g = g0 + blockIdx.x * blockDim.x + threadIdx.x; g < g1; g += gridDim.x * blockDim.x) {
    unsigned long long ka = keyA[g], kb = keyB[g];
    if (ka) tie |= (kCiMask - (unsigned)(ka & kCiMask)) != (unsigned)(kb & kCiMask);
  }
  if (__any_sync(EMU_FULL, tie) && (threadIdx.x & 31) == 0) ctl->tie = 1;
}

__device__ __forceinline__ unsigned owner_of(int g, const FindCtl* ctl, const unsigned long long* keyA,
                                             const unsigned* owner) {
  unsigned long long ka = keyA[g];
  if (!ka) return kNone;
  return ctl->tie ? owner[g] : (kCiMask - (unsigned)(ka & kCiMask));
}

// A5 part 2: members won per candidate
__global__ void __launch_bounds__(256)
k_wins(const int* __restrict__ view_off, int v0, int v1, const FindCtl* __restrict__ ctl,
       const unsigned long long* __restrict__ keyA, const unsigned* __restrict__ owner, int* __restrict__ wins) {
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  for (int g = g0 + blockIdx.x * blockDim.x + threadIdx.x; g < g1; g += gridDim.x * blockDim.x) {
    unsigned ci = owner_of(g, ctl, keyA, owner);
    if (ci != kNone) atomicAdd(wins + ci, 1);
  }
}

// A5 part 3: "again the threshold on number of grains is applied to all tracks"
__global__ void __launch_bounds__(256)
k_select(EmuDev P, const Cand* __restrict__ cands, const FindCtl* __restrict__ ctl, const int* __restrict__ wins,
         int* __restrict__ view_ntracks, unsigned* __restrict__ view_tracks, unsigned long long* __restrict__ counts) {
  const unsigned n = ctl->cand_count;
  for (unsigned ci = blockIdx.x * blockDim.x + threadIdx.x; ci < n; ci += gridDim.x * blockDim.x) {
    if (wins[ci] >= P.min_grains) {
      int vl = cands[ci].n_tube_view >> 16;
      int slot = atomicAdd(view_ntracks + vl, 1);
      if (slot < P.max_tracks) view_tracks[(size_t)vl * P.max_tracks + slot] = ci;
      else atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)EMU_ST_TRACK_OVERFLOW);
    }
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
  for (int v = v0 + blockIdx.x; v < v1; v += gridDim.x) {
    const int nt = view_ntracks[v - v0];
    const unsigned* list = view_tracks + (size_t)(v - v0) * P.max_tracks;
    const int t0 = track_off[v];
    for (int i = threadIdx.x; i < nt; i += blockDim.x) {
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
      tracks[t].member_off = (int)off;
      cursor[t - t0] = 0;
      if (off + x > members_capacity) atomicOr(counts + EMU_CNT_STATUS, (unsigned long long)EMU_ST_MEMBER_OVERFLOW);
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
                 const unsigned* __restrict__ owner, const unsigned* __restrict__ cand_track,
                 const int* __restrict__ track_off, const emu_track* __restrict__ tracks,
                 int* __restrict__ cursor, int* __restrict__ members, long long members_capacity) {
  const int g0 = __ldg(view_off + v0), g1 = __ldg(view_off + v1);
  const int t0 = track_off[v0];
  for (int g = g0 + blockIdx.x * blockDim.x + threadIdx.x; g < g1; g += gridDim.x * blockDim.x) {
    unsigned ci = owner_of(g, ctl, keyA, owner);
    if (ci == kNone) continue;
    unsigned t = cand_track[ci];
    if (t == kNone) continue;
    int k = atomicAdd(cursor + (t - t0), 1);
    long long pos = (long long)tracks[t].member_off + k;
    if (pos < members_capacity) members[pos] = sorted[g].w;
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

struct FindWs {
  EmuBox* bbox; unsigned long long* keyA; unsigned long long* keyB; unsigned* owner; FindCtl* ctl;
  int* view_ntracks; unsigned* view_tracks; Cand* cands; int* wins; unsigned* cand_track;
  size_t cand_cap; int views_per_chunk;
};

size_t fixed_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views, int views_per_chunk) {
  size_t b = 0;
  b += emu_align256((size_t)n_views * sizeof(EmuBox));
  b += 2 * emu_align256((size_t)n_grains * sizeof(unsigned long long));
  b += emu_align256((size_t)n_grains * sizeof(unsigned));
  b += emu_align256(sizeof(FindCtl));
  b += emu_align256((size_t)views_per_chunk * sizeof(int));
  b += emu_align256((size_t)views_per_chunk * P.max_tracks * sizeof(unsigned));
  return b + 256;
}

constexpr size_t kCandBytes = sizeof(Cand) + sizeof(int) + sizeof(unsigned);
constexpr size_t kMinCandCap = 1u << 16;

}  // namespace

size_t emu_find_ws_min_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views) {
  return fixed_bytes(P, n_grains, n_views, 1) + kMinCandCap * kCandBytes + 3 * 256;
}

size_t emu_find_ws_recommended_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views, int cand_per_grain) {
  int64_t want = emu_max64((int64_t)kMinCandCap, emu_min64(n_grains * (int64_t)cand_per_grain, (int64_t)1 << 27));
  int64_t per_view = emu_max64(1, n_grains / emu_max64(1, n_views)) * cand_per_grain;
  int vpc = (int)emu_max64(1, emu_min64(n_views, want / emu_max64(1, per_view)));
  return fixed_bytes(P, n_grains, n_views, vpc) + (size_t)want * kCandBytes + 3 * 256;
}

static int carve(const EmuDev& P, int cand_per_grain, int64_t n_grains, int32_t n_views, void* d_ws, size_t ws_bytes,
                 FindWs& W) {
  if (ws_bytes < emu_find_ws_min_bytes(P, n_grains, n_views)) return EMU_ERR_CAPACITY;
  // choose views per chunk: as many as the candidate estimate allows in what is left after the fixed part
  int64_t per_view = emu_max64(1, n_grains / emu_max64(1, n_views)) * cand_per_grain;
  int vpc = n_views > 0 ? n_views : 1;
  size_t cap = 0;
  for (;;) {
    size_t fx = fixed_bytes(P, n_grains, n_views, vpc);
    if (fx + kMinCandCap * kCandBytes + 3 * 256 <= ws_bytes) {
      cap = (ws_bytes - fx - 3 * 256) / kCandBytes;
      if ((int64_t)cap >= per_view * vpc || vpc == 1) break;
    }
    if (vpc == 1) return EMU_ERR_CAPACITY;
    vpc = (vpc + 1) / 2;
  }
  if (cap > (size_t)kCiMask) cap = kCiMask;
  if (vpc > 65535) vpc = 65535;                      // view-in-chunk field of Cand: 16 bits
  char* p = (char*)emu_align_ptr(d_ws);
  auto take = [&](size_t bytes) { char* r = p; p += emu_align256(bytes); return r; };
  W.bbox = (EmuBox*)take((size_t)n_views * sizeof(EmuBox));
  W.keyA = (unsigned long long*)take((size_t)n_grains * sizeof(unsigned long long));
  W.keyB = (unsigned long long*)take((size_t)n_grains * sizeof(unsigned long long));
  W.owner = (unsigned*)take((size_t)n_grains * sizeof(unsigned));
  W.ctl = (FindCtl*)take(sizeof(FindCtl));
  W.view_ntracks = (int*)take((size_t)vpc * sizeof(int));
  W.view_tracks = (unsigned*)take((size_t)vpc * P.max_tracks * sizeof(unsigned));
  W.cands = (Cand*)take(cap * sizeof(Cand));
  W.wins = (int*)take(cap * sizeof(int));
  W.cand_track = (unsigned*)take(cap * sizeof(unsigned));
  W.cand_cap = cap; W.views_per_chunk = vpc;
  return EMU_OK;
}

static int grid_for(int64_t n, int threads, int max_blocks) {
  int64_t b = (n + threads - 1) / threads;
  if (b < 1) b = 1;
  return (int)emu_min64(b, max_blocks);
}

int emu_find_launch(const EmuDev& P, int cand_per_grain, const int32_t* d_sorted, const int32_t* d_cell_start,
                    const int32_t* d_view_off, int64_t n_grains, int32_t n_views, emu_track* d_tracks,
                    int32_t* d_track_off, int32_t* d_members, int64_t members_capacity, int64_t* d_counts,
                    void* d_ws, size_t ws_bytes, cudaStream_t st) {
  FindWs W;
  int rc = carve(P, cand_per_grain, n_grains, n_views, d_ws, ws_bytes, W);
  if (rc != EMU_OK) return rc;
  const int4* sorted = (const int4*)d_sorted;
  unsigned long long* counts = (unsigned long long*)d_counts;
  const int n = (int)n_grains;
  const int kSM = 148;
  if (cudaMemsetAsync(d_counts, 0, 8 * sizeof(int64_t), st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaMemsetAsync(d_track_off, 0, ((size_t)n_views + 1) * sizeof(int32_t), st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaMemsetAsync(W.keyA, 0, (size_t)n_grains * sizeof(unsigned long long), st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaMemsetAsync(W.keyB, 0, (size_t)n_grains * sizeof(unsigned long long), st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaMemsetAsync(W.owner, 0xff, (size_t)n_grains * sizeof(unsigned), st) != cudaSuccess) return EMU_ERR_CUDA;
  EMU_LAUNCH(EMU_STAGE_PREP, st, k_bbox_init<<<grid_for(n_views, 256, 1 << 20), 256, 0, st>>>(W.bbox, n_views));
  EMU_LAUNCH(EMU_STAGE_PREP, st, k_bbox<<<grid_for(n, 256, kSM * 8), 256, 0, st>>>(sorted, d_view_off, n_views, n, W.bbox));

  for (int v0 = 0; v0 < n_views; v0 += W.views_per_chunk) {
    const int v1 = (int)emu_min64(n_views, (int64_t)v0 + W.views_per_chunk);
    const int nv = v1 - v0;
    if (cudaMemsetAsync(W.ctl, 0, sizeof(FindCtl), st) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaMemsetAsync(W.view_ntracks, 0, (size_t)nv * sizeof(int), st) != cudaSuccess) return EMU_ERR_CUDA;
    EMU_LAUNCH(EMU_STAGE_VOTE, st, k_vote<false><<<kSM * 16, kVoteThreads, 0, st>>>(P, sorted, d_cell_start, d_view_off, W.bbox, v0, v1, W.cands,
                                                     (unsigned)W.cand_cap, W.ctl, nullptr, 0, counts));
    EMU_LAUNCH(EMU_STAGE_PREP, st, k_vote_finish<<<1, 1, 0, st>>>(W.ctl, (unsigned)W.cand_cap, counts));
    EMU_LAUNCH(EMU_STAGE_PREP, st, k_reset_cand_arrays<<<kSM * 8, 256, 0, st>>>(W.ctl, W.wins, W.cand_track));
    EMU_LAUNCH(EMU_STAGE_ASSOC, st, k_assoc<0><<<kSM * 16, kVoteThreads, 0, st>>>(P, sorted, d_cell_start, W.bbox, v0, W.cands, W.ctl, W.keyA, W.keyB, W.owner));
    EMU_LAUNCH(EMU_STAGE_ASSOC, st, k_tie_detect<<<kSM * 4, 256, 0, st>>>(d_view_off, v0, v1, W.keyA, W.keyB, W.ctl));
    EMU_LAUNCH(EMU_STAGE_ASSOC, st, k_assoc<1><<<kSM * 16, kVoteThreads, 0, st>>>(P, sorted, d_cell_start, W.bbox, v0, W.cands, W.ctl, W.keyA, W.keyB, W.owner));
    EMU_LAUNCH(EMU_STAGE_SELECT, st, k_wins<<<kSM * 4, 256, 0, st>>>(d_view_off, v0, v1, W.ctl, W.keyA, W.owner, W.wins));
    EMU_LAUNCH(EMU_STAGE_SELECT, st, k_select<<<kSM * 8, 256, 0, st>>>(P, W.cands, W.ctl, W.wins, W.view_ntracks, W.view_tracks, counts));
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_track_scan<<<1, 1024, 0, st>>>(P, v0, v1, W.view_ntracks, d_track_off));
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_track_emit<<<grid_for(nv, 1, kSM * 8), 256, 0, st>>>(P, sorted, v0, v1, W.cands, W.wins, W.view_ntracks,
                                                          W.view_tracks, d_track_off, d_tracks, W.cand_track));
    // the per-track fill cursors reuse view_tracks (its contents are dead after k_track_emit)
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_member_scan<<<1, 1024, 0, st>>>(v0, v1, d_track_off, d_tracks, (int*)W.view_tracks, counts, members_capacity));
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_member_scatter<<<kSM * 4, 256, 0, st>>>(sorted, d_view_off, v0, v1, W.ctl, W.keyA, W.owner, W.cand_track,
                                              d_track_off, d_tracks, (int*)W.view_tracks, d_members, members_capacity));
    EMU_LAUNCH(EMU_STAGE_EMIT, st, k_member_sort<<<kSM * 4, 256, 0, st>>>(v0, v1, d_track_off, d_tracks, d_members, members_capacity));
  }
  return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
}

int emu_count_seeds_launch(const EmuDev& P, const int32_t* d_sorted, const int32_t* d_cell_start,
                           const int32_t* d_view_off, int64_t n_grains, int32_t n_views, int32_t* d_seed_dump,
                           int64_t dump_capacity, int64_t* d_counts, void* d_ws, size_t ws_bytes, cudaStream_t st) {
  if (ws_bytes < emu_align256((size_t)n_views * sizeof(EmuBox)) + 256) return EMU_ERR_CAPACITY;
  EmuBox* bbox = (EmuBox*)emu_align_ptr(d_ws);
  const int n = (int)n_grains;
  if (cudaMemsetAsync(d_counts, 0, 8 * sizeof(int64_t), st) != cudaSuccess) return EMU_ERR_CUDA;
  EMU_LAUNCH(EMU_STAGE_PREP, st, k_bbox_init<<<grid_for(n_views, 256, 1 << 20), 256, 0, st>>>(bbox, n_views));
  EMU_LAUNCH(EMU_STAGE_PREP, st, k_bbox<<<grid_for(n, 256, 148 * 8), 256, 0, st>>>((const int4*)d_sorted, d_view_off, n_views, n, bbox));
  EMU_LAUNCH(EMU_STAGE_VOTE, st, k_vote<true><<<148 * 16, kVoteThreads, 0, st>>>(P, (const int4*)d_sorted, d_cell_start, d_view_off, bbox, 0, n_views,
                                                  nullptr, 0, nullptr, (int4*)d_seed_dump, dump_capacity,
                                                  (unsigned long long*)d_counts));
  return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
}
