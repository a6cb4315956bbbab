// emu_bin.cu - A1: attribute every grain to its 3D cell as a counting sort.
//   count (per-(view,cell) histogram) -> per-view exclusive scan -> scatter -> rank inside the cell.
// Output order is (view, cell, row): the canonical order SURVEY 8(c) O1 defines.
#include <stdlib.h>

#include "emu_dev.cuh"
#include "emu_host.h"

namespace {

constexpr int kBinThreads = 256;

// histogram: one thread per grain, int4 (16 B) coalesced loads
__global__ void __launch_bounds__(kBinThreads)
k_bin_count(EmuDev P, int frame, const int4* __restrict__ grains, const int* __restrict__ view_off, int n_views,
            int n_grains, int* __restrict__ count, unsigned long long* __restrict__ status) {
  const int ncell = P.fr[frame].ncell;
  int stride = gridDim.x * blockDim.x;
  bool bad = false;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_grains; i += stride) {
    int4 g = emu_to_frame(frame, __ldg(grains + i));
    int v = emu_find_view(view_off, 0, n_views, i);
    bad |= (abs(g.x) >= (1 << 17)) | (abs(g.y) >= (1 << 17)) | (abs(g.z) >= (1 << 17));
    atomicAdd(count + (size_t)v * ncell + emu_cell_of_frame(P, frame, g.x, g.y, g.z), 1);
  }
  if (status && __any_sync(EMU_FULL, bad) && (threadIdx.x & 31) == 0) atomicOr(status, (unsigned long long)EMU_ST_COORD);
}

// per-view exclusive scan of the cell counts: cell_start[v*ncell + c] = view_off[v] + #grains in cells < c
__global__ void __launch_bounds__(1024)
k_bin_scan(int ncell, const int* __restrict__ view_off, int n_views, int n_grains,
           const int* __restrict__ count, int* __restrict__ cell_start) {
  __shared__ int warp_sum[32];
  __shared__ int carry_s;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int v = blockIdx.x; v < n_views; v += gridDim.x) {
    if (threadIdx.x == 0) carry_s = __ldg(view_off + v);
    __syncthreads();
    const size_t base = (size_t)v * ncell;
    for (int c0 = 0; c0 < ncell; c0 += blockDim.x) {
      int c = c0 + threadIdx.x;
      int x = (c < ncell) ? count[base + c] : 0;
      int incl = x;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += y; }
      if (lane == 31) warp_sum[wid] = incl;
      __syncthreads();
      if (wid == 0) {
        int w = warp_sum[lane], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(EMU_FULL, wi, o); if (lane >= o) wi += y; }
        warp_sum[lane] = wi - w;               // exclusive offset of each warp
      }
      __syncthreads();
      int carry = carry_s;
      if (c < ncell) cell_start[base + c] = carry + warp_sum[wid] + incl - x;
      __syncthreads();
      if (threadIdx.x == blockDim.x - 1) carry_s = carry + warp_sum[wid] + incl;
      __syncthreads();
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) cell_start[(size_t)n_views * ncell] = n_grains;
}

// scatter into cell order (arbitrary order inside a cell; fixed by k_bin_place)
__global__ void __launch_bounds__(kBinThreads)
k_bin_scatter(EmuDev P, int frame, const int4* __restrict__ grains, const int* __restrict__ view_off, int n_views,
              int n_grains, int* __restrict__ count, const int* __restrict__ cell_start, int4* __restrict__ tmp) {
  int stride = gridDim.x * blockDim.x;
  const int ncell = P.fr[frame].ncell;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_grains; i += stride) {
    int4 g = emu_to_frame(frame, __ldg(grains + i));
    int v = emu_find_view(view_off, 0, n_views, i);
    size_t gc = (size_t)v * ncell + emu_cell_of_frame(P, frame, g.x, g.y, g.z);
    int k = atomicSub(count + gc, 1) - 1;
    if (frame == 0) g.w = i;                        // payload replaced by the row (original index); frames 1, 2 are
                                                    // binned from frame 0's output, whose w is the row already
    tmp[cell_start[gc] + k] = g;
  }
}

// canonical order inside a cell: ascending row.  rank = #cell-mates with a smaller row.
__global__ void __launch_bounds__(kBinThreads)
k_bin_place(EmuDev P, int frame, const int4* __restrict__ tmp, const int* __restrict__ view_off, int n_views,
            int n_grains, const int* __restrict__ cell_start, int4* __restrict__ sorted) {
  int stride = gridDim.x * blockDim.x;
  const int ncell = P.fr[frame].ncell;
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_grains; j += stride) {
    int4 g = tmp[j];
    int v = emu_find_view(view_off, 0, n_views, g.w);   // rows and sorted positions share the view ranges
    size_t gc = (size_t)v * ncell + emu_cell_of_frame(P, frame, g.x, g.y, g.z);
    int s = cell_start[gc], e = cell_start[gc + 1];
    int rank = 0;
    for (int k = s; k < e; ++k) rank += (tmp[k].w < g.w);
    sorted[s + rank] = g;
  }
}

// ---------------------------------------------------------------------------------------------
// The fast path: ONE kernel, one block per view.  The per-cell counters of a view live in shared memory
// as BYTES (four to a word), so the histogram and the scatter cursors never touch HBM; the grains are
// read twice (the second time mostly from L2: a view is about 1 MB) and written once, cell_start is
// written once and read back from L2.
//   A  histogram: byte counters (a cell that overflows 255 sends the view to the slow variant)
//   B  exclusive scan over the cells, four cells per thread and tile -> cell_start
//   C  scatter: position = cell_start[cell] + (counter-- - 1); the order inside a cell is arbitrary
//   D  canonical order inside a cell (ascending row): cells of 2..8 grains are sorted in place by
//      one thread, larger ones by the whole block through the scratch array
// kSmem = false is the same algorithm with 32-bit counters in global memory, for the views the fast
// variant flagged (redo[v] != 0).
constexpr int kViewThreads = 512;
constexpr int kUnroll = 8;                          // independent grain loads per thread (the kernel is latency-bound otherwise)
constexpr int kSmallCell = 8;
constexpr int kBigCap = 64;
#ifndef EMU_BIN_SMEM_CELLS
#define EMU_BIN_SMEM_CELLS (200 * 1024)
#endif
constexpr int kMaxSmemCells = EMU_BIN_SMEM_CELLS;          // byte counters that fit the shared memory of one block

template <bool kSmem>
__global__ void __launch_bounds__(kViewThreads)
k_bin_view(EmuDev P, int frame, const int4* __restrict__ grains, const int* __restrict__ view_off, int n_views,
           int n_grains, int4* __restrict__ sorted, int* __restrict__ cell_start, int* __restrict__ gcount,
           int4* __restrict__ tmp, int* __restrict__ redo, unsigned long long* __restrict__ status) {
  extern __shared__ unsigned cnt_s[];               // kSmem: ceil(ncell / 4) words of byte counters
  __shared__ int warp_sum[kViewThreads / 32];
  __shared__ int carry_s, flag_s, nbig_s;
  __shared__ int big_s[kBigCap];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int ncell = P.fr[frame].ncell;
  const int nwords = (ncell + 3) >> 2;
  bool bad = false;

  for (int v = blockIdx.x; v < n_views; v += gridDim.x) {
    if (!kSmem && redo[v] == 0) continue;
    const int g0 = __ldg(view_off + v), g1 = __ldg(view_off + v + 1);
    const size_t cbase = (size_t)v * ncell;
    int* gc = kSmem ? nullptr : gcount + cbase;
    // ---- zero the counters ----
    if (kSmem) { for (int w = tid; w < nwords; w += kViewThreads) cnt_s[w] = 0u; }
    else { for (int c = tid; c < ncell; c += kViewThreads) gc[c] = 0; }
    if (tid == 0) { flag_s = 0; nbig_s = 0; carry_s = g0; }
    __syncthreads();
    // ---- A: histogram ----
    bool ovf = false;
    for (int i0 = g0 + tid; i0 < g1; i0 += kUnroll * kViewThreads) {
      int4 gg[kUnroll];
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {              // kUnroll independent 16-byte loads in flight per thread
        const int i = i0 + u * kViewThreads;
        gg[u] = i < g1 ? __ldg(grains + i) : make_int4(0, 0, 0, 0);
      }
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {
        if (i0 + u * kViewThreads >= g1) break;
        const int4 g = emu_to_frame(frame, gg[u]);
        bad |= (abs(g.x) >= (1 << 17)) | (abs(g.y) >= (1 << 17)) | (abs(g.z) >= (1 << 17));
        const int c = emu_cell_of_frame(P, frame, g.x, g.y, g.z);
        if (kSmem) {
          const int sh = 8 * (c & 3);
          const unsigned old = atomicAdd(&cnt_s[c >> 2], 1u << sh);
          ovf |= ((old >> sh) & 0xffu) == 0xffu;
        } else {
          atomicAdd(gc + c, 1);
        }
      }
    }
    if (kSmem) {
      if (ovf) flag_s = 1;
      __syncthreads();
      if (flag_s) {                                   // a cell holds more than 255 grains: the slow variant redoes the view
        if (tid == 0) redo[v] = 1;
        __syncthreads();
        continue;
      }
    } else {
      __syncthreads();
    }
    // ---- B: exclusive scan, four cells per thread and tile ----
    for (int w0 = 0; w0 < nwords; w0 += kViewThreads) {
      const int w = w0 + tid;
      int c4[4] = {0, 0, 0, 0};
      if (w < nwords) {
        if (kSmem) {
          const unsigned x = cnt_s[w];
          c4[0] = x & 0xff; c4[1] = (x >> 8) & 0xff; c4[2] = (x >> 16) & 0xff; c4[3] = x >> 24;
        } else {
#pragma unroll
          for (int k = 0; k < 4; ++k) if (4 * w + k < ncell) c4[k] = gc[4 * w + k];
        }
      }
      const int mine = c4[0] + c4[1] + c4[2] + c4[3];
      int incl = mine;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += y; }
      if (lane == 31) warp_sum[wid] = incl;
      __syncthreads();
      if (wid == 0) {
        int x = (lane < kViewThreads / 32) ? warp_sum[lane] : 0, xi = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(EMU_FULL, xi, o); if (lane >= o) xi += y; }
        if (lane < kViewThreads / 32) warp_sum[lane] = xi - x;
      }
      __syncthreads();
      int run = carry_s + warp_sum[wid] + incl - mine;
      if (w < nwords) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (4 * w + k < ncell) cell_start[cbase + 4 * w + k] = run;
          run += c4[k];
        }
      }
      __syncthreads();
      if (tid == kViewThreads - 1) carry_s = run;
      __syncthreads();
    }
    // ---- C: scatter.  The counters start again from zero and count up: a grain's rank inside its cell is the old
    //      value, and afterwards every counter holds its cell's count again (phase D reads it) ----
    if (kSmem) { for (int w = tid; w < nwords; w += kViewThreads) cnt_s[w] = 0u; }
    else { for (int c = tid; c < ncell; c += kViewThreads) gc[c] = 0; }
    __syncthreads();
    for (int i0 = g0 + tid; i0 < g1; i0 += kUnroll * kViewThreads) {
      int4 gg[kUnroll];
      int start[kUnroll], rank[kUnroll];
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {
        const int i = i0 + u * kViewThreads;
        gg[u] = i < g1 ? __ldg(grains + i) : make_int4(0, 0, 0, 0);
      }
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {              // all the cell_start loads are issued before any is used
        const int i = i0 + u * kViewThreads;
        start[u] = -1; rank[u] = 0;
        if (i < g1) {
          gg[u] = emu_to_frame(frame, gg[u]);
          const int c = emu_cell_of_frame(P, frame, gg[u].x, gg[u].y, gg[u].z);
          start[u] = cell_start[cbase + c];
          if (kSmem) {
            const int sh = 8 * (c & 3);
            rank[u] = (int)((atomicAdd(&cnt_s[c >> 2], 1u << sh) >> sh) & 0xffu);
          } else {
            rank[u] = atomicAdd(gc + c, 1);
          }
          if (frame == 0) gg[u].w = i;                // payload replaced by the row; frames 1, 2 carry it already
        }
      }
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) if (start[u] >= 0) sorted[start[u] + rank[u]] = gg[u];
    }
    __syncthreads();
    // ---- D: ascending row inside every cell (only cells of two or more grains touch memory) ----
    for (int w = tid; w < nwords; w += kViewThreads) {
      int c4[4] = {0, 0, 0, 0};
      if (kSmem) {
        const unsigned x = cnt_s[w];
        if (!((x + 0x7e7e7e7eu) & 0x80808080u) && !(x & 0x80808080u)) continue;    // every byte is 0 or 1
        c4[0] = x & 0xff; c4[1] = (x >> 8) & 0xff; c4[2] = (x >> 16) & 0xff; c4[3] = x >> 24;
      } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) if (4 * w + k < ncell) c4[k] = gc[4 * w + k];
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int n = c4[k];
        if (n < 2) continue;
        const int c = 4 * w + k;
        int slot = kBigCap;
        if (n > kSmallCell) slot = atomicAdd(&nbig_s, 1);
        if (slot < kBigCap) { big_s[slot] = c; continue; }
        const int s = cell_start[cbase + c];
        if (n == 2) {                                 // the common case: one compare, at most one swap
          const int4 p = sorted[s], q = sorted[s + 1];
          if (q.w < p.w) { sorted[s] = q; sorted[s + 1] = p; }
          continue;
        }
        for (int i = 1; i < n; ++i) {                 // insertion sort in place
          const int4 key = sorted[s + i];
          int j = i - 1;
          while (j >= 0) {
            const int4 q = sorted[s + j];
            if (q.w <= key.w) break;
            sorted[s + j + 1] = q;
            --j;
          }
          if (j != i - 1) sorted[s + j + 1] = key;
        }
      }
    }
    __syncthreads();
    const int nbig = min(nbig_s, kBigCap);
    for (int b = 0; b < nbig; ++b) {                  // big cells: rank sort by the whole block through tmp
      const int c = big_s[b];
      const int s = cell_start[cbase + c];
      const int e = (c + 1 < ncell) ? cell_start[cbase + c + 1] : g1;
      for (int i = s + tid; i < e; i += kViewThreads) {
        const int4 g = sorted[i];
        int rank = 0;
        for (int k = s; k < e; ++k) rank += (sorted[k].w < g.w);
        tmp[s + rank] = g;
      }
      __syncthreads();
      for (int i = s + tid; i < e; i += kViewThreads) sorted[i] = tmp[i];
      __syncthreads();
    }
  }
  if (status && __any_sync(EMU_FULL, bad) && lane == 0) atomicOr(status, (unsigned long long)EMU_ST_COORD);
  if (kSmem && blockIdx.x == 0 && tid == 0) cell_start[(size_t)n_views * ncell] = n_grains;
}

// ---------------------------------------------------------------------------------------------
// The two-pass path (the default whenever its plan fits): HBM sees only streams.
//   pass 1  k_bin_split: the cell range of a view is cut into K chunks of cpc cells; every grain goes to
//           the scratch region of its (view, chunk).  A block takes tiles of 2 048 grains of one view (eight
//           per thread, held in registers), counts them per chunk in shared memory, reserves its ranges
//           with K atomics and writes the grains out: a tile leaves about 1 KB per chunk in one piece.
//   pass 2  k_bin_chunk: one block per (view, chunk).  The chunk (<= kChunkCap grains) is read in a stream,
//           counted per cell and scanned in shared memory (16-bit counters), placed into a shared-memory
//           buffer in cell order, put into ascending row order inside every cell, and written out in a
//           stream, with its part of cell_start.
// A view with a chunk fuller than the scratch region is flagged and redone by k_bin_view<false>.
constexpr int kSplitThreads = 256;
#ifndef EMU_SPLIT_PER
#define EMU_SPLIT_PER 8
#endif
constexpr int kSplitPer = EMU_SPLIT_PER;                         // grains per thread and tile
#ifndef EMU_CHUNK_THREADS
#define EMU_CHUNK_THREADS 256
#endif
#ifndef EMU_CHUNK_SLACK
#define EMU_CHUNK_SLACK 1.3
#endif
#ifndef EMU_CHUNK_PER
#define EMU_CHUNK_PER 10
#endif
#ifndef EMU_CHUNK_MINB
#define EMU_CHUNK_MINB 3
#endif
constexpr int kChunkThreads = EMU_CHUNK_THREADS;
constexpr int kChunkPer = EMU_CHUNK_PER;                         // grains per thread of a chunk block (held in registers)
constexpr int kChunkCap = kChunkThreads * kChunkPer; // grains of a chunk: 2 560 = 40 KB of shared memory
constexpr int kMaxChunks = 128;
constexpr int kMaxChunkCells = 12288;                // cells of a chunk: 2 x 16 bits each in shared memory

struct SplitPlan { int K, cpc, cap; float inv_cpc; };

__device__ __forceinline__ int chunk_of(int cell, const SplitPlan& S) {
  int k = (int)(((float)cell + 0.5f) * S.inv_cpc);    // cell < 2^24: within one of the truth
  k -= (k * S.cpc > cell);
  k += ((k + 1) * S.cpc <= cell);
  return k;
}

__global__ void __launch_bounds__(kSplitThreads)
k_bin_split(EmuDev P, int frame, SplitPlan S, const int4* __restrict__ grains, const int* __restrict__ view_off,
            int v_first, int4* __restrict__ tmp, int* __restrict__ cur, int* __restrict__ redo,
            unsigned long long* __restrict__ status) {
  // grid = (tiles, views of the group): block (t, y) takes tile t of view v_first + y; a view with more tiles than the
  // grid has is flagged.  The scratch regions are those of the GROUP (indexed by y): every group reuses the same
  // addresses, so the round trip through the scratch stays in the L2.
  __shared__ int hist_s[kMaxChunks], base_s[kMaxChunks];
  const int tid = threadIdx.x;
  const int v = v_first + (int)blockIdx.y;
  const int g0 = __ldg(view_off + v), g1 = __ldg(view_off + v + 1);
  const int t0 = g0 + (int)blockIdx.x * (kSplitThreads * kSplitPer);
  if (blockIdx.x == 0 && tid == 0 && (long long)(g1 - g0) > (long long)gridDim.x * (kSplitThreads * kSplitPer)) redo[v] = 1;
  if (t0 >= g1) return;
  bool bad = false;
  int4 gg[kSplitPer];
  int kk[kSplitPer], rr[kSplitPer];
  if (tid < S.K) hist_s[tid] = 0;
#pragma unroll
  for (int u = 0; u < kSplitPer; ++u) {
    const int i = t0 + u * kSplitThreads + tid;
    gg[u] = i < g1 ? __ldg(grains + i) : make_int4(0, 0, 0, 0);
  }
  __syncthreads();
#pragma unroll
  for (int u = 0; u < kSplitPer; ++u) {
    const int i = t0 + u * kSplitThreads + tid;
    kk[u] = -1; rr[u] = 0;
    if (i < g1) {
      gg[u] = emu_to_frame(frame, gg[u]);
      if (frame == 0) gg[u].w = i;                     // payload replaced by the row; frames 1, 2 carry it already
      bad |= (abs(gg[u].x) >= (1 << 17)) | (abs(gg[u].y) >= (1 << 17)) | (abs(gg[u].z) >= (1 << 17));
      const int cell = emu_cell_of_frame(P, frame, gg[u].x, gg[u].y, gg[u].z);
      kk[u] = chunk_of(cell, S);
      rr[u] = atomicAdd(&hist_s[kk[u]], 1);
      // the scratch record carries the cell inside its chunk (< 2^14) above the 18 bits of x, so that pass 2 does not
      // derive it again (a coordinate out of range is reported through `status`; the outputs are then unspecified)
      gg[u].x = (gg[u].x & 0x3ffff) | ((cell - kk[u] * S.cpc) << 18);
    }
  }
  __syncthreads();
  if (tid < S.K) {
    const int h = hist_s[tid];
    int b = 0;
    if (h) {
      b = atomicAdd(cur + (size_t)v * S.K + tid, h);
      if (b + h > S.cap) redo[v] = 1;                  // the region is full: k_bin_view<false> redoes the view
    }
    base_s[tid] = b;
  }
  __syncthreads();
#pragma unroll
  for (int u = 0; u < kSplitPer; ++u) {
    if (kk[u] < 0) continue;
    const int slot = base_s[kk[u]] + rr[u];
    if (slot < S.cap) tmp[((size_t)blockIdx.y * S.K + kk[u]) * S.cap + slot] = gg[u];
  }
  if (status && __any_sync(EMU_FULL, bad) && (tid & 31) == 0) atomicOr(status, (unsigned long long)EMU_ST_COORD);
}

// 1: pass 2 stores every grain straight to its place instead of staging the chunk in shared memory and streaming it
// out (one barrier and 39 KB of shared memory less; 1.154 -> 1.126 ms on the bench; more blocks per SM only spill)
#ifndef EMU_BIN_DIRECT
#define EMU_BIN_DIRECT 1
#endif
__global__ void __launch_bounds__(kChunkThreads, EMU_CHUNK_MINB)
k_bin_chunk(EmuDev P, int frame, SplitPlan S, const int* __restrict__ view_off, int n_views, int n_grains, int v_first,
            const int4* __restrict__ tmp, const int* __restrict__ cur, const int* __restrict__ redo,
            int4* __restrict__ sorted, int* __restrict__ cell_start) {
  extern __shared__ __align__(16) unsigned char chunk_smem[];
  __shared__ int warp_sum[kChunkThreads / 32];
  __shared__ int base_s;
  const int k = blockIdx.x, v = v_first + (int)blockIdx.y;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int ncell = P.fr[frame].ncell;
  if (k == 0 && v == 0 && tid == 0) cell_start[(size_t)n_views * ncell] = n_grains;
  if (redo[v]) return;
  const int c_lo = k * S.cpc, nc = min(ncell, c_lo + S.cpc) - c_lo;
  if (nc <= 0) return;
#if EMU_BIN_DIRECT
  unsigned short* cnt = reinterpret_cast<unsigned short*>(chunk_smem);                // [cpc] counts
#else
  int4* buf = reinterpret_cast<int4*>(chunk_smem);                                   // [cap]
  unsigned short* cnt = reinterpret_cast<unsigned short*>(chunk_smem + (size_t)S.cap * 16);   // [cpc] counts
#endif
  unsigned short* pre = cnt + ((S.cpc + 1) & ~1);                                    // [cpc] exclusive prefix
  unsigned* cntw = reinterpret_cast<unsigned*>(cnt);
  int* wbuf = reinterpret_cast<int*>(pre + ((S.cpc + 1) & ~1));                      // [cap] rows in arrival order
  const int4* src = tmp + ((size_t)blockIdx.y * S.K + k) * S.cap;
  const int n = min(cur[(size_t)v * S.K + k], S.cap);
  int4 gg[kChunkPer];                                  // the chunk's grains stay in registers: one batch of independent loads
#pragma unroll
  for (int u = 0; u < kChunkPer; ++u) {
    const int i = tid + u * kChunkThreads;
    gg[u] = i < n ? __ldg(src + i) : make_int4(0, 0, 0, 0);
  }
  // position of the chunk's first grain: the view's start + the grains of the chunks before
  if (wid == 0) {
    int sum = 0;
    for (int q = lane; q < k; q += 32) sum += cur[(size_t)v * S.K + q];
    sum = __reduce_add_sync(EMU_FULL, sum);
    if (lane == 0) base_s = __ldg(view_off + v) + sum;
  }
  for (int w = tid; w < (nc + 1) / 2; w += kChunkThreads) cntw[w] = 0u;
  __syncthreads();
  const int base = base_s;
  // ---- count per cell (the chunk's grains stay in registers: one batch of independent loads) ----
  int cc[kChunkPer], rk[kChunkPer];                            // cell inside the chunk, arrival rank inside the cell
#pragma unroll
  for (int u = 0; u < kChunkPer; ++u) {
    cc[u] = -1; rk[u] = 0;
    if (tid + u * kChunkThreads < n) {
      cc[u] = min((int)((unsigned)gg[u].x >> 18), nc - 1);     // the cell inside the chunk, packed by pass 1
      gg[u].x = (gg[u].x << 14) >> 14;                         // x again (sign-extended 18 bits)
      const int sh = 16 * (cc[u] & 1);
      rk[u] = (int)((atomicAdd(&cntw[cc[u] >> 1], 1u << sh) >> sh) & 0xffffu);
    }
  }
  __syncthreads();
  // ---- exclusive scan over the cells of the chunk: a run of consecutive cells per thread ----
  const int per = (nc + kChunkThreads - 1) / kChunkThreads;
  const int c0 = tid * per, c1 = min(nc, c0 + per);
  int mine = 0;
  for (int c = c0; c < c1; ++c) mine += cnt[c];
  int incl = mine;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += y; }
  if (lane == 31) warp_sum[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    int x = (lane < kChunkThreads / 32) ? warp_sum[lane] : 0, xi = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(EMU_FULL, xi, o); if (lane >= o) xi += y; }
    if (lane < kChunkThreads / 32) warp_sum[lane] = xi - x;
  }
  __syncthreads();
  int run = warp_sum[wid] + incl - mine;
  for (int c = c0; c < c1; ++c) { pre[c] = (unsigned short)run; run += cnt[c]; }
  __syncthreads();
  for (int c = tid; c < nc; c += kChunkThreads) cell_start[(size_t)v * ncell + c_lo + c] = base + (int)pre[c];
  // ---- the rows of the grains go to their cell's range in arrival order ...
#pragma unroll
  for (int u = 0; u < kChunkPer; ++u) if (cc[u] >= 0) wbuf[(int)pre[cc[u]] + rk[u]] = gg[u].w;
  __syncthreads();
  // ---- ... and every grain takes the place its row deserves among its cell-mates (ascending row inside every cell;
  //      rows are distinct: the ranks are a permutation) ----
#pragma unroll
  for (int u = 0; u < kChunkPer; ++u) {
    if (cc[u] < 0) continue;
    const int m = cnt[cc[u]], p0 = pre[cc[u]];
    int r = 0;
    if (m >= 2) for (int t = 0; t < m; ++t) r += (wbuf[p0 + t] < gg[u].w);
#if EMU_BIN_DIRECT
    sorted[base + p0 + r] = gg[u];                     // straight to its place (the L2 merges the 16-byte stores of a chunk)
#else
    buf[p0 + r] = gg[u];
#endif
  }
#if !EMU_BIN_DIRECT
  __syncthreads();
  for (int i = tid; i < n; i += kChunkThreads) sorted[base + i] = buf[i];
#endif
}

// plan of the two-pass path for one frame; K = 0: not applicable (the one-kernel paths take over)
SplitPlan split_plan(const EmuDev& P, int frame, int64_t n_grains, int32_t n_views) {
  SplitPlan S; S.K = 0; S.cpc = 1; S.cap = 0; S.inv_cpc = 1.0f;
  const int ncell = P.fr[frame].ncell;
  if (n_views < 1 || n_grains < 1 || ncell >= (1 << 24)) return S;
  const double avg = (double)n_grains / n_views;
  // the fewest chunks whose scratch region (EMU_CHUNK_SLACK = 1.3 x the average chunk + 256) fits the shared-memory buffer
  int K = (int)emu_max64(1, (int64_t)(avg * EMU_CHUNK_SLACK / (double)(kChunkCap - 256 - 64)) + 1);
  K = (int)emu_max64(K, ((int64_t)ncell + kMaxChunkCells - 1) / kMaxChunkCells);
  if (K > kMaxChunks) return S;
  const int cpc = (ncell + K - 1) / K;
  const int cap = (((int)(avg / K * EMU_CHUNK_SLACK) + 256) + 63) & ~63;
  if (cap > kChunkCap) return S;
  S.K = (ncell + cpc - 1) / cpc; S.cpc = cpc; S.cap = cap; S.inv_cpc = 1.0f / (float)cpc;
  return S;
}

// views per group of the two-pass path.  A group's scratch regions (K x cap grains per view) are reused by the next
// group; with groups that fit the L2 the round trip through the scratch could stay on chip.  Measured on the bench
// (1 024 views): one group 1.14 ms; groups of 128 / 96 / 64 / 48 / 32 / 16 MB: 1.34 / 1.40 / 1.50 / 1.56 / 1.71 / 2.31 ms -
// the tail of every small launch costs more than the traffic saves, so the default is ONE group (the hook stays for
// the record).
#ifndef EMU_BIN_GROUP_MB
#define EMU_BIN_GROUP_MB (1 << 20)
#endif
int split_group_views(const SplitPlan& S, int32_t n_views) {
  const int mb = EMU_BIN_GROUP_MB;                   // compile-time only: the library reads no environment
  const int64_t per_view = (int64_t)S.K * S.cap * 16;
  const int64_t g = emu_max64(1, ((int64_t)mb << 20) / emu_max64(1, per_view));
  return (int)emu_min64(emu_min64(g, 65535), emu_max64(1, n_views));
}

size_t split_tmp_grains(const EmuDev& P, int64_t n_grains, int32_t n_views) {
  size_t m = (size_t)n_grains;                       // (the one-kernel paths sort big cells through it)
  for (int f = 0; f < 3; ++f) {
    const SplitPlan S = split_plan(P, f, n_grains, n_views);
    if (S.K) m = emu_max64((int64_t)m, (int64_t)split_group_views(S, n_views) * S.K * S.cap);
  }
  return m;
}

}  // namespace

size_t emu_bin_ws_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views) {
  int ncell = P.fr[0].ncell;
  for (int f = 1; f < 3; ++f) if (P.fr[f].ncell > ncell) ncell = P.fr[f].ncell;     // one scratch serves every frame
  size_t cnt = emu_align256((size_t)n_views * ncell * sizeof(int));
  size_t tmp = emu_align256(split_tmp_grains(P, n_grains, n_views) * sizeof(int4));
  size_t redo = emu_align256(((size_t)n_views + 1) * sizeof(int));
  size_t cur = emu_align256((size_t)n_views * kMaxChunks * sizeof(int));
  return cnt + tmp + redo + cur + 256;
}

int emu_bin_launch(const EmuDev& P, int frame, const int32_t* d_grains, const int32_t* d_view_off, int64_t n_grains,
                   int32_t n_views, int32_t* d_sorted, int32_t* d_cell_start, int64_t* d_status, void* d_ws,
                   size_t ws_bytes, cudaStream_t st) {
  if (ws_bytes < emu_bin_ws_bytes(P, n_grains, n_views)) return EMU_ERR_CAPACITY;
  char* ws = (char*)emu_align_ptr(d_ws);
  int* count = (int*)ws;
  const int ncell = P.fr[frame].ncell;
  int ncell_max = P.fr[0].ncell;
  for (int f = 1; f < 3; ++f) if (P.fr[f].ncell > ncell_max) ncell_max = P.fr[f].ncell;
  int4* tmp = (int4*)(ws + emu_align256((size_t)n_views * ncell_max * sizeof(int)));
  int* redo = (int*)((char*)tmp + emu_align256(split_tmp_grains(P, n_grains, n_views) * sizeof(int4)));
  int* cur = (int*)((char*)redo + emu_align256(((size_t)n_views + 1) * sizeof(int)));
  const int n = (int)n_grains;
  const SplitPlan S = split_plan(P, frame, n_grains, n_views);
  if (S.K > 0) {
    // two passes: split into chunks of cells, then one chunk per block in shared memory
    const size_t smem = (EMU_BIN_DIRECT ? 0 : (size_t)S.cap * 16) + 2 * (size_t)((S.cpc + 1) & ~1) * sizeof(unsigned short) + (size_t)S.cap * 4;
    if (cudaFuncSetAttribute(k_bin_chunk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaMemsetAsync(redo, 0, ((size_t)n_views + 1) * sizeof(int), st) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaMemsetAsync(cur, 0, (size_t)n_views * S.K * sizeof(int), st) != cudaSuccess) return EMU_ERR_CUDA;
    const int blocks = (int)emu_max64(1, emu_min64(n_views, emu_sm_count() * 8));
    const int tile = kSplitThreads * kSplitPer;
    const int tiles = (int)emu_min64(65535, 2 * ((n_grains / n_views + tile - 1) / tile) + 2);   // per view; larger views are redone
    const int G = split_group_views(S, n_views);
    for (int v0 = 0; v0 < n_views; v0 += G) {
      const int gv = (int)emu_min64(G, n_views - v0);
      EMU_LAUNCH(frame == 0 ? EMU_STAGE_BIN_COUNT : EMU_STAGE_PREP, st, k_bin_split<<<dim3(tiles, gv), kSplitThreads, 0, st>>>(
          P, frame, S, (const int4*)d_grains, d_view_off, v0, tmp, cur, redo, (unsigned long long*)d_status));
      EMU_LAUNCH(frame == 0 ? EMU_STAGE_BIN_SCATTER : EMU_STAGE_PREP, st, k_bin_chunk<<<dim3(S.K, gv), kChunkThreads, smem, st>>>(
          P, frame, S, d_view_off, n_views, n, v0, tmp, cur, redo, (int4*)d_sorted, d_cell_start));
    }
    EMU_LAUNCH(frame == 0 ? EMU_STAGE_BIN_PLACE : EMU_STAGE_PREP, st, k_bin_view<false><<<blocks, kViewThreads, 0, st>>>(
        P, frame, (const int4*)d_grains, d_view_off, n_views, n, (int4*)d_sorted, d_cell_start, count, tmp, redo,
        (unsigned long long*)d_status));
    return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
  }
  if (ncell <= kMaxSmemCells) {
    // one block per view, byte counters in shared memory; the views it flags are redone with global counters
    const size_t smem = (size_t)((ncell + 3) / 4) * 4;
    if (cudaFuncSetAttribute(k_bin_view<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaMemsetAsync(redo, 0, ((size_t)n_views + 1) * sizeof(int), st) != cudaSuccess) return EMU_ERR_CUDA;
    const int blocks = (int)emu_max64(1, emu_min64(n_views, emu_sm_count() * 8));
    EMU_LAUNCH(frame == 0 ? EMU_STAGE_BIN_SCATTER : EMU_STAGE_PREP, st, k_bin_view<true><<<blocks, kViewThreads, smem, st>>>(
        P, frame, (const int4*)d_grains, d_view_off, n_views, n, (int4*)d_sorted, d_cell_start, count, tmp, redo,
        (unsigned long long*)d_status));
    EMU_LAUNCH(frame == 0 ? EMU_STAGE_BIN_PLACE : EMU_STAGE_PREP, st, k_bin_view<false><<<blocks, kViewThreads, 0, st>>>(
        P, frame, (const int4*)d_grains, d_view_off, n_views, n, (int4*)d_sorted, d_cell_start, count, tmp, redo,
        (unsigned long long*)d_status));
    return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
  }
  if (cudaMemsetAsync(count, 0, (size_t)n_views * ncell * sizeof(int), st) != cudaSuccess) return EMU_ERR_CUDA;
  int blocks = (int)emu_min64((n_grains + kBinThreads - 1) / kBinThreads, emu_sm_count() * 16);
  if (blocks < 1) blocks = 1;
  EMU_LAUNCH(EMU_STAGE_BIN_COUNT, st, k_bin_count<<<blocks, kBinThreads, 0, st>>>(P, frame, (const int4*)d_grains, d_view_off, n_views, n, count,
                                              (unsigned long long*)d_status));
  EMU_LAUNCH(EMU_STAGE_BIN_SCAN, st, k_bin_scan<<<(int)emu_min64(n_views > 0 ? n_views : 1, emu_sm_count() * 2), 1024, 0, st>>>(ncell, d_view_off, n_views, n, count, d_cell_start));
  EMU_LAUNCH(EMU_STAGE_BIN_SCATTER, st, k_bin_scatter<<<blocks, kBinThreads, 0, st>>>(P, frame, (const int4*)d_grains, d_view_off, n_views, n, count, d_cell_start, tmp));
  EMU_LAUNCH(EMU_STAGE_BIN_PLACE, st, k_bin_place<<<blocks, kBinThreads, 0, st>>>(P, frame, tmp, d_view_off, n_views, n, d_cell_start, (int4*)d_sorted));
  return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
}
