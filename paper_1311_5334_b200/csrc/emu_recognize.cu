// emu_recognize.cu - A0, upstream of the hot path: 3D grain recognition on a stack of
// filtered frames ("Each pixel with a pulse height higher than a given threshold is compared to the
// 3 x 3 x 3 neighboring pixels; the pixel with the highest pulse height among these will be defining the grain.
// The spatial coordinates of the grains are then computed with a center-of-mass method using the pulse height of
// each pixel").  Readings R1-R5 of DESIGN.md section 3b.  Product code: shares nothing with oracle/.
//
// HBM-bound: the stack is read twice (1 byte per voxel each time; the second time from L2 when a view fits it),
// the 26 neighbours only for the few voxels above the threshold.
//   k_recog<0>   one warp per row (z, y) of a view: number of grains whose defining voxel lies in the row
//   k_row_scan   exclusive scan over the rows of every view (one block per view) + k_view_offsets over the views
//   k_recog<1>   the same detection; the grains of a row are written in x order at the row's offset, so the output
//                is in raster order of the defining voxel (R5), view after view
#include "emu_dev.cuh"
#include "emu_host.h"

namespace {

struct Recog {
  int nx, ny, nz, thr;
  int pitch[3];
};

__device__ __forceinline__ int vox_at(const unsigned char* __restrict__ v, const Recog& R, int x, int y, int z) {
  if ((unsigned)x >= (unsigned)R.nx || (unsigned)y >= (unsigned)R.ny || (unsigned)z >= (unsigned)R.nz) return 0;   // R2
  return (int)__ldg(v + ((size_t)z * R.ny + y) * R.nx + x);
}

// is voxel (x, y, z) of pulse height c > thr the highest of its 3x3x3 neighbourhood (R2)?  If so, the grain record.
__device__ bool grain_of(const unsigned char* __restrict__ v, const Recog& R, int x, int y, int z, int c, int4& out) {
  long long sw = 0, sx = 0, sy = 0, sz = 0;
  bool ok = true;
  // which neighbours exist (voxels outside the stack count as 0, R2): six comparisons for all 26
  const bool in_lo[3] = {x > 0, y > 0, z > 0}, in_hi[3] = {x + 1 < R.nx, y + 1 < R.ny, z + 1 < R.nz};
  const long long sy_ = R.nx, sz_ = (long long)R.nx * R.ny;
  const unsigned char* p0 = v + ((size_t)z * R.ny + y) * R.nx + x;
#pragma unroll
  for (int dz = -1; dz <= 1; ++dz)
#pragma unroll
    for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
      for (int dx = -1; dx <= 1; ++dx) {
        const bool inside = (dx < 0 ? in_lo[0] : (dx > 0 ? in_hi[0] : true)) && (dy < 0 ? in_lo[1] : (dy > 0 ? in_hi[1] : true)) &&
                            (dz < 0 ? in_lo[2] : (dz > 0 ? in_hi[2] : true));
        const int n = inside ? (int)__ldg(p0 + (dz * sz_ + dy * sy_ + dx)) : 0;
        const bool before = dz < 0 || (dz == 0 && (dy < 0 || (dy == 0 && dx < 0)));     // raster order (z, y, x)
        if ((dz | dy | dx) != 0 && (n > c || (before && n == c))) ok = false;
        const int w = n > R.thr ? n : 0;                                               // R3
        sw += w; sx += (long long)(w * dx); sy += (long long)(w * dy); sz += (long long)(w * dz);
      }
  if (!ok) return false;
  sx += sw * x; sy += sw * y; sz += sw * z;                     // sums of w * absolute index
  // R4: pos_q = floor(p (sum(w i) / sum(w) + 1/2) + 1/2), exact in integers (sw >= c > 0)
  out.x = (int)((2ll * R.pitch[0] * sx + (long long)R.pitch[0] * sw + sw) / (2ll * sw));
  out.y = (int)((2ll * R.pitch[1] * sy + (long long)R.pitch[1] * sw + sw) / (2ll * sw));
  out.z = (int)((2ll * R.pitch[2] * sz + (long long)R.pitch[2] * sw + sw) / (2ll * sw));
  out.w = c;
  return true;
}

constexpr int kRecogThreads = 256;

// One warp per row.  The voxels above the threshold (1-2 % of a filtered frame) are first gathered, in x order, in a
// small ring of the warp; whenever 32 of them wait (and at the end of the row) every lane examines ONE of them - its 26
// neighbours, the raster tie rule, the centre of mass - so the expensive part runs with full warps instead of for one
// or two lanes of every 128 voxels.
constexpr int kRing = 1024;                                     // >= 31 waiting + 512 new

#ifndef EMU_RECOG_MINB
#define EMU_RECOG_MINB 4
#endif
template <int kFill>
__global__ void __launch_bounds__(kRecogThreads, EMU_RECOG_MINB)
k_recog(Recog R, const unsigned char* __restrict__ vox, int n_views, int* __restrict__ row_cnt,
        const int* __restrict__ row_off, int4* __restrict__ grains, long long capacity,
        unsigned long long* __restrict__ status) {
  __shared__ unsigned short ring_s[kRecogThreads / 32][kRing];
  const int lane = threadIdx.x & 31;
  unsigned short* ring = ring_s[threadIdx.x >> 5];
  const unsigned thr4 = (unsigned)R.thr * 0x01010101u;
  const long long rows_per_view = (long long)R.nz * R.ny, n_rows = rows_per_view * n_views;
  const long long warp0 = (long long)blockIdx.x * (kRecogThreads / 32) + (threadIdx.x >> 5);
  const long long n_warps = (long long)gridDim.x * (kRecogThreads / 32);
  for (long long row = warp0; row < n_rows; row += n_warps) {
    const int view = (int)(row / rows_per_view);
    const int zy = (int)(row - (long long)view * rows_per_view);
    const int z = zy / R.ny, y = zy - z * R.ny;
    const unsigned char* v = vox + (size_t)view * rows_per_view * R.nx;
    const unsigned char* line = v + ((size_t)z * R.ny + y) * R.nx;
    int n_row = 0;                                              // grains of the row so far (warp-uniform)
    int head = 0, qn = 0;                                       // the ring: first waiting entry, number waiting
    const int base = kFill ? row_off[row] : 0;

    // examine the first m (<= 32) waiting voxels, one per lane; they are in x order, and so are the grains written
    auto flush = [&](int m) {
      __syncwarp();
      int4 g = make_int4(0, 0, 0, 0);
      bool ok = false;
      if (lane < m) {
        const int x = (int)ring[(head + lane) & (kRing - 1)];
        ok = grain_of(v, R, x, y, z, (int)__ldg(line + x), g);
      }
      const unsigned mk = __ballot_sync(EMU_FULL, ok);
      if (kFill && ok) {
        const long long at = (long long)base + n_row + __popc(mk & ((1u << lane) - 1u));
        if (at < capacity) grains[at] = g;
        else if (status) atomicOr(status, (unsigned long long)EMU_ST_GRAIN_OVERFLOW);
      }
      n_row += __popc(mk);
      head = (head + m) & (kRing - 1); qn -= m;
    };

    // 16 voxels per lane and step: one 16-byte load, the load of the next step already in flight
    auto load16 = [&](int x) {
      uint4 t = make_uint4(0u, 0u, 0u, 0u);
      if (x + 15 < R.nx && (((size_t)(line + x)) & 15) == 0) {
        t = __ldg(reinterpret_cast<const uint4*>(line + x));
      } else if (x < R.nx) {
        unsigned w[4] = {0u, 0u, 0u, 0u};
#pragma unroll
        for (int k = 0; k < 16; ++k) if (x + k < R.nx) w[k >> 2] |= (unsigned)__ldg(line + x + k) << (8 * (k & 3));
        t = make_uint4(w[0], w[1], w[2], w[3]);
      }
      return t;
    };
    uint4 nxt = load16(16 * lane);
    for (int x0 = 0; x0 < R.nx; x0 += 512) {
      const int x = x0 + 16 * lane;
      const uint4 cur = nxt;
      if (x0 + 512 < R.nx) nxt = load16(x + 512);
      const unsigned q[4] = {cur.x, cur.y, cur.z, cur.w};
      // four voxels per SIMD byte compare: one mask bit per voxel above the threshold
      unsigned mk[4];
      int cnt = 0;
#pragma unroll
      for (int w = 0; w < 4; ++w) { mk[w] = __vcmpgtu4(q[w], thr4) & 0x01010101u; cnt += __popc(mk[w]); }
      if (!__ballot_sync(EMU_FULL, cnt > 0)) continue;
      int incl = cnt;                                           // x order: lanes in order, voxels of a lane in order
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += t; }
      int at = head + qn + incl - cnt;
      if (cnt) {
#pragma unroll
        for (int w = 0; w < 4; ++w)
          for (unsigned m = mk[w]; m; m &= m - 1u) {            // the set bits in ascending order = ascending x
            ring[at & (kRing - 1)] = (unsigned short)(x + 4 * w + ((__ffs((int)m) - 1) >> 3));
            ++at;
          }
      }
      qn += __shfl_sync(EMU_FULL, incl, 31);
      while (qn >= 32) flush(32);
    }
    while (qn > 0) flush(min(qn, 32));
    if (!kFill && lane == 0) row_cnt[row] = n_row;
  }
}

// exclusive scan (in place) over the rows of every view: row_cnt -> offset inside the view; view_tot[v] = grains of the view
__global__ void __launch_bounds__(1024)
k_row_scan(int rows_per_view, int n_views, int* __restrict__ row_cnt, int* __restrict__ view_tot) {
  __shared__ int warp_sum[32];
  __shared__ int carry_s;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int v = blockIdx.x; v < n_views; v += gridDim.x) {
    int* a = row_cnt + (size_t)v * rows_per_view;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int b = 0; b < rows_per_view; b += blockDim.x) {
      const int i = b + threadIdx.x;
      const int x = i < rows_per_view ? a[i] : 0;
      int incl = x;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += t; }
      if (lane == 31) warp_sum[wid] = incl;
      __syncthreads();
      if (wid == 0) {
        const int w = warp_sum[lane]; int wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(EMU_FULL, wi, o); if (lane >= o) wi += t; }
        warp_sum[lane] = wi - w;
      }
      __syncthreads();
      const int mine = carry_s + warp_sum[wid] + incl;
      if (i < rows_per_view) a[i] = mine - x;
      __syncthreads();
      if (threadIdx.x == blockDim.x - 1) carry_s = mine;
      __syncthreads();
    }
    if (threadIdx.x == 0) view_tot[v] = carry_s;
    __syncthreads();
  }
}

// view_off[0..n_views] from the per-view totals (one thread: n_views is small), and the total
__global__ void k_view_offsets(int n_views, const int* __restrict__ view_tot, int* __restrict__ view_off,
                               long long* __restrict__ count) {
  long long run = 0;
  for (int v = 0; v < n_views; ++v) { view_off[v] = (int)run; run += view_tot[v]; }
  view_off[n_views] = (int)(run > 0x7fffffffll ? 0x7fffffffll : run);
  *count = run;
}

// offsets inside the view -> positions in the output
__global__ void __launch_bounds__(256)
k_row_rebase(int rows_per_view, int n_views, int* __restrict__ row_off, const int* __restrict__ view_off) {
  const long long n = (long long)rows_per_view * n_views;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    row_off[i] += view_off[(int)(i / rows_per_view)];
}

}  // namespace

size_t emu_recognize_ws_bytes(int32_t n_views, int32_t ny, int32_t nz) {
  return emu_align256((size_t)n_views * ny * nz * sizeof(int)) + emu_align256((size_t)(n_views + 1) * sizeof(int)) + 512;
}

int emu_recognize_launch(const uint8_t* d_vox, int32_t n_views, int32_t nx, int32_t ny, int32_t nz, int32_t thr,
                         const int32_t* pitch_q, int32_t* d_grains, int64_t capacity, int32_t* d_view_off,
                         int64_t* d_count, int64_t* d_status, void* d_ws, size_t ws_bytes, cudaStream_t st) {
  if (ws_bytes < emu_recognize_ws_bytes(n_views, ny, nz)) return EMU_ERR_CAPACITY;
  Recog R; R.nx = nx; R.ny = ny; R.nz = nz; R.thr = thr;
  for (int a = 0; a < 3; ++a) R.pitch[a] = pitch_q[a];
  char* ws = (char*)emu_align_ptr(d_ws);
  int* row = (int*)ws;
  int* view_tot = (int*)(ws + emu_align256((size_t)n_views * ny * nz * sizeof(int)));
  const int rows_per_view = ny * nz;
  const long long n_rows = (long long)rows_per_view * n_views;
  const int blocks = (int)emu_max64(1, emu_min64((n_rows + 7) / 8, emu_sm_count() * 32));
  EMU_LAUNCH(EMU_STAGE_RECOG, st, k_recog<0><<<blocks, kRecogThreads, 0, st>>>(R, d_vox, n_views, row, nullptr, nullptr, 0,
                                                                                (unsigned long long*)d_status));
  EMU_LAUNCH(EMU_STAGE_RECOG, st, k_row_scan<<<(int)emu_max64(1, emu_min64(n_views, emu_sm_count() * 2)), 1024, 0, st>>>(rows_per_view, n_views, row, view_tot));
  EMU_LAUNCH(EMU_STAGE_RECOG, st, k_view_offsets<<<1, 1, 0, st>>>(n_views, view_tot, d_view_off, (long long*)d_count));
  EMU_LAUNCH(EMU_STAGE_RECOG, st, k_row_rebase<<<(int)emu_max64(1, emu_min64((n_rows + 255) / 256, emu_sm_count() * 8)), 256, 0, st>>>(rows_per_view, n_views, row, d_view_off));
  EMU_LAUNCH(EMU_STAGE_RECOG, st, k_recog<1><<<blocks, kRecogThreads, 0, st>>>(R, d_vox, n_views, row, row, (int4*)d_grains, capacity,
                                                                                (unsigned long long*)d_status));
  return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
}
