// emu_bin.cu - A1: attribute every grain to its 3D cell as a counting sort.
//   count (per-(view,cell) histogram) -> per-view exclusive scan -> scatter -> rank inside the cell.
// Output order is (view, cell, row): the canonical order SURVEY 8(c) O1 defines.
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

}  // namespace

size_t emu_bin_ws_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views) {
  int ncell = P.fr[0].ncell;
  for (int f = 1; f < 3; ++f) if (P.fr[f].ncell > ncell) ncell = P.fr[f].ncell;     // one scratch serves every frame
  size_t cnt = emu_align256((size_t)n_views * ncell * sizeof(int));
  size_t tmp = emu_align256((size_t)n_grains * sizeof(int4));
  return cnt + tmp + 256;
}

int emu_bin_launch(const EmuDev& P, int frame, const int32_t* d_grains, const int32_t* d_view_off, int64_t n_grains,
                   int32_t n_views, int32_t* d_sorted, int32_t* d_cell_start, int64_t* d_status, void* d_ws,
                   size_t ws_bytes, cudaStream_t st) {
  if (ws_bytes < emu_bin_ws_bytes(P, n_grains, n_views)) return EMU_ERR_CAPACITY;
  char* ws = (char*)emu_align_ptr(d_ws);
  int* count = (int*)ws;
  const int ncell = P.fr[frame].ncell;
  int4* tmp = (int4*)(ws + emu_align256((size_t)n_views * ncell * sizeof(int)));
  const int n = (int)n_grains;
  if (cudaMemsetAsync(count, 0, (size_t)n_views * ncell * sizeof(int), st) != cudaSuccess) return EMU_ERR_CUDA;
  int blocks = (int)emu_min64((n_grains + kBinThreads - 1) / kBinThreads, 148 * 16);
  if (blocks < 1) blocks = 1;
  EMU_LAUNCH(EMU_STAGE_BIN_COUNT, st, k_bin_count<<<blocks, kBinThreads, 0, st>>>(P, frame, (const int4*)d_grains, d_view_off, n_views, n, count,
                                              (unsigned long long*)d_status));
  EMU_LAUNCH(EMU_STAGE_BIN_SCAN, st, k_bin_scan<<<(int)emu_min64(n_views > 0 ? n_views : 1, 148 * 2), 1024, 0, st>>>(ncell, d_view_off, n_views, n, count, d_cell_start));
  EMU_LAUNCH(EMU_STAGE_BIN_SCATTER, st, k_bin_scatter<<<blocks, kBinThreads, 0, st>>>(P, frame, (const int4*)d_grains, d_view_off, n_views, n, count, d_cell_start, tmp));
  EMU_LAUNCH(EMU_STAGE_BIN_PLACE, st, k_bin_place<<<blocks, kBinThreads, 0, st>>>(P, frame, tmp, d_view_off, n_views, n, d_cell_start, (int4*)d_sorted));
  return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
}
