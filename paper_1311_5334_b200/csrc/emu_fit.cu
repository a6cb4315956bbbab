// emu_fit.cu - A6: least-squares line per track (BASELINE.json north_star; reading Q9; the paper only
// draws "the start and the end of the tracks").  One warp per track: exact int64 moment sums
// (order-free), then a handful of float64 operations on lane 0.
#include "emu_dev.cuh"
#include "emu_host.h"

namespace {

__device__ __forceinline__ long long warp_sum_ll(long long x) {
#pragma unroll
  for (int o = 16; o; o >>= 1) x += __shfl_xor_sync(EMU_FULL, x, o);
  return x;
}

__global__ void __launch_bounds__(256)
k_fit(const int4* __restrict__ grains, const emu_track* __restrict__ tracks, const int* __restrict__ track_off,
      const int* __restrict__ members, int n_views, emu_fit* __restrict__ fits) {
  const int lane = threadIdx.x & 31;
  const int n_tracks = track_off[n_views];
  const int wpb = blockDim.x >> 5;
  for (int t = blockIdx.x * wpb + (threadIdx.x >> 5); t < n_tracks; t += gridDim.x * wpb) {
    const int n = tracks[t].n_members;
    const int* m = members + tracks[t].member_off;
    int lo[3] = {0x7fffffff, 0x7fffffff, 0x7fffffff};
    int hi[3] = {(int)0x80000000, (int)0x80000000, (int)0x80000000};
    for (int i = lane; i < n; i += 32) {
      int4 g = __ldg(grains + m[i]);
      lo[0] = min(lo[0], g.x); hi[0] = max(hi[0], g.x);
      lo[1] = min(lo[1], g.y); hi[1] = max(hi[1], g.y);
      lo[2] = min(lo[2], g.z); hi[2] = max(hi[2], g.z);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) { lo[a] = __reduce_min_sync(EMU_FULL, lo[a]); hi[a] = __reduce_max_sync(EMU_FULL, hi[a]); }
    // dominant axis by member extent; ties prefer z, then x (reading Q9)
    const long long ex = (long long)hi[0] - lo[0], ey = (long long)hi[1] - lo[1], ez = (long long)hi[2] - lo[2];
    int u, v, w;
    if (ez >= ex && ez >= ey) { u = 2; v = 0; w = 1; }
    else if (ex >= ey)        { u = 0; v = 1; w = 2; }
    else                      { u = 1; v = 0; w = 2; }
    long long Su = 0, Sv = 0, Sw = 0, Suu = 0, Suv = 0, Suw = 0;
    for (int i = lane; i < n; i += 32) {
      int4 g = __ldg(grains + m[i]);
      long long c[3] = {g.x, g.y, g.z};
      Su += c[u]; Sv += c[v]; Sw += c[w];
      Suu += c[u] * c[u]; Suv += c[u] * c[v]; Suw += c[u] * c[w];
    }
    Su = warp_sum_ll(Su); Sv = warp_sum_ll(Sv); Sw = warp_sum_ll(Sw);
    Suu = warp_sum_ll(Suu); Suv = warp_sum_ll(Suv); Suw = warp_sum_ll(Suw);
    if (lane == 0) {
      // n < 2^13 and |coord| < 2^17: n*Suu, Su^2, n*Suv, Su*Sv all stay below 2^60
      const long long N = n, den = N * Suu - Su * Su;
      emu_fit f;
      f.axis = u; f.n = n; f.u_min = lo[u]; f.u_max = hi[u];
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
      fits[t] = f;
    }
  }
}

}  // namespace

int emu_fit_launch(const int32_t* d_grains, const emu_track* d_tracks, const int32_t* d_track_off,
                   const int32_t* d_members, int32_t n_views, emu_fit* d_fits, cudaStream_t st) {
  EMU_LAUNCH(EMU_STAGE_FIT, st, k_fit<<<emu_sm_count() * 4, 256, 0, st>>>((const int4*)d_grains, d_tracks, d_track_off, d_members, n_views, d_fits));
  return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
}
