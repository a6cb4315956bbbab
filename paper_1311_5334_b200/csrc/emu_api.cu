// emu_api.cu - the C ABI of include/emu.h: argument validation and marshalling only; every step of
// the path runs in the kernels of emu_bin.cu / emu_find.cu / emu_fit.cu.
#include <math.h>

#include "emu_dev.cuh"
#include "emu_host.h"

namespace {

bool params_ok(const emu_params* p) {
  if (!p || p->struct_size != (int32_t)sizeof(emu_params)) return false;
  for (int i = 0; i < 3; ++i)
    if (p->view_size_q[i] < 1 || p->view_size_q[i] > 65536 || p->cell_size_q[i] < 1) return false;
  if (p->sep_min_q < 1 || p->sep_max_q <= p->sep_min_q || p->sep_max_q > 2048) return false;
  if (p->tube_r2_q < 0 || p->tube_r2_q >= (1 << 20)) return false;
  if (p->tube_ext_q != -1) return false;            // bounded tube: DESIGN.md "next" row, not built
  if (p->min_grains < 2 || p->min_grains > 8191) return false;
  if (p->max_tracks_per_view < 1 || p->max_tracks_per_view > 65536) return false;
  if (p->reserved[0] < 0 || p->reserved[1] || p->reserved[2] || p->reserved[3]) return false;
  return true;
}

EmuDev make_dev(const emu_params* p) {
  EmuDev d;
  int64_t nc = 1;
  for (int i = 0; i < 3; ++i) {
    d.cs[i] = p->cell_size_q[i];
    d.n[i] = (p->view_size_q[i] + d.cs[i] - 1) / d.cs[i];
    d.inv_cs[i] = 1.0f / (float)d.cs[i];
    nc *= d.n[i];
  }
  d.ncell = nc > 0x7fffffff ? -1 : (int)nc;
  d.sep_max = p->sep_max_q;
  d.sep_min2 = p->sep_min_q * p->sep_min_q;
  d.sep_max2 = p->sep_max_q * p->sep_max_q;
  d.r2 = p->tube_r2_q;
  int r = 0; while ((int64_t)r * r < p->tube_r2_q) ++r;
  d.Rw = (float)(r + 2);
  d.min_grains = p->min_grains;
  d.max_tracks = p->max_tracks_per_view;
  return d;
}

bool shape_ok(const EmuDev& d, int64_t n_grains, int32_t n_views) {
  if (d.ncell < 1 || n_views < 0 || n_grains < 0 || n_grains >= ((int64_t)1 << 31) - 64) return false;
  if ((int64_t)n_views * d.ncell >= ((int64_t)1 << 31) - 64) return false;
  return true;
}

bool aligned16(const void* p) { return ((uintptr_t)p & 15) == 0; }
int cand_per_grain(const emu_params* p) { return p->reserved[0] > 0 ? p->reserved[0] : 48; }

}  // namespace

extern "C" {

int emu_workspace_bytes(const emu_params* params, int64_t n_grains, int32_t n_views, size_t* bin_bytes,
                        size_t* find_bytes) {
  if (!params_ok(params)) return EMU_ERR_INVALID;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, n_grains, n_views)) return EMU_ERR_INVALID;
  if (bin_bytes) *bin_bytes = emu_bin_ws_bytes(d, n_grains, n_views);
  if (find_bytes) *find_bytes = emu_find_ws_recommended_bytes(d, n_grains, n_views, cand_per_grain(params));
  return EMU_OK;
}

int64_t emu_grid_cells(const emu_params* params, int32_t dims_out[3]) {
  if (!params || params->struct_size != (int32_t)sizeof(emu_params)) return EMU_ERR_INVALID;
  int64_t nc = 1;
  for (int i = 0; i < 3; ++i) {
    if (params->view_size_q[i] < 1 || params->cell_size_q[i] < 1) return EMU_ERR_INVALID;
    int n = (params->view_size_q[i] + params->cell_size_q[i] - 1) / params->cell_size_q[i];
    if (dims_out) dims_out[i] = n;
    nc *= n;
  }
  return nc;
}

int emu_bin_grains(const emu_params* params, const int32_t* d_grains, const int32_t* d_view_off, int64_t n_grains,
                   int32_t n_views, int32_t* d_sorted, int32_t* d_cell_start, int64_t* d_status, void* d_ws,
                   size_t ws_bytes, void* stream) {
  if (!params_ok(params)) return EMU_ERR_INVALID;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, n_grains, n_views)) return EMU_ERR_INVALID;
  if (!d_view_off || !d_cell_start || !d_status || !d_ws) return EMU_ERR_INVALID;
  if (n_grains > 0 && (!d_grains || !d_sorted)) return EMU_ERR_INVALID;
  if (!aligned16(d_grains) || !aligned16(d_sorted)) return EMU_ERR_INVALID;
  return emu_bin_launch(d, d_grains, d_view_off, n_grains, n_views, d_sorted, d_cell_start, d_status, d_ws, ws_bytes,
                        (cudaStream_t)stream);
}

int emu_find_tracks(const emu_params* params, const int32_t* d_sorted, const int32_t* d_cell_start,
                    const int32_t* d_view_off, int64_t n_grains, int32_t n_views, emu_track* d_tracks,
                    int32_t* d_track_off, int32_t* d_members, int64_t members_capacity, int64_t* d_counts, void* d_ws,
                    size_t ws_bytes, void* stream) {
  if (!params_ok(params)) return EMU_ERR_INVALID;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, n_grains, n_views)) return EMU_ERR_INVALID;
  if (!d_view_off || !d_cell_start || !d_track_off || !d_counts || !d_ws || !d_tracks || !d_members) return EMU_ERR_INVALID;
  if (n_grains > 0 && !d_sorted) return EMU_ERR_INVALID;
  if (!aligned16(d_sorted) || !aligned16(d_tracks) || members_capacity < 0) return EMU_ERR_INVALID;
  return emu_find_launch(d, cand_per_grain(params), d_sorted, d_cell_start, d_view_off, n_grains, n_views, d_tracks,
                         d_track_off, d_members, members_capacity, d_counts, d_ws, ws_bytes, (cudaStream_t)stream);
}

int emu_count_seeds(const emu_params* params, const int32_t* d_sorted, const int32_t* d_cell_start,
                    const int32_t* d_view_off, int64_t n_grains, int32_t n_views, int32_t* d_seed_dump,
                    int64_t dump_capacity, int64_t* d_counts, void* d_ws, size_t ws_bytes, void* stream) {
  if (!params_ok(params)) return EMU_ERR_INVALID;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, n_grains, n_views)) return EMU_ERR_INVALID;
  if (!d_view_off || !d_cell_start || !d_counts || !d_ws || dump_capacity < 0) return EMU_ERR_INVALID;
  if (dump_capacity > 0 && !d_seed_dump) return EMU_ERR_INVALID;
  if (!aligned16(d_sorted) || !aligned16(d_seed_dump)) return EMU_ERR_INVALID;
  return emu_count_seeds_launch(d, d_sorted, d_cell_start, d_view_off, n_grains, n_views, d_seed_dump, dump_capacity,
                                d_counts, d_ws, ws_bytes, (cudaStream_t)stream);
}

int emu_fit_tracks(const emu_params* params, const int32_t* d_grains, const emu_track* d_tracks,
                   const int32_t* d_track_off, const int32_t* d_members, int32_t n_views, emu_fit* d_fits,
                   void* stream) {
  if (!params_ok(params) || n_views < 0) return EMU_ERR_INVALID;
  if (!d_tracks || !d_track_off || !d_members || !d_fits) return EMU_ERR_INVALID;   // d_grains may be NULL when there are no grains
  if (!aligned16(d_grains) || !aligned16(d_tracks) || ((uintptr_t)d_fits & 7)) return EMU_ERR_INVALID;
  return emu_fit_launch(d_grains, d_tracks, d_track_off, d_members, n_views, d_fits, (cudaStream_t)stream);
}

}  // extern "C"
