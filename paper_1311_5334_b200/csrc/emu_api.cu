// emu_api.cu - the C ABI of include/emu.h: argument validation and marshalling only; every step of
// the path runs in the kernels of emu_bin.cu / emu_find.cu / emu_fit.cu.
#include <math.h>

#include <mutex>
#include <new>
#include <vector>

#include "emu_dev.cuh"
#include "emu_host.h"

namespace {

bool params_ok(const emu_params* p) {
  if (!p || p->struct_size != (int32_t)sizeof(emu_params)) return false;
  for (int i = 0; i < 3; ++i)
    if (p->view_size_q[i] < 1 || p->view_size_q[i] > 65536 || p->cell_size_q[i] < 1) return false;
  if (p->sep_min_q < 1 || p->sep_max_q <= p->sep_min_q || p->sep_max_q > 2048) return false;
  if (p->tube_r2_q < 0 || p->tube_r2_q >= (1 << 20)) return false;
  if (p->tube_ext_q < -1 || p->tube_ext_q > 65536) return false;   // -1 = whole line; >= 0 = bounded tube
  if (p->min_grains < 2 || p->min_grains > 8191) return false;
  if (p->max_tracks_per_view < 1 || p->max_tracks_per_view > 65536) return false;
  if (p->reserved[0] < 0 || p->reserved[1] < 0 || p->reserved[2] || p->reserved[3]) return false;
  for (int k = 0; k < 8; ++k) if (p->angle_min_grains[k] < 0 || p->angle_min_grains[k] > 8191) return false;
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
  d.Rup = (float)r;
  for (int i = 0; i < 3; ++i) {
    d.csf[i] = (float)d.cs[i];
    d.klo[i] = -(d.Rw * d.inv_cs[i] + 0.5f);
    d.khi[i] = d.Rw * d.inv_cs[i] - 0.5f;
  }
  // frames: permutations of the axes (emu_dev.cuh), the same cell size triple applied to (u,v,w)
  // 4-byte grains: u in 16 bits, v and w relative to their cell in 8 bits each (emu_find.cu)
  d.packed_ok = (d.cs[1] <= 256 && d.cs[2] <= 256) ? 1 : 0;
  for (int f = 0; f < 3; ++f) {
    int64_t fc = 1;
    for (int i = 0; i < 3; ++i) {
      d.fr[f].n[i] = (p->view_size_q[emu_frame_axis(f, i)] + d.cs[i] - 1) / d.cs[i];
      fc *= d.fr[f].n[i];
    }
    d.fr[f].ncell = fc > 0x7fffffff ? -1 : (int)fc;
    if ((int64_t)d.fr[f].n[0] * d.cs[0] > 65536) d.packed_ok = 0;
  }
  d.ext = p->tube_ext_q;
  d.angle_cut = 0;
  for (int k = 0; k < 8; ++k) {
    d.angle_min[k] = p->angle_min_grains[k];
    if (d.angle_min[k] > p->min_grains) d.angle_cut = 1;
  }
  d.min_grains = p->min_grains;
  d.max_tracks = p->max_tracks_per_view;
  return d;
}

bool shape_ok(const EmuDev& d, int64_t n_grains, int32_t n_views) {
  if (d.ncell < 1 || n_views < 0 || n_grains < 0 || n_grains >= ((int64_t)1 << 31) - 64) return false;
  for (int f = 0; f < 3; ++f)
    if (d.fr[f].ncell < 1 || (int64_t)n_views * d.fr[f].ncell >= ((int64_t)1 << 31) - 64) return false;
  return true;
}

bool aligned16(const void* p) { return ((uintptr_t)p & 15) == 0; }
int cand_per_grain(const emu_params* p) { return p->reserved[0] > 0 ? p->reserved[0] : 48; }
int seeds_per_grain(const emu_params* p) { return p->reserved[1] > 0 ? p->reserved[1] : 192; }

}  // namespace

int emu_sm_count() {
  int dev = 0, v = 0;
  if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) return v;
  return 148;                                     // B200
}

// ---- per-stage timing ---------------------------------------------------------------------------
struct emu_profile {
  struct Rec { int stage; cudaEvent_t a, b; };
  std::vector<Rec> recs;              // recorded since the last read
  std::vector<cudaEvent_t> pool;      // events free for reuse
  cudaEvent_t take() {
    if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
  }
};
static thread_local emu_profile* g_prof = nullptr;
emu_profile* emu_prof_current() { return g_prof; }
void emu_prof_before(emu_profile* p, int stage, cudaStream_t st) {
  emu_profile::Rec r; r.stage = stage; r.a = p->take(); r.b = p->take();
  cudaEventRecord(r.a, st);
  p->recs.push_back(r);
}
void emu_prof_after(emu_profile* p, int, cudaStream_t st) { cudaEventRecord(p->recs.back().b, st); }

extern "C" {

emu_profile* emu_profile_create(void) { return new (std::nothrow) emu_profile(); }
void emu_profile_destroy(emu_profile* p) {
  if (!p) return;
  if (g_prof == p) g_prof = nullptr;
  for (auto& r : p->recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (auto e : p->pool) cudaEventDestroy(e);
  delete p;
}
int emu_profile_begin(emu_profile* p) {
  if (!p || g_prof) return EMU_ERR_INVALID;
  g_prof = p;
  return EMU_OK;
}
int emu_profile_end(void) { g_prof = nullptr; return EMU_OK; }
int emu_profile_read(emu_profile* p, double* ms, int64_t* launches) {
  if (!p) return EMU_ERR_INVALID;
  int rc = EMU_OK;
  for (auto& r : p->recs) {
    float t = 0.f;
    if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&t, r.a, r.b) != cudaSuccess) rc = EMU_ERR_CUDA;
    if (r.stage >= 0 && r.stage < EMU_STAGE_COUNT) {
      if (ms) ms[r.stage] += (double)t;
      if (launches) launches[r.stage] += 1;
    }
    p->pool.push_back(r.a); p->pool.push_back(r.b);
  }
  p->recs.clear();
  return rc;
}

int emu_workspace_bytes(const emu_params* params, int64_t n_grains, int32_t n_views, size_t* bin_bytes,
                        size_t* find_bytes) {
  if (!params_ok(params)) return EMU_ERR_INVALID;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, n_grains, n_views)) return EMU_ERR_INVALID;
  if (bin_bytes) *bin_bytes = emu_bin_ws_bytes(d, n_grains, n_views);
  if (find_bytes) *find_bytes = emu_find_ws_recommended_bytes(d, n_grains, n_views, seeds_per_grain(params), cand_per_grain(params));
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
  return emu_bin_launch(d, 0, d_grains, d_view_off, n_grains, n_views, d_sorted, d_cell_start, d_status, d_ws, ws_bytes,
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
  return emu_find_launch(d, seeds_per_grain(params), cand_per_grain(params), d_sorted, d_cell_start, d_view_off, n_grains, n_views, d_tracks,
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
  return emu_count_seeds_launch(d, seeds_per_grain(params), cand_per_grain(params), d_sorted, d_cell_start, d_view_off, n_grains, n_views, d_seed_dump, dump_capacity,
                                d_counts, d_ws, ws_bytes, (cudaStream_t)stream);
}

namespace {
struct HostArena {
  int32_t *grains, *view_off, *sorted, *cell_start, *track_off, *members;
  emu_track* tracks; emu_fit* fits; int64_t* counts; int64_t* status; void* ws;
  size_t ws_bytes, total;
};
// carve (base may be NULL: then only the sizes are computed)
void carve_host_arena(const emu_params* p, const EmuDev& d, int64_t n, int32_t nv, char* base, HostArena& A) {
  size_t off = 0;
  auto take = [&](size_t bytes) { char* r = base ? base + off : nullptr; off += emu_align256(bytes ? bytes : 1); return r; };
  const size_t tcap = (size_t)(nv > 0 ? nv : 1) * (size_t)p->max_tracks_per_view;
  A.grains = (int32_t*)take((size_t)n * 16);
  A.view_off = (int32_t*)take(((size_t)nv + 1) * 4);
  A.sorted = (int32_t*)take((size_t)n * 16);
  A.cell_start = (int32_t*)take(((size_t)nv * d.ncell + 1) * 4);
  A.tracks = (emu_track*)take(tcap * sizeof(emu_track));
  A.fits = (emu_fit*)take(tcap * sizeof(emu_fit));
  A.track_off = (int32_t*)take(((size_t)nv + 1) * 4);
  A.members = (int32_t*)take((size_t)n * 4);
  A.counts = (int64_t*)take(8 * 8);
  A.status = (int64_t*)take(8);
  size_t b = emu_bin_ws_bytes(d, n, nv), f = emu_find_ws_recommended_bytes(d, n, nv, seeds_per_grain(p), cand_per_grain(p));
  A.ws_bytes = b > f ? b : f;
  A.ws = take(A.ws_bytes);
  A.total = off + 256;
}
}  // namespace

int emu_host_arena_bytes(const emu_params* params, int64_t n_grains, int32_t n_views, size_t* arena_bytes) {
  if (!params_ok(params) || !arena_bytes) return EMU_ERR_INVALID;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, n_grains, n_views)) return EMU_ERR_INVALID;
  HostArena A;
  carve_host_arena(params, d, n_grains, n_views, nullptr, A);
  *arena_bytes = A.total;
  return EMU_OK;
}

int emu_track_views_host(const emu_params* params, const int32_t* h_grains, const int32_t* h_view_off,
                         int64_t n_grains, int32_t n_views, emu_track* h_tracks, emu_fit* h_fits,
                         int64_t tracks_capacity, int32_t* h_track_off, int32_t* h_members,
                         int64_t members_capacity, int64_t* h_counts, void* d_arena, size_t arena_bytes,
                         void* stream) {
  if (!params_ok(params)) return EMU_ERR_INVALID;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, n_grains, n_views)) return EMU_ERR_INVALID;
  if (!h_view_off || !h_track_off || !h_counts || !d_arena || tracks_capacity < 0 || members_capacity < 0) return EMU_ERR_INVALID;
  if (n_grains > 0 && !h_grains) return EMU_ERR_INVALID;
  HostArena A;
  carve_host_arena(params, d, n_grains, n_views, (char*)emu_align_ptr(d_arena), A);
  if (arena_bytes < A.total) return EMU_ERR_CAPACITY;
  cudaStream_t st = (cudaStream_t)stream;
  if (n_grains > 0 && cudaMemcpyAsync(A.grains, h_grains, (size_t)n_grains * 16, cudaMemcpyHostToDevice, st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaMemcpyAsync(A.view_off, h_view_off, ((size_t)n_views + 1) * 4, cudaMemcpyHostToDevice, st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaMemsetAsync(A.status, 0, 8, st) != cudaSuccess) return EMU_ERR_CUDA;
  int rc = emu_bin_launch(d, 0, A.grains, A.view_off, n_grains, n_views, A.sorted, A.cell_start, A.status, A.ws, A.ws_bytes, st);
  if (rc != EMU_OK) return rc;
  rc = emu_find_launch(d, seeds_per_grain(params), cand_per_grain(params), A.sorted, A.cell_start, A.view_off, n_grains, n_views, A.tracks,
                       A.track_off, A.members, n_grains, A.counts, A.ws, A.ws_bytes, st);
  if (rc != EMU_OK) return rc;
  rc = emu_fit_launch(A.grains, A.tracks, A.track_off, A.members, n_views, A.fits, st);
  if (rc != EMU_OK) return rc;
  int64_t status = 0;
  if (cudaMemcpyAsync(h_counts, A.counts, 64, cudaMemcpyDeviceToHost, st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaMemcpyAsync(&status, A.status, 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaMemcpyAsync(h_track_off, A.track_off, ((size_t)n_views + 1) * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return EMU_ERR_CUDA;
  h_counts[EMU_CNT_STATUS] |= status;
  const int64_t nt = h_counts[EMU_CNT_TRACKS], nm = h_counts[EMU_CNT_MEMBERS];
  if (h_counts[EMU_CNT_STATUS] != 0) return EMU_OK;            // device-side condition: outputs unspecified
  if (nt > tracks_capacity || nm > members_capacity) return EMU_ERR_CAPACITY;
  if (nt > 0 && (!h_tracks || !h_fits)) return EMU_ERR_INVALID;
  if (nm > 0 && !h_members) return EMU_ERR_INVALID;
  if (nt > 0) {
    if (cudaMemcpyAsync(h_tracks, A.tracks, (size_t)nt * sizeof(emu_track), cudaMemcpyDeviceToHost, st) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaMemcpyAsync(h_fits, A.fits, (size_t)nt * sizeof(emu_fit), cudaMemcpyDeviceToHost, st) != cudaSuccess) return EMU_ERR_CUDA;
  }
  if (nm > 0 && cudaMemcpyAsync(h_members, A.members, (size_t)nm * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return EMU_ERR_CUDA;
  return EMU_OK;
}

// ---- streaming (include/emu.h): two slots of inputs / outputs, one workspace, three streams ----------------------
struct emu_stream {
  emu_params params; EmuDev dev;
  int64_t max_grains; int32_t max_views;
  cudaStream_t s_in, s_run, s_out;
  struct Slot {
    int32_t *grains, *view_off, *track_off, *members; emu_track* tracks; emu_fit* fits; int64_t *counts, *status;
    cudaEvent_t in_done, run_done;
    int64_t n_grains; int32_t n_views;
    int64_t* h_small;                      // pinned: counts[8], status
  } slot[2];
  int32_t *sorted, *cell_start; void* ws; size_t ws_bytes;
  unsigned long long submitted, collected;
};

namespace {
size_t stream_carve(const emu_params* p, const EmuDev& d, int64_t n, int32_t nv, char* base, emu_stream* S) {
  size_t off = 0;
  auto take = [&](size_t bytes) { char* r = base ? base + off : nullptr; off += emu_align256(bytes ? bytes : 1); return r; };
  const size_t tcap = (size_t)(nv > 0 ? nv : 1) * (size_t)p->max_tracks_per_view;
  for (int k = 0; k < 2; ++k) {
    int32_t* g = (int32_t*)take((size_t)n * 16); int32_t* vo = (int32_t*)take(((size_t)nv + 1) * 4);
    emu_track* t = (emu_track*)take(tcap * sizeof(emu_track)); emu_fit* f = (emu_fit*)take(tcap * sizeof(emu_fit));
    int32_t* to = (int32_t*)take(((size_t)nv + 1) * 4); int32_t* m = (int32_t*)take((size_t)n * 4);
    int64_t* c = (int64_t*)take(64); int64_t* st = (int64_t*)take(8);
    if (S) { auto& L = S->slot[k]; L.grains = g; L.view_off = vo; L.tracks = t; L.fits = f; L.track_off = to; L.members = m; L.counts = c; L.status = st; }
  }
  int32_t* srt = (int32_t*)take((size_t)n * 16);
  int32_t* cs = (int32_t*)take(((size_t)nv * d.ncell + 1) * 4);
  const size_t b = emu_bin_ws_bytes(d, n, nv), f = emu_find_ws_recommended_bytes(d, n, nv, seeds_per_grain(p), cand_per_grain(p));
  const size_t wsb = b > f ? b : f;
  void* ws = take(wsb);
  if (S) { S->sorted = srt; S->cell_start = cs; S->ws = ws; S->ws_bytes = wsb; }
  return off + 256;
}
}  // namespace

int emu_stream_arena_bytes(const emu_params* params, int64_t max_grains, int32_t max_views, size_t* arena_bytes) {
  if (!params_ok(params) || !arena_bytes) return EMU_ERR_INVALID;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, max_grains, max_views)) return EMU_ERR_INVALID;
  *arena_bytes = stream_carve(params, d, max_grains, max_views, nullptr, nullptr);
  return EMU_OK;
}

emu_stream* emu_stream_create(const emu_params* params, int64_t max_grains, int32_t max_views, void* d_arena, size_t arena_bytes) {
  if (!params_ok(params) || !d_arena) return nullptr;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, max_grains, max_views)) return nullptr;
  if (arena_bytes < stream_carve(params, d, max_grains, max_views, nullptr, nullptr)) return nullptr;
  emu_stream* S = new (std::nothrow) emu_stream();
  if (!S) return nullptr;
  S->params = *params; S->dev = d; S->max_grains = max_grains; S->max_views = max_views;
  S->submitted = S->collected = 0;
  S->s_in = S->s_run = S->s_out = nullptr;
  for (int k = 0; k < 2; ++k) { S->slot[k].in_done = S->slot[k].run_done = nullptr; S->slot[k].h_small = nullptr; }
  stream_carve(params, d, max_grains, max_views, (char*)emu_align_ptr(d_arena), S);
  bool ok = cudaStreamCreateWithFlags(&S->s_in, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&S->s_run, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&S->s_out, cudaStreamNonBlocking) == cudaSuccess;
  for (int k = 0; k < 2 && ok; ++k)
    ok = cudaEventCreateWithFlags(&S->slot[k].in_done, cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&S->slot[k].run_done, cudaEventDisableTiming) == cudaSuccess &&
         cudaMallocHost((void**)&S->slot[k].h_small, 16 * sizeof(int64_t)) == cudaSuccess;
  if (!ok) { emu_stream_destroy(S); return nullptr; }
  return S;
}

void emu_stream_destroy(emu_stream* S) {
  if (!S) return;
  if (S->s_in) { cudaStreamSynchronize(S->s_in); cudaStreamDestroy(S->s_in); }
  if (S->s_run) { cudaStreamSynchronize(S->s_run); cudaStreamDestroy(S->s_run); }
  if (S->s_out) { cudaStreamSynchronize(S->s_out); cudaStreamDestroy(S->s_out); }
  for (int k = 0; k < 2; ++k) {
    if (S->slot[k].in_done) cudaEventDestroy(S->slot[k].in_done);
    if (S->slot[k].run_done) cudaEventDestroy(S->slot[k].run_done);
    if (S->slot[k].h_small) cudaFreeHost(S->slot[k].h_small);
  }
  delete S;
}

int emu_stream_submit(emu_stream* S, const int32_t* h_grains, const int32_t* h_view_off, int64_t n_grains, int32_t n_views) {
  if (!S || !h_view_off || n_grains < 0 || n_views < 0 || (n_grains > 0 && !h_grains)) return EMU_ERR_INVALID;
  if (n_grains > S->max_grains || n_views > S->max_views) return EMU_ERR_INVALID;
  if (S->submitted - S->collected >= 2) return EMU_ERR_CAPACITY;            // both slots are in flight
  auto& L = S->slot[S->submitted & 1];
  const EmuDev& d = S->dev;
  // the slot's buffers are free: its previous batch was collected (collect waits for the kernels and the output copy)
  auto enqueue = [&]() -> int {
    if (n_grains > 0 && cudaMemcpyAsync(L.grains, h_grains, (size_t)n_grains * 16, cudaMemcpyHostToDevice, S->s_in) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaMemcpyAsync(L.view_off, h_view_off, ((size_t)n_views + 1) * 4, cudaMemcpyHostToDevice, S->s_in) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaEventRecord(L.in_done, S->s_in) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaStreamWaitEvent(S->s_run, L.in_done, 0) != cudaSuccess) return EMU_ERR_CUDA;
    cudaStream_t st = S->s_run;
    if (cudaMemsetAsync(L.status, 0, 8, st) != cudaSuccess) return EMU_ERR_CUDA;
    int rc = emu_bin_launch(d, 0, L.grains, L.view_off, n_grains, n_views, S->sorted, S->cell_start, L.status, S->ws, S->ws_bytes, st);
    if (rc != EMU_OK) return rc;
    rc = emu_find_launch(d, seeds_per_grain(&S->params), cand_per_grain(&S->params), S->sorted, S->cell_start, L.view_off, n_grains, n_views,
                         L.tracks, L.track_off, L.members, n_grains, L.counts, S->ws, S->ws_bytes, st);
    if (rc != EMU_OK) return rc;
    rc = emu_fit_launch(L.grains, L.tracks, L.track_off, L.members, n_views, L.fits, st);
    if (rc != EMU_OK) return rc;
    if (cudaMemcpyAsync(L.h_small, L.counts, 64, cudaMemcpyDeviceToHost, st) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaMemcpyAsync(L.h_small + 8, L.status, 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return EMU_ERR_CUDA;
    if (cudaEventRecord(L.run_done, st) != cudaSuccess) return EMU_ERR_CUDA;
    return EMU_OK;
  };
  const int erc = enqueue();
  if (erc != EMU_OK) {
    // part of the batch may already be queued (copies, kernels).  Nothing of it will be collected - `submitted` does
    // not advance - so drain both streams before handing the error back: the slot and the shared work buffers are
    // idle again and the next submit may reuse them.  (A sticky CUDA error makes these calls fail too; the caller
    // then sees EMU_ERR_CUDA from every later call and has to destroy the stream object.)
    cudaStreamSynchronize(S->s_in);
    cudaStreamSynchronize(S->s_run);
    return erc;
  }
  L.n_grains = n_grains; L.n_views = n_views;
  return (int)(S->submitted++ & 0x3fffffff);
}

int emu_stream_collect(emu_stream* S, emu_track* h_tracks, emu_fit* h_fits, int64_t tracks_capacity, int32_t* h_track_off,
                       int32_t* h_members, int64_t members_capacity, int64_t* h_counts) {
  if (!S || !h_track_off || !h_counts || tracks_capacity < 0 || members_capacity < 0) return EMU_ERR_INVALID;
  if (S->collected == S->submitted) return EMU_ERR_INVALID;                 // nothing in flight
  auto& L = S->slot[S->collected & 1];
  S->collected++;                                                          // the slot is given back whatever happens
  if (cudaEventSynchronize(L.run_done) != cudaSuccess) return EMU_ERR_CUDA;
  for (int k = 0; k < 8; ++k) h_counts[k] = L.h_small[k];
  h_counts[EMU_CNT_STATUS] |= L.h_small[8];
  cudaStream_t so = S->s_out;
  if (cudaMemcpyAsync(h_track_off, L.track_off, ((size_t)L.n_views + 1) * 4, cudaMemcpyDeviceToHost, so) != cudaSuccess) return EMU_ERR_CUDA;
  const int64_t nt = h_counts[EMU_CNT_TRACKS], nm = h_counts[EMU_CNT_MEMBERS];
  int rc = EMU_OK;
  if (h_counts[EMU_CNT_STATUS] == 0) {
    if (nt > tracks_capacity || nm > members_capacity) rc = EMU_ERR_CAPACITY;
    else if ((nt > 0 && (!h_tracks || !h_fits)) || (nm > 0 && !h_members)) rc = EMU_ERR_INVALID;
    else {
      if (nt > 0) {
        if (cudaMemcpyAsync(h_tracks, L.tracks, (size_t)nt * sizeof(emu_track), cudaMemcpyDeviceToHost, so) != cudaSuccess) rc = EMU_ERR_CUDA;
        if (cudaMemcpyAsync(h_fits, L.fits, (size_t)nt * sizeof(emu_fit), cudaMemcpyDeviceToHost, so) != cudaSuccess) rc = EMU_ERR_CUDA;
      }
      if (nm > 0 && cudaMemcpyAsync(h_members, L.members, (size_t)nm * 4, cudaMemcpyDeviceToHost, so) != cudaSuccess) rc = EMU_ERR_CUDA;
    }
  }
  if (cudaStreamSynchronize(so) != cudaSuccess) return EMU_ERR_CUDA;
  return rc;
}

int emu_recognize_grains(const uint8_t* d_vox, int32_t n_views, int32_t nx, int32_t ny, int32_t nz, int32_t threshold,
                         const int32_t* pitch_q, int32_t* d_grains, int64_t capacity, int32_t* d_view_off,
                         int64_t* d_count, int64_t* d_status, void* d_ws, size_t ws_bytes, void* stream) {
  if (n_views < 0 || nx < 1 || ny < 1 || nz < 1 || threshold < 0 || threshold > 254 || capacity < 0) return EMU_ERR_INVALID;
  if ((int64_t)n_views * ny * nz >= ((int64_t)1 << 31) - 64 || nx > 65535) return EMU_ERR_INVALID;
  if (!pitch_q || !d_view_off || !d_count || !d_status || !d_ws || (n_views > 0 && !d_vox) || (capacity > 0 && !d_grains)) return EMU_ERR_INVALID;
  for (int a = 0; a < 3; ++a) if (pitch_q[a] < 1 || pitch_q[a] > 4096) return EMU_ERR_INVALID;
  if (!aligned16(d_grains)) return EMU_ERR_INVALID;
  return emu_recognize_launch(d_vox, n_views, nx, ny, nz, threshold, pitch_q, d_grains, capacity, d_view_off, d_count,
                              d_status, d_ws, ws_bytes, (cudaStream_t)stream);
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

// ---- emu_bin_grains_noalloc: A1 for callers that have no device memory to give as a workspace --------------------
// (include/emu.h has the contract.)  The binning kernels need scratch next to their inputs and outputs: the per-cell
// counters, the staging copy of the grains between the two passes, the per-view redo flags and chunk cursors.  The
// normal entry point takes it from the caller; this one keeps a fixed block of it inside the library image, so every
// device that loads libemu4pi.so carries EMU_BIN_NOALLOC_BYTES of it until the process exits, used or not.
//
// g_bin_scratch below is a DEVICE array.  On the host its name is only a handle for the runtime - not an address a
// kernel may be given - so the device address is asked for once per device with cudaGetSymbolAddress, with that device
// current, and it is this address that goes to the launcher.
static __device__ __align__(256) unsigned char g_bin_scratch[EMU_BIN_NOALLOC_BYTES];

namespace {
constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
void* g_noalloc_ptr[kNoallocMaxDevices];          // device address of g_bin_scratch on device i, NULL = not asked yet

// the scratch of the CURRENT device (first call on a device: one cudaGetSymbolAddress; afterwards a table look-up)
int noalloc_scratch(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return EMU_ERR_CUDA;
  if (dev < 0 || dev >= kNoallocMaxDevices) return EMU_ERR_INVALID;
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_bin_scratch) != cudaSuccess || !p) return EMU_ERR_CUDA;
    g_noalloc_ptr[dev] = p;
  }
  *out = g_noalloc_ptr[dev];
  return EMU_OK;
}
}  // namespace

extern "C" {

size_t emu_bin_noalloc_max_bytes(void) { return (size_t)EMU_BIN_NOALLOC_BYTES; }

int emu_bin_grains_noalloc(const emu_params* params, const int32_t* d_grains, const int32_t* d_view_off, int64_t n_grains,
                           int32_t n_views, int32_t* d_sorted, int32_t* d_cell_start, int64_t* d_status, void* stream) {
  if (!params_ok(params)) return EMU_ERR_INVALID;
  EmuDev d = make_dev(params);
  if (!shape_ok(d, n_grains, n_views)) return EMU_ERR_INVALID;
  if (!d_view_off || !d_cell_start || !d_status) return EMU_ERR_INVALID;
  if (n_grains > 0 && (!d_grains || !d_sorted)) return EMU_ERR_INVALID;
  if (!aligned16(d_grains) || !aligned16(d_sorted)) return EMU_ERR_INVALID;
  // the size check comes first and runs on the host alone: a batch beyond the fixed block is refused before any CUDA call
  if (emu_bin_ws_bytes(d, n_grains, n_views) > (size_t)EMU_BIN_NOALLOC_BYTES) return EMU_ERR_CAPACITY;
  void* scratch = nullptr;
  const int rc = noalloc_scratch(&scratch);
  if (rc != EMU_OK) return rc;
  // the block still holds whatever the previous call left in it.  The launcher does not rely on its contents: what has
  // to start at zero (redo flags, chunk cursors, the global counters of the counting-sort path) it clears itself with
  // cudaMemsetAsync on `stream`, ahead of the kernels, exactly as it does for a caller's uninitialised workspace.
  return emu_bin_launch(d, 0, d_grains, d_view_off, n_grains, n_views, d_sorted, d_cell_start, d_status, scratch,
                        (size_t)EMU_BIN_NOALLOC_BYTES, (cudaStream_t)stream);
}

}  // extern "C"
