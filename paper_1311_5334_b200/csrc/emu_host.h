// emu_host.h - host-side helpers and the launcher prototypes behind the C ABI (emu_api.cu).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "emu_dev.cuh"

static inline size_t emu_align256(size_t x) { return (x + 255) & ~(size_t)255; }
static inline void* emu_align_ptr(void* p) { return (void*)(((uintptr_t)p + 255) & ~(uintptr_t)255); }
static inline int64_t emu_min64(int64_t a, int64_t b) { return a < b ? a : b; }
static inline int64_t emu_max64(int64_t a, int64_t b) { return a > b ? a : b; }

int emu_sm_count();     // multiprocessors of the current device (grids are sized in multiples of it)

// ---- optional per-stage timing (emu_profile_* of include/emu.h) -------------------------------
// While a profile is active on the calling host thread, every kernel launch of the library is
// bracketed by a pair of CUDA events on the launch stream and counted.  Without one, EMU_LAUNCH
// is just the launch.
struct emu_profile;
emu_profile* emu_prof_current();
void emu_prof_before(emu_profile* p, int stage, cudaStream_t st);
void emu_prof_after(emu_profile* p, int stage, cudaStream_t st);
#define EMU_LAUNCH(stage, st, ...)                          \
  do {                                                      \
    emu_profile* prof__ = emu_prof_current();               \
    if (prof__) emu_prof_before(prof__, (stage), (st));     \
    __VA_ARGS__;                                            \
    if (prof__) emu_prof_after(prof__, (stage), (st));      \
  } while (0)

// emu_bin.cu
size_t emu_bin_ws_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views);
// frame 0: the C ABI's A1 (w := row).  frames 1, 2: d_grains is frame 0's output (w = row is kept), the output
// holds the grains in the frame's coordinates (emu_dev.cuh "Frames").
int emu_bin_launch(const EmuDev& P, int frame, const int32_t* d_grains, const int32_t* d_view_off, int64_t n_grains,
                   int32_t n_views, int32_t* d_sorted, int32_t* d_cell_start, int64_t* d_status, void* d_ws,
                   size_t ws_bytes, cudaStream_t st);

// emu_find.cu
size_t emu_find_ws_min_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views);
size_t emu_find_ws_recommended_bytes(const EmuDev& P, int64_t n_grains, int32_t n_views, int seeds_per_grain,
                                     int cand_per_grain);
int emu_find_launch(const EmuDev& P, int seeds_per_grain, int cand_per_grain, const int32_t* d_sorted, const int32_t* d_cell_start,
                    const int32_t* d_view_off, int64_t n_grains, int32_t n_views, emu_track* d_tracks,
                    int32_t* d_track_off, int32_t* d_members, int64_t members_capacity, int64_t* d_counts,
                    void* d_ws, size_t ws_bytes, cudaStream_t st);
int emu_count_seeds_launch(const EmuDev& P, int seeds_per_grain, int cand_per_grain, const int32_t* d_sorted, const int32_t* d_cell_start,
                           const int32_t* d_view_off, int64_t n_grains, int32_t n_views, int32_t* d_seed_dump,
                           int64_t dump_capacity, int64_t* d_counts, void* d_ws, size_t ws_bytes,
                           cudaStream_t st);

// emu_recognize.cu
int emu_recognize_launch(const uint8_t* d_vox, int32_t n_views, int32_t nx, int32_t ny, int32_t nz, int32_t thr,
                         const int32_t* pitch_q, int32_t* d_grains, int64_t capacity, int32_t* d_view_off,
                         int64_t* d_count, int64_t* d_status, void* d_ws, size_t ws_bytes, cudaStream_t st);

// emu_fit.cu
int emu_fit_launch(const int32_t* d_grains, const emu_track* d_tracks, const int32_t* d_track_off,
                   const int32_t* d_members, int32_t n_views, emu_fit* d_fits, cudaStream_t st);
