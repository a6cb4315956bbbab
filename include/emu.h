/* emu.h - C ABI of libemu4pi: 4pi track finding over the 3D grain cloud of emulsion views
 * (Ariga & Ariga, arXiv 1311.5334, section 2), hand-written CUDA for sm_100a (B200).
 *
 * Citations: P:NN = /root/reference/PAPER.md line NN; "reading Qn" = DESIGN.md section 3.
 *
 * Conventions for every call
 *  - Pointers prefixed d_ are DEVICE pointers owned by the CALLER (e.g. torch.empty(..., device="cuda")).
 *    `stream` is a cudaStream_t passed as void* (NULL = default stream).  The library keeps no global
 *    state, allocates no persistent memory and is re-entrant per stream.
 *  - Every call only ENQUEUES work on `stream` and returns without synchronising:
 *      EMU_OK            0
 *      EMU_ERR_INVALID  -1  null / misaligned pointer, bad params, a documented range violated
 *      EMU_ERR_CAPACITY -2  workspace (or an output array) too small, detected on the host
 *      EMU_ERR_CUDA     -3  a CUDA runtime call failed (cudaGetLastError != cudaSuccess)
 *    Conditions only the device can see (too many candidates / tracks / members, coordinates out of
 *    range) are reported in d_counts[EMU_CNT_STATUS]; outputs are then unspecified and the caller
 *    retries with larger buffers.  No exceptions, no aborts, no printing.
 *  - Units: q = 1/64 um; all coordinates int32.  |coordinate| < 2^17 (box <= 2^16 plus slack for
 *    out-of-box grains) so that every product of the tube test fits in 64 bits.
 *  - A "row" is a row index of the caller's d_grains array (the "original index" of a grain).
 */
#ifndef EMU_H_
#define EMU_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EMU_OK 0
#define EMU_ERR_INVALID (-1)
#define EMU_ERR_CAPACITY (-2)
#define EMU_ERR_CUDA (-3)

typedef struct emu_params {
  int32_t struct_size;         /* = sizeof(emu_params): ABI check                                          */
  int32_t view_size_q[3];      /* box [0,size) per axis; 1 <= size <= 65536 (1024 um)                      */
  int32_t cell_size_q[3];      /* > 0.  Paper: 32 px x 32 px x 1 frame.  Has NO effect on the      */
                               /* track list (reading Q10); it only steers the speed of the search.        */
                               /* emu_find_tracks bins every view twice more with permuted axes (y,x,z)    */
                               /* and (z,x,y) and applies the SAME triple to the permuted coordinates:     */
                               /* [0] = size along a line's dominant axis, [1], [2] = across it.           */
  int32_t sep_min_q;           /* seed <=> sep_min_q^2 <= D2 < sep_max_q^2 (reading Q1; "smaller      */
  int32_t sep_max_q;           /*  than 25 um" = 1600).  1 <= sep_min_q < sep_max_q <= 2048                */
  int32_t tube_r2_q;           /* tube radius squared, q^2; 0.8 um -> floor(0.64*4096) = 2621 (reading Q3) */
  int32_t tube_ext_q;          /* -1 = count along the whole line (reading Q4, the contract).  >= 0 (<=     */
                               /* 65536): bounded tube (Fig. 4(b) "along the seed"): a grain counts   */
                               /* only if its foot on the line lies between the seed grains or at most     */
                               /* tube_ext_q beyond either (exact: compared through squares in 64 bits)     */
  int32_t min_grains;          /* threshold, >= 2: n >= min_grains (reading Q6; "e.g. 5")             */
  int32_t max_tracks_per_view; /* capacity of the track list per view, 1..65536                            */
  int32_t reserved[4];         /* sizing hints for the internal chunks of emu_find_tracks:                 */
                               /* [0] = expected candidates per grain (0 = default 48; 48 B each),         */
                               /* [1] = expected seeds per grain (0 = default 192; 240 B each: geometry,   */
                               /*       counter, the hit record of the voting pass and 2.5 per-brick list  */
                               /*       records of 32 B); [2], [3] must be 0                               */
  int32_t angle_min_grains[8]; /* angle-dependent cut on the number of grains (Fig. 8(c): "a cut on */
                               /* the number of grains is applied according to the line drawn in the       */
                               /* figure"; the line is not given, hence a table - reading Q17): entry k    */
                               /* is the minimum n_members of a track whose FITTED direction has           */
                               /* floor(8 |cos theta|) = k (7 for |cos theta| = 1), theta = angle to z,    */
                               /* decided exactly in integers from the moments of emu_fit.  Applied after  */
                               /* the exclusive association; a track that fails is dropped and its grains  */
                               /* stay unassigned.  0 (or <= min_grains) = no cut in that bin; each 0..8191 */
} emu_params;

typedef struct emu_track {     /* 32 B */
  int32_t view;
  int32_t seed_a, seed_b;      /* rows of the two seed grains, seed_a < seed_b                             */
  int32_t n_tube;              /* grains inside the tube of the seed line, seed grains included     */
  int32_t n_members;           /* grains kept after the exclusive association                       */
  int32_t member_off;          /* first member in d_members                                                */
  int32_t seed_d2;             /* |B-A|^2 in q^2                                                           */
  int32_t pad;                 /* 0                                                                        */
} emu_track;

typedef struct emu_fit {       /* 48 B */
  int32_t axis;                /* dominant axis u: 0=x 1=y 2=z; |0x100 if all members share u (den = 0)    */
  int32_t n;                   /* members                                                                  */
  int32_t u_min, u_max;        /* extent of the members along u (segment start / end, Fig. 5), q      */
  double slope[2], icpt[2];    /* minor coords (x,y | y,z | x,z for u = z | x | y) = slope*u + icpt, q     */
} emu_fit;

/* d_counts[8] (int64), written by emu_find_tracks / emu_count_seeds */
#define EMU_CNT_SEEDS 0        /* grain pairs inside the separation window                          */
#define EMU_CNT_TESTS 1        /* point-line tests executed (implementation figure, not compared)          */
#define EMU_CNT_CANDIDATES 2   /* seeds with n_tube >= min_grains                                          */
#define EMU_CNT_TRACKS 3
#define EMU_CNT_MEMBERS 4
#define EMU_CNT_STATUS 5       /* 0 = fine, else OR of the EMU_ST_* bits                                   */
#define EMU_CNT_PAIR_TESTS 6   /* pair-distance tests executed (implementation figure)                     */
#define EMU_CNT_NEED 7         /* largest seed CAPACITY one internal chunk needed: its seeds, or - when a   */
                               /* seed's line crosses many bricks (fine cells, whole-line tube) - its      */
                               /* per-brick list records / 2.5, whichever is larger.  After                */
                               /* EMU_ST_SEED_OVERFLOW: raise reserved[1] to NEED / (grains of the chunk)  */
#define EMU_ST_CAND_OVERFLOW 1    /* candidate workspace too small: give more workspace / raise reserved[0] */
#define EMU_ST_TRACK_OVERFLOW 2   /* a view has more than max_tracks_per_view tracks                       */
#define EMU_ST_MEMBER_OVERFLOW 4  /* members_capacity too small                                            */
#define EMU_ST_RANGE 8            /* a count does not fit its field (n_tube >= 8192)                       */
#define EMU_ST_COORD 16           /* emu_bin_grains saw |coordinate| >= 2^17                               */
#define EMU_ST_SEED_OVERFLOW 32   /* seed workspace too small: give more workspace / raise reserved[1]     */
#define EMU_ST_GRAIN_OVERFLOW 64  /* emu_recognize_grains found more grains than d_grains can hold         */

/* Host-only (no CUDA call).  Workspace each call needs for this batch shape; both outputs optional.
 * find_bytes is a recommendation (internal view chunks adapt to whatever >= the minimum is given). */
int emu_workspace_bytes(const emu_params* params, int64_t n_grains, int32_t n_views,
                        size_t* bin_bytes, size_t* find_bytes);

/* Number of cells per view and grid dimensions, ceil(view_size/cell_size) per axis (the paper's
 * geometry 1280x1024x40 with cells 32x32x1 gives 40x32x40 = 51 200).  Host-only. */
int64_t emu_grid_cells(const emu_params* params, int32_t dims_out[3]);

/* A1 "3D hash table" ("All recognized grains are then attributed to these cells").
 *  in : d_grains  int32[n_grains][4] = x,y,z,w (w = caller payload, ignored), 16-byte aligned;
 *       d_view_off int32[n_views+1], non-decreasing, [0] = 0, [n_views] = n_grains < 2^31.
 *  out: d_sorted  int32[n_grains][4] = x,y,z,row ordered by (view, cell, row), where
 *       cell = cx + nx*(cy + ny*cz), c = clamp(floor(coord/cell_size), 0, n-1) (out-of-box grains are
 *       legal and land in the boundary cells, reading Q13);
 *       d_cell_start int32[n_views*n_cells+1]: first position in d_sorted of every (view, cell).
 *  d_status: int64[1], OR-ed with EMU_ST_COORD if a coordinate is out of range; never cleared here.  (Not
 *       d_counts + EMU_CNT_STATUS: emu_find_tracks zeroes all of d_counts when it starts.)
 *  d_ws / ws_bytes: scratch of at least the size emu_workspace_bytes reports. */
int emu_bin_grains(const emu_params* params, const int32_t* d_grains, const int32_t* d_view_off,
                   int64_t n_grains, int32_t n_views, int32_t* d_sorted, int32_t* d_cell_start,
                   int64_t* d_status, void* d_ws, size_t ws_bytes, void* stream);

/* A1 again, for callers that cannot hand over a workspace because they cannot allocate device memory at the point
 * where a view has to be binned.  Who that is: the thread that follows the microscope (a view every 0.2 s),
 * where a cudaMalloc or cudaFree would wait for every stream of the device and stall the camera copies running beside
 * it; a plug-in inside a process whose own memory pool already holds the whole HBM, so a further allocation fails; a
 * caller that was given input and output buffers by a framework and has no allocator of its own to ask for more.
 * Same inputs, outputs, ordering and status as emu_bin_grains (the kernels are the same ones); only d_ws / ws_bytes are
 * gone.  The scratch is a fixed block of EMU_BIN_NOALLOC_BYTES inside the library image: every GPU that loads the
 * library holds it from load until the process exits, whether or not this call is ever made.
 *  - Limit: emu_workspace_bytes(...)'s bin_bytes for the batch must be <= EMU_BIN_NOALLOC_BYTES (8 MiB: e.g. four
 *    views of 64 k grains in 114 k cells each).  A larger batch gets EMU_ERR_CAPACITY before anything is
 *    enqueued - split it into smaller calls, or use emu_bin_grains with a workspace.  emu_bin_noalloc_max_bytes() returns the limit.
 *  - The call makes no cudaMalloc / cudaFree and calls nothing that does (kernel launches and cudaMemsetAsync on
 *    `stream` only, with no emu_profile active).  The first call on each device looks up the device address of the
 *    block (one cudaGetSymbolAddress, with the caller's current device); make that first call at set-up time, on the
 *    device it will be used on and before any stream capture is begun; later calls on that device only read a table.
 *  - All calls on one device share the one block.  Nothing in it has to be cleared by the caller: whatever must start at
 *    zero is cleared on `stream` ahead of the kernels.  But two calls whose GPU work overlaps in time (different
 *    streams, or two host threads) write the same scratch and corrupt each other: keep them on one stream or order
 *    them with events.  emu_bin_grains with separate workspaces has no such restriction. */
#define EMU_BIN_NOALLOC_BYTES (8u << 20)
size_t emu_bin_noalloc_max_bytes(void);
int emu_bin_grains_noalloc(const emu_params* params, const int32_t* d_grains, const int32_t* d_view_off,
                           int64_t n_grains, int32_t n_views, int32_t* d_sorted, int32_t* d_cell_start,
                           int64_t* d_status, void* stream);

/* A2..A5 + A7: seeds -> tube count -> threshold -> exclusive association -> threshold -> order
 * (Fig. 4).
 *  in : d_sorted, d_cell_start as written by emu_bin_grains with the SAME params; d_view_off.
 *  out: d_tracks emu_track[<= n_views*max_tracks_per_view], written compactly: view v owns entries
 *       d_track_off[v] .. d_track_off[v+1]-1, best first (reading Q7 order); d_track_off int32[n_views+1];
 *       d_members int32[members_capacity]: rows, each track's members contiguous at member_off, ascending;
 *       d_counts int64[8] (see EMU_CNT_*), zeroed by the call. */
int emu_find_tracks(const emu_params* params, const int32_t* d_sorted, const int32_t* d_cell_start,
                    const int32_t* d_view_off, int64_t n_grains, int32_t n_views,
                    emu_track* d_tracks, int32_t* d_track_off, int32_t* d_members, int64_t members_capacity,
                    int64_t* d_counts, void* d_ws, size_t ws_bytes, void* stream);

/* A2 + A3 only, for per-seed parity checks: writes (view, row_a, row_b, n_tube), row_a < row_b, for
 * every seed, in no particular order, to d_seed_dump int32[dump_capacity][4].  d_counts[EMU_CNT_SEEDS]
 * receives the number of seeds (which may exceed dump_capacity; the excess is not written).
 * d_ws: scratch of the find_bytes emu_workspace_bytes reports; the batch must fit ONE internal chunk
 * (a test aid for a few views), else EMU_ERR_CAPACITY. */
int emu_count_seeds(const emu_params* params, const int32_t* d_sorted, const int32_t* d_cell_start,
                    const int32_t* d_view_off, int64_t n_grains, int32_t n_views,
                    int32_t* d_seed_dump, int64_t dump_capacity, int64_t* d_counts,
                    void* d_ws, size_t ws_bytes, void* stream);

/* A6 least-squares line per track (BASELINE.json north_star; reading Q9; not in the paper).
 *  in : d_grains in ORIGINAL order (members are rows of it); tracks / offsets / members from
 *       emu_find_tracks.  n_tracks is read on the device from d_track_off[n_views].
 *  out: d_fits emu_fit[same capacity as d_tracks], entry t for track t.
 *  Safe after a device-side overflow of emu_find_tracks (status != 0): the tracks of a chunk that overflowed are
 *  not emitted, and a track whose members did not fit members_capacity carries n_members = 0. */
int emu_fit_tracks(const emu_params* params, const int32_t* d_grains, const emu_track* d_tracks,
                   const int32_t* d_track_off, const int32_t* d_members, int32_t n_views,
                   emu_fit* d_fits, void* stream);

/* A0, upstream of the hot path: 3D grain recognition on stacks of filtered frames (P:68-70:
 * "Each pixel with a pulse height higher than a given threshold is compared to the 3 x 3 x 3 neighboring pixels; the
 * pixel with the highest pulse height among these will be defining the grain.  The spatial coordinates of the grains
 * are then computed with a center-of-mass method using the pulse height of each pixel").  Readings R1-R5, DESIGN.md 3b:
 * voxels outside the stack count as 0; of equal maxima the first in raster order (z, y, x) defines the grain; centre
 * of mass over the 3x3x3 neighbourhood with weight = pulse height where it exceeds the threshold, else 0;
 * pos_q = floor(pitch_q * (sum(w i) / sum(w) + 1/2) + 1/2) per axis, exact in integers.
 *  in : d_vox uint8[n_views][nz][ny][nx] (x fastest); threshold 0..254; pitch_q[3] = voxel pitch in q along x, y, z
 *       (HOST array, 1..4096 each); 1 <= nx <= 65535, ny, nz >= 1, n_views * ny * nz < 2^31.
 *  out: d_grains int32[<= capacity][4] = x_q, y_q, z_q, pulse height of the defining voxel, view after view, inside
 *       a view in raster order of the defining voxel - the layout emu_bin_grains takes (its w is payload);
 *       d_view_off int32[n_views+1]; d_count int64[1] = grains found (may exceed capacity: then d_status gets
 *       EMU_ST_GRAIN_OVERFLOW and the excess is not written); d_status int64[1], OR-ed, never cleared here.
 *  d_ws: scratch of emu_recognize_ws_bytes(n_views, ny, nz, capacity) bytes (a counter per row of voxels and a 32-byte
 *       staging record per grain d_grains can hold).  n_views, ny, nz <= 65535. */
size_t emu_recognize_ws_bytes(int32_t n_views, int32_t ny, int32_t nz, int64_t capacity);
int emu_recognize_grains(const uint8_t* d_vox, int32_t n_views, int32_t nx, int32_t ny, int32_t nz, int32_t threshold,
                         const int32_t* pitch_q, int32_t* d_grains, int64_t capacity, int32_t* d_view_off,
                         int64_t* d_count, int64_t* d_status, void* d_ws, size_t ws_bytes, void* stream);

/* ---- the whole path on HOST buffers (the end-to-end call: copies in, A1..A7, copies out) --------
 * h_* are HOST pointers owned by the caller (pinned memory makes the copies asynchronous and fast;
 * pageable memory works).  d_arena is one caller-owned DEVICE allocation of at least
 * emu_host_arena_bytes() bytes from which the call carves every device buffer it needs (input copy,
 * sorted grains, cell_start, outputs, workspaces).  Unlike the device calls above this one is
 * SYNCHRONOUS: it enqueues the host->device copies, emu_bin_grains, emu_find_tracks and
 * emu_fit_tracks on `stream`, reads d_counts back, copies the valid part of every output to the
 * host and returns after the stream has drained.
 *  out: h_tracks[<= tracks_capacity], h_fits[<= tracks_capacity], h_track_off[n_views+1],
 *       h_members[<= members_capacity], h_counts[8] (EMU_CNT_*; status includes EMU_ST_COORD).
 *  Returns EMU_ERR_CAPACITY if the arena or a host output array is too small for what was found
 *  (h_counts then still holds the required sizes), else as the device calls. */
int emu_host_arena_bytes(const emu_params* params, int64_t n_grains, int32_t n_views, size_t* arena_bytes);
int emu_track_views_host(const emu_params* params, const int32_t* h_grains, const int32_t* h_view_off,
                         int64_t n_grains, int32_t n_views, emu_track* h_tracks, emu_fit* h_fits,
                         int64_t tracks_capacity, int32_t* h_track_off, int32_t* h_members,
                         int64_t members_capacity, int64_t* h_counts, void* d_arena, size_t arena_bytes,
                         void* stream);

/* ---- streaming: batches of views through one GPU, copies overlapped with the kernels -------
 * The microscope delivers a view every 0.2 s and the paper's run spends 0.04 of 0.14 s per view on I/O
 * (P:136).  An emu_stream is a host-side object that owns three CUDA streams (copy-in, compute, copy-out), a few
 * events and a small pinned staging buffer; the device memory is the CALLER's: one arena of emu_stream_arena_bytes()
 * from which it carves TWO slots of inputs and outputs and ONE set of work buffers (the kernels of successive batches
 * run one after the other on the compute stream, so they can share the workspace).
 *   submit(k)   host->device copy of batch k on the copy-in stream, A1..A7 on the compute stream behind batch k-1;
 *               returns at once.  At most two batches may be in flight; a third submit returns EMU_ERR_CAPACITY.
 *               h_grains / h_view_off (HOST, pinned for a truly asynchronous copy) must stay untouched until collect.
 *   collect()   waits for the OLDEST batch in flight, copies the valid part of its outputs to the host arrays on the
 *               copy-out stream (while the next batch computes) and returns when they have arrived.  Outputs and
 *               return codes as emu_track_views_host.
 * With submit(k+1) called before collect(k), the input copy of k+1 and the output copy of k-1 hide behind the
 * kernels of k.  Every batch must satisfy n_grains <= max_grains, n_views <= max_views.
 * The three streams are the object's own (non-blocking) and are not ordered against any stream of the caller: d_arena
 * must be IDLE when emu_stream_create is called (no work still queued anywhere that reads or writes it - with a caching
 * allocator, synchronise the stream it was last used on) and must not be touched by the caller until destroy.
 * If submit fails after part of the batch was queued (a launcher's error code, EMU_ERR_CUDA), it drains its copy-in and
 * compute streams before returning: the batch does not count as in flight, nothing is left running, and the next
 * submit may follow. */
typedef struct emu_stream emu_stream;
int emu_stream_arena_bytes(const emu_params* params, int64_t max_grains, int32_t max_views, size_t* arena_bytes);
emu_stream* emu_stream_create(const emu_params* params, int64_t max_grains, int32_t max_views, void* d_arena,
                              size_t arena_bytes);                   /* NULL on failure */
void emu_stream_destroy(emu_stream* s);                              /* s may be NULL; drains the streams first */
int emu_stream_submit(emu_stream* s, const int32_t* h_grains, const int32_t* h_view_off, int64_t n_grains,
                      int32_t n_views);
int emu_stream_collect(emu_stream* s, emu_track* h_tracks, emu_fit* h_fits, int64_t tracks_capacity,
                       int32_t* h_track_off, int32_t* h_members, int64_t members_capacity, int64_t* h_counts);

/* ---- optional per-stage timing (measurement aid for bench.py) -------------
 * An emu_profile is a host-side object that owns CUDA events.  Between emu_profile_begin(p) and
 * emu_profile_end() every kernel the library launches FROM THE CALLING HOST THREAD is bracketed by
 * a pair of events on its launch stream and counted under its stage; nothing else changes (same
 * kernels, same launch configuration).  This is the only state the library keeps, and only while
 * the caller asks for it.  emu_profile_read synchronises on the recorded events and ADDS, per
 * stage, the elapsed milliseconds to ms[EMU_STAGE_COUNT] and the launch counts to
 * launches[EMU_STAGE_COUNT] (either may be NULL), then forgets the recorded events. */
#define EMU_STAGE_BIN_COUNT 0    /* A1 histogram                                                    */
#define EMU_STAGE_BIN_SCAN 1     /* A1 exclusive scan -> cell_start                                 */
#define EMU_STAGE_BIN_SCATTER 2  /* A1 scatter into cell order                                      */
#define EMU_STAGE_BIN_PLACE 3    /* A1 canonical order inside a cell                                */
#define EMU_STAGE_PREP 4         /* bounding boxes, resets, bookkeeping kernels                     */
#define EMU_STAGE_VOTE 5         /* A2 + A3 + A4: seeds, tube count, threshold (the hot loop)       */
#define EMU_STAGE_ASSOC 6        /* A5: exclusive association (priority max, tie settlement)        */
#define EMU_STAGE_SELECT 7       /* A5: wins per candidate, threshold again                         */
#define EMU_STAGE_EMIT 8         /* A7: ordered track list and member lists                         */
#define EMU_STAGE_FIT 9          /* A6                                                              */
#define EMU_STAGE_SEEDS 10       /* A2: seed pairs (count, offsets, fill)                           */
#define EMU_STAGE_CANDS 11       /* A4: threshold -> candidate list                                 */
#define EMU_STAGE_RECOG 12       /* A0: grain recognition (emu_recognize_grains)                    */
#define EMU_STAGE_GENERIC 13     /* global-memory fallback of A2..A4 for chunks the bricks cannot hold
                                    (launched for every chunk; returns at once when the bricks did the work) */
#define EMU_STAGE_COUNT 16
typedef struct emu_profile emu_profile;
emu_profile* emu_profile_create(void);              /* NULL on failure                              */
void emu_profile_destroy(emu_profile* p);           /* p may be NULL                                */
int emu_profile_begin(emu_profile* p);              /* EMU_ERR_INVALID if p is NULL or one is active */
int emu_profile_end(void);
int emu_profile_read(emu_profile* p, double* ms, int64_t* launches);

#ifdef __cplusplus
}
#endif
#endif /* EMU_H_ */
