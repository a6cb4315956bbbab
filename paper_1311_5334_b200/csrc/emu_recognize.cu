// emu_recognize.cu - A0, upstream of the hot path: 3D grain recognition on a stack of
// filtered frames ("Each pixel with a pulse height higher than a given threshold is compared to the
// 3 x 3 x 3 neighboring pixels; the pixel with the highest pulse height among these will be defining the grain.
// The spatial coordinates of the grains are then computed with a center-of-mass method using the pulse height of
// each pixel").  Readings R1-R5 of DESIGN.md section 3b.  Product code: shares nothing with oracle/.
//
// HBM-bound by design: the stack is read once (1 byte per voxel), the other neighbours only for the few voxels that
// pass the in-row test.
//   k_recog        one warp per row (z, y): detection; every grain to a staging record with its row and its rank in the row
//   k_row_scan     exclusive scan over the rows of every view (one block per view) + k_view_offsets over the views
//   k_recog_place  staging record -> row_off[row] + rank: raster order of the defining voxel (R5), view after view
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

// ONE pass over the stack.  One warp per row at a time (rows dealt round-robin, so that neighbouring rows are in
// flight together and their lines are hot in the caches).  A voxel can only define a grain if it is above the threshold,
// higher than its left and at least as high as its right neighbour IN THE ROW (R2's raster tie rule along x); that test
// runs on the 16 bytes a lane has just loaded, four voxels per byte-SIMD compare, and leaves about a third of the voxels
// above the threshold.  The survivors are queued (x, y, z, view) in a ring of the warp that is carried ACROSS rows, and
// whenever 32 wait every lane examines ONE of them - its other 24 neighbours, the tie rule, the centre of mass - so the
// expensive part always runs with full warps.  A grain goes to a staging record with its row and its rank inside the
// row (the ring is in raster order, so ranks are running counts); k_recog_place then puts it at row_off[row] + rank,
// which is the raster order R5 asks for.  (The first version ran the whole detection twice, count and fill, and
// examined the 17 voxels a row holds with half-empty warps: 0.43 ms per 4 views.)
constexpr int kRing = 512;                                      // entries of 8 bytes: >= 31 waiting + 256 new per step (at most
                                                                // every other voxel of a row passes the in-row test)

#ifndef EMU_RECOG_MINB
#define EMU_RECOG_MINB 4
#endif

struct RecogTmp { int4 g; int row, rank, pad0, pad1; };         // 32 B staging record

__global__ void __launch_bounds__(kRecogThreads, EMU_RECOG_MINB)
k_recog(Recog R, const unsigned char* __restrict__ vox, int n_views, int* __restrict__ row_cnt,
        RecogTmp* __restrict__ tmp, long long capacity, unsigned long long* __restrict__ cursor) {
  __shared__ unsigned long long ring_s[kRecogThreads / 32][kRing];
  const int lane = threadIdx.x & 31;
  unsigned long long* ring = ring_s[threadIdx.x >> 5];
  const unsigned thr4 = (unsigned)R.thr * 0x01010101u;
  const long long rows_per_view = (long long)R.nz * R.ny, n_rows = rows_per_view * n_views;
  const long long warp0 = (long long)blockIdx.x * (kRecogThreads / 32) + (threadIdx.x >> 5);
  const long long n_warps = (long long)gridDim.x * (kRecogThreads / 32);
  int head = 0, qn = 0;                                         // the ring: first waiting entry, number waiting
  int carry_row = -1, carry_cnt = 0;                            // the row of the last entry examined, its grains so far

  // examine the first m (<= 32) waiting voxels, one per lane; they are in raster order, and so are the ranks
  auto flush = [&](int m) {
    __syncwarp();
    int4 g = make_int4(0, 0, 0, 0);
    bool ok = false;
    int row = -2 - lane;                                        // (idle lanes: rows nobody else has)
    if (lane < m) {
      const unsigned long long en = ring[(head + lane) & (kRing - 1)];
      const int x = (int)(en & 0xffffu), y = (int)((en >> 16) & 0xffffu), z = (int)((en >> 32) & 0xffffu), view = (int)(en >> 48);
      const unsigned char* v = vox + (size_t)view * rows_per_view * R.nx;
      row = (int)((long long)view * rows_per_view + (long long)z * R.ny + y);
      ok = grain_of(v, R, x, y, z, (int)__ldg(v + ((size_t)z * R.ny + y) * R.nx + x), g);
    }
    const unsigned mk = __ballot_sync(EMU_FULL, ok);
    const unsigned same = __match_any_sync(EMU_FULL, row);      // the lanes of my row
    const unsigned lt = (1u << lane) - 1u;
    const int before = __popc(mk & same & lt) + (row == carry_row ? carry_cnt : 0);
    if (mk) {
      unsigned long long base = 0;
      if (lane == 0) base = atomicAdd(cursor, (unsigned long long)__popc(mk));
      base = __shfl_sync(EMU_FULL, base, 0);
      if (ok) {
        const long long at = (long long)base + __popc(mk & lt);
        if (at < capacity) { RecogTmp t; t.g = g; t.row = row; t.rank = before; t.pad0 = 0; t.pad1 = 0; tmp[at] = t; }
      }
      // the first lane of every row adds the row's grains of this flush to its count
      if (lane < m && (same & lt) == 0u && (mk & same)) atomicAdd(row_cnt + row, __popc(mk & same));
    }
    const int last_row = __shfl_sync(EMU_FULL, row, m - 1);
    const unsigned last_same = __shfl_sync(EMU_FULL, same, m - 1);
    carry_cnt = (last_row == carry_row ? carry_cnt : 0) + __popc(mk & last_same);
    carry_row = last_row;
    head = (head + m) & (kRing - 1); qn -= m;
  };

  for (long long row = warp0; row < n_rows; row += n_warps) {
    // (n_rows < 2^31 is checked by the C ABI: 32-bit divisions)
    const unsigned urow = (unsigned)row, rpv = (unsigned)rows_per_view;
    const int view = (int)(urow / rpv);
    const unsigned zy = urow - (unsigned)view * rpv;
    const int z = (int)(zy / (unsigned)R.ny), y = (int)(zy - (unsigned)z * (unsigned)R.ny);
    const unsigned char* line = vox + (size_t)view * rows_per_view * R.nx + ((size_t)z * R.ny + y) * R.nx;
    const unsigned long long tag = ((unsigned long long)(unsigned)y << 16) | ((unsigned long long)(unsigned)z << 32) | ((unsigned long long)(unsigned)view << 48);

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
    unsigned prev_last = 0u;                                    // the voxel before this step's first (0 outside the stack)
    for (int x0 = 0; x0 < R.nx; x0 += 512) {
      const int x = x0 + 16 * lane;
      const uint4 cur = nxt;
      nxt = (x0 + 512 < R.nx) ? load16(x + 512) : make_uint4(0u, 0u, 0u, 0u);
      const unsigned q[4] = {cur.x, cur.y, cur.z, cur.w};
      // the voxel before my 16 and the one after them
      unsigned left_in = __shfl_up_sync(EMU_FULL, cur.w >> 24, 1);
      if (lane == 0) left_in = prev_last;
      unsigned right_in = __shfl_down_sync(EMU_FULL, cur.x & 0xffu, 1);
      const unsigned next_first = __shfl_sync(EMU_FULL, nxt.x & 0xffu, 0);
      if (lane == 31) right_in = next_first;
      prev_last = __shfl_sync(EMU_FULL, cur.w >> 24, 31);
      // per byte: above the threshold, higher than the left neighbour, at least as high as the right one
      // (one bit per voxel of my 16: the 0x01 bytes of a word are gathered into four bits by a multiply)
      unsigned m16 = 0u;
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        const unsigned lf = __funnelshift_l(w ? q[w - 1] : (left_in << 24), q[w], 8);
        const unsigned rt = __funnelshift_r(q[w], w < 3 ? q[w + 1] : right_in, 8);
        const unsigned mk = __vsetgtu4(q[w], thr4) & __vsetgtu4(q[w], lf) & __vsetgeu4(q[w], rt);   // 0x01 per byte that passes
        m16 |= ((mk * 0x01020408u) >> 24) << (4 * w);
      }
      const int cnt = __popc(m16);
      // x order: lanes in order, voxels of a lane in order.  A lane rarely holds more than one or two survivors, so the
      // exclusive prefix over the lanes is a sum of ballots ("at least k survivors") rather than a shuffle scan
      unsigned any = __ballot_sync(EMU_FULL, cnt > 0);
      if (!any) continue;
      const unsigned lt = (1u << lane) - 1u;
      int excl = 0, total = 0;
      for (int k = 1; any; ++k) {
        excl += __popc(any & lt); total += __popc(any);
        any = __ballot_sync(EMU_FULL, cnt > k);
      }
      int at = head + qn + excl;
      for (; m16; m16 &= m16 - 1u) {                            // the set bits in ascending order = ascending x
        ring[at & (kRing - 1)] = tag | (unsigned long long)(unsigned)(x + __ffs((int)m16) - 1);
        ++at;
      }
      qn += total;
      while (qn >= 32) flush(32);
    }
  }
  while (qn > 0) flush(min(qn, 32));
}

// staging record -> its place in raster order
__global__ void __launch_bounds__(256)
k_recog_place(const RecogTmp* __restrict__ tmp, const unsigned long long* __restrict__ cursor, const int* __restrict__ row_off,
              int4* __restrict__ grains, long long capacity, unsigned long long* __restrict__ status) {
  const long long n = (long long)min(*cursor, (unsigned long long)capacity);
  if (*cursor > (unsigned long long)capacity && blockIdx.x == 0 && threadIdx.x == 0 && status)
    atomicOr(status, (unsigned long long)EMU_ST_GRAIN_OVERFLOW);
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const RecogTmp t = tmp[i];
    const long long at = (long long)row_off[t.row] + t.rank;
    if (at < capacity) grains[at] = t.g;
  }
}

// exclusive scan over the rows of every view, in kScanParts parts per view so that a few views still fill the GPU
// (one block per view took 39 us for four views).  Block (p, v): a thread sums a short run of consecutive rows of
// part p, the block scans the 1 024 sums once, and the thread walks its run again -> offsets inside the part;
// part_tot[v * kScanParts + p] = grains of the part.
constexpr int kScanParts = 16;

__global__ void __launch_bounds__(1024)
k_row_scan(int rows_per_view, int* __restrict__ row_cnt, int* __restrict__ part_tot) {
  __shared__ int warp_sum[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int p = blockIdx.x, v = blockIdx.y;
  const int seg = (rows_per_view + kScanParts - 1) / kScanParts;
  const int s0 = min(rows_per_view, p * seg), s1 = min(rows_per_view, s0 + seg);
  const int per = (seg + (int)blockDim.x - 1) / (int)blockDim.x;
  int* a = row_cnt + (size_t)v * rows_per_view;
  const int r0 = min(s1, s0 + (int)threadIdx.x * per), r1 = min(s1, r0 + per);
  int mine = 0;
  for (int i = r0; i < r1; ++i) mine += a[i];
  int incl = mine;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(EMU_FULL, incl, o); if (lane >= o) incl += t; }
  if (lane == 31) warp_sum[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    const int w = warp_sum[lane]; int wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(EMU_FULL, wi, o); if (lane >= o) wi += t; }
    warp_sum[lane] = wi - w;
    if (lane == 31) part_tot[v * kScanParts + p] = wi;
  }
  __syncthreads();
  int run = warp_sum[wid] + incl - mine;
  for (int i = r0; i < r1; ++i) { const int x = a[i]; a[i] = run; run += x; }
}

// view_off[0..n_views] and the position of every part in the output, from the totals of the parts (one thread: the
// number of views is small), and the total
__global__ void k_view_offsets(int n_views, const int* __restrict__ part_tot, int* __restrict__ part_off,
                               int* __restrict__ view_off, long long* __restrict__ count) {
  long long run = 0;
  for (int v = 0; v < n_views; ++v) {
    view_off[v] = (int)(run > 0x7fffffffll ? 0x7fffffffll : run);
    for (int p = 0; p < kScanParts; ++p) {
      part_off[v * kScanParts + p] = (int)(run > 0x7fffffffll ? 0x7fffffffll : run);
      run += part_tot[v * kScanParts + p];
    }
  }
  view_off[n_views] = (int)(run > 0x7fffffffll ? 0x7fffffffll : run);
  *count = run;
}

// offsets inside the part -> positions in the output
__global__ void __launch_bounds__(256)
k_row_rebase(int rows_per_view, int n_views, int* __restrict__ row_off, const int* __restrict__ part_off) {
  const long long n = (long long)rows_per_view * n_views;
  const int seg = (rows_per_view + kScanParts - 1) / kScanParts;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int v = (int)(i / rows_per_view), r = (int)(i - (long long)v * rows_per_view);
    row_off[i] += part_off[v * kScanParts + r / seg];
  }
}

}  // namespace

size_t emu_recognize_ws_bytes(int32_t n_views, int32_t ny, int32_t nz, int64_t capacity) {
  return emu_align256((size_t)n_views * ny * nz * sizeof(int)) + emu_align256(2 * (size_t)(n_views + 1) * kScanParts * sizeof(int)) + 256 +
         emu_align256((size_t)(capacity > 0 ? capacity : 1) * sizeof(RecogTmp)) + 512;
}

int emu_recognize_launch(const uint8_t* d_vox, int32_t n_views, int32_t nx, int32_t ny, int32_t nz, int32_t thr,
                         const int32_t* pitch_q, int32_t* d_grains, int64_t capacity, int32_t* d_view_off,
                         int64_t* d_count, int64_t* d_status, void* d_ws, size_t ws_bytes, cudaStream_t st) {
  if (ws_bytes < emu_recognize_ws_bytes(n_views, ny, nz, capacity)) return EMU_ERR_CAPACITY;
  if (n_views > 65535 || ny > 65535 || nz > 65535) return EMU_ERR_INVALID;      // the ring packs x, y, z, view in 16 bits each
  Recog R; R.nx = nx; R.ny = ny; R.nz = nz; R.thr = thr;
  for (int a = 0; a < 3; ++a) R.pitch[a] = pitch_q[a];
  char* ws = (char*)emu_align_ptr(d_ws);
  int* row = (int*)ws;
  int* part_tot = (int*)(ws + emu_align256((size_t)n_views * ny * nz * sizeof(int)));
  int* part_off = part_tot + (size_t)(n_views + 1) * kScanParts;
  unsigned long long* cursor = (unsigned long long*)((char*)part_tot + emu_align256(2 * (size_t)(n_views + 1) * kScanParts * sizeof(int)));
  RecogTmp* tmp = (RecogTmp*)((char*)cursor + 256);
  const int rows_per_view = ny * nz;
  const long long n_rows = (long long)rows_per_view * n_views;
  const int blocks = (int)emu_max64(1, emu_min64((n_rows + 7) / 8, emu_sm_count() * 32));
  if (cudaMemsetAsync(row, 0, (size_t)n_rows * sizeof(int), st) != cudaSuccess) return EMU_ERR_CUDA;
  if (cudaMemsetAsync(cursor, 0, 256, st) != cudaSuccess) return EMU_ERR_CUDA;
  EMU_LAUNCH(EMU_STAGE_RECOG, st, k_recog<<<blocks, kRecogThreads, 0, st>>>(R, d_vox, n_views, row, tmp, capacity, cursor));
  if (n_views > 0) EMU_LAUNCH(EMU_STAGE_RECOG, st, k_row_scan<<<dim3(kScanParts, n_views), 1024, 0, st>>>(rows_per_view, row, part_tot));
  EMU_LAUNCH(EMU_STAGE_RECOG, st, k_view_offsets<<<1, 1, 0, st>>>(n_views, part_tot, part_off, d_view_off, (long long*)d_count));
  EMU_LAUNCH(EMU_STAGE_RECOG, st, k_row_rebase<<<(int)emu_max64(1, emu_min64((n_rows + 255) / 256, emu_sm_count() * 8)), 256, 0, st>>>(rows_per_view, n_views, row, part_off));
  EMU_LAUNCH(EMU_STAGE_RECOG, st, k_recog_place<<<emu_sm_count() * 4, 256, 0, st>>>(tmp, cursor, row, (int4*)d_grains, capacity,
                                                                                   (unsigned long long*)d_status));
  return cudaGetLastError() == cudaSuccess ? EMU_OK : EMU_ERR_CUDA;
}
