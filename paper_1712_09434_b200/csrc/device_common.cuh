// Device-side context, grid (spatial index) helpers and the ordered block scan
// shared by the stage kernels of the TPC sector tracker (include/tpc_tracker.h).
//
// Arithmetic rules (docs/ARITH_SPEC.md section 0): this translation unit is
// compiled with -fmad=false -prec-div=true -prec-sqrt=true -ftz=false, so every
// `a*b + c` below is a rounded multiply followed by a rounded add, and `/`,
// sqrtf are IEEE correctly rounded.  No libdevice transcendental is used.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tpc_tracker.h"

namespace tpc {

constexpr int kMaxRows = 1024;        // include/tpc_tracker.h: n_rows <= 1024
#ifndef TPC_BINS_PER_CLUSTER
#define TPC_BINS_PER_CLUSTER 2
#endif
constexpr uint32_t kBinsPerCluster = TPC_BINS_PER_CLUSTER;  // grid density: bins per cluster of a row (the clusters bunch at small |z|)
constexpr uint32_t kBinPad = 96;      // bins of row-block tr start at kBinsPerCluster*row_off[tr] + tr*kBinPad
// entries of one tracklet's row map in Ctx::trk_hits: n_rows rounded up to whole 32-byte sectors
__host__ __device__ inline size_t map_stride(int n_rows) { return (size_t)((n_rows + 7) & ~7); }
constexpr uint32_t kMaxBinsPerRow = 4096;  // shared-memory histogram of the grid build
constexpr float kGridMargin = 0.01f;  // SPEC 2: windows are widened by this before binning
constexpr uint32_t kOwnedBit = 0x80000000u;  // row map entry: the tracklet keeps this hit (set by k_resolve; idx < 2^31)
#ifndef TPC_SEED_THREADS
#define TPC_SEED_THREADS 256
#endif
#ifndef TPC_SEED_ITEMS
#define TPC_SEED_ITEMS 8
#endif
constexpr uint32_t kSeedTileIdx = TPC_SEED_ITEMS * TPC_SEED_THREADS;  // idx per tile of the start-hit finder; Ctx::tile_tr notes the row of every tile start
constexpr float kCoordClamp = 1.0e5f; // grid extents only: coordinates beyond +-1 km (or non-finite) count as this

enum CounterId {
  CN_CLUSTERS = 0, CN_BINS, CN_START_HITS, CN_TRACKLETS_BUILT, CN_TRACKLETS_KEPT, CN_CHAIN_HITS, CN_SEARCHES,
  CN_CANDIDATES, CN_TRACKLET_HITS, CN_ROW_STEPS, CN_NF_PAIRS, CN_RESERVED, CN_SEARCHES_UP, CN_CANDIDATES_UP,
  CN_REFIT_STEPS, CN_RESERVED2, CN_COUNT
};
static_assert(CN_COUNT == TPC_N_COUNTERS, "counter list and header disagree");

// Grid of one (task,row): bin = iz*ny + iy, iy = clamp((y - y0)*inv), iz likewise.  The grid spans the
// bounding box of the row's clusters, not the geometric extent of the row: the clusters of a central event
// fill a third of the drift length in the inner rows, and a grid over the whole row would put three of
// them in every occupied bin.  Coordinates outside the box clamp to the edge bins (monotone), so a window's
// bin range still holds every cluster inside the window.
// 32 bytes = one sector: two vector loads fetch everything a search needs to know about a row.
struct __align__(16) RowInfo {
  float inv;          // 1 / bin size
  float y0, z0;       // origin of the grid
  uint32_t ny_nz;     // ny | nz << 16  (bins across y, along z; both <= kMaxBinsPerRow)
  uint32_t bins_off;  // first entry of this row in Ctx::bins
  uint32_t row_lo;    // idx of the first cluster of the row (= row_off[tr])
  uint32_t pad0, pad1;
};
__device__ __forceinline__ int info_ny(const RowInfo& g) { return (int)(g.ny_nz & 0xFFFFu); }
__device__ __forceinline__ int info_nz(const RowInfo& g) { return (int)(g.ny_nz >> 16); }
__device__ __forceinline__ RowInfo load_row_info(const RowInfo* p) {
  const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
  const uint2 w = __ldg(reinterpret_cast<const uint2*>(p) + 2);
  RowInfo g;
  g.inv = __uint_as_float(v.x); g.y0 = __uint_as_float(v.y); g.z0 = __uint_as_float(v.z); g.ny_nz = v.w;
  g.bins_off = w.x; g.row_lo = w.y; g.pad0 = 0u; g.pad1 = 0u;
  return g;
}

// Seed record of a tracklet, 3 x 16 bytes, so that a5 starts a tracklet with ONE round of loads:
//   [0] h0 (idx of the start hit), tr0 (task*n_rows + row of h0), h1 = clean_up[h0], h2 = clean_up[h1] (or -1)
//   [1] y0, z0, y1, z1 (the (y,z) of h0 and h1 as float bits)
//   [2] y2, z2 (the (y,z) of h2 as float bits), gid(h0), h3 = clean_up[h2] (or -1)
constexpr int kSeedU4 = 3;
constexpr int kRecFloat4 = 8;  // tracklet record: 7 float4, layout in stage_tracklet.cuh

// Everything a kernel needs, passed by value (about 300 bytes of kernel parameters).
struct Ctx {
  // geometry and tables (SPEC 1), device pointers [n_rows]
  int32_t n_sectors, n_rows;
  const float *X, *ymax, *dx_up, *dx_dn, *ratio_up, *ratio_dn;
  float z_max;
  float a, sy2, sz2, wy, wz, smax2;  // T6..T8
  tpc_params prm;
  // input (device)
  const float *y, *z;
  const uint32_t* row_off;  // [n_tr + 1]
  uint32_t n, n_tasks, n_tr;
  // workspace (device); "idx" = position of a cluster in the bin-sorted order, the internal identity
  float2* yz;              // [n]  (y,z) in bin-sorted order: rows keep their [row_off[tr], row_off[tr+1]) range
  uint32_t* gid;           // [n]  idx -> gid (index in the input arrays)
  uint32_t* bins;          // [kBinsPerCluster*n + n_tr*kBinPad + 1]  first idx of every bin (+ one end entry per row)
  RowInfo* rowinfo;        // [n_tr]
  uint32_t* tile_tr;       // [seed_tiles] task*n_rows + row that holds idx = tile * kSeedTile (written by a1 for a4)
  int32_t *link_up, *link_dn;  // [n] raw links as idx (SPEC 3), -1 none
  int32_t* clean_up;       // [n] cleaned up-link (C1)
  uint4* trk_seed;         // [max_tracklets][kSeedU4] seed record written by a4 (layout: kSeedU4 above)
  uint32_t* trk_hits;      // [max_tracklets][map_stride(n_rows)] row map of the tracklet: idx of its hit in that row or kNoHit;
                           // valid for the rows first_row..last_row of the tracklet record
  float4* trk_rec;         // [max_tracklets][kRecFloat4] tracklet record
  uint4* trk_meta;         // [max_tracklets] nHits, firstRow | lastRow << 16, gid of the start hit, 0: what K7 needs
  uint32_t* out_trk;       // [max_tracklets] tracklet of output track `slot` (written by a7 for the merger)
  uint32_t* out_rows;      // [max_tracklets] row of the first kept hit | row of the last kept hit << 16, per output track
  uint32_t* trk_kept;      // [max_tracklets] hits the tracklet keeps (L1), counted by k_resolve; cleared per call
  uint32_t* trk_task_off;  // [n_tasks + 1] first tracklet of every task (tracklets are in task order)
  uint32_t* trk_perm;      // [max_tracklets] queue order of a5: ticket k stands for tracklet trk_perm[k] (k_order_*, stage_tracklet.cuh)
  uint32_t* trk_key;       // [max_tracklets] task * n_rows + row where the next a5 kernel takes the tracklet up (order_note)
  uint32_t* order_cnt;     // [4 kernels][2][order_keys()] tracklets per diagonal of that order, then the slots handed out; cleared per call
  unsigned long long* scan_seed;  // look-back state of the start-hit compaction, [seed_tiles]
  unsigned long long* scan_out;   // look-back state of the output compaction, [out_tiles]
  uint32_t* tickets;       // [8] 0 seed tiles, 1 output tiles, 2..5 queue heads of the four tracklet kernels
  uint32_t* n_tracklets;   // [1] tracklets built (clamped to max_tracklets)
  uint32_t max_tracklets;
  unsigned long long* counters;  // [CN_COUNT] or nullptr
  // outputs (device)
  tpc_tracks out;
};

// ---- queue order of the tracklet constructor (a5); the kernels and the reasons are in stage_tracklet.cuh ----
// Diagonal of a tracklet in front of kernel KIND (0 chain fit, 1 up pass, 2 refit, 3 rest of the down pass):
//     d = (rows between the tracklet's next row and the row where that pass begins) + stagger * task
// The lanes consume one diagonal per row step - every tracklet of a task then starts when the task's wavefront
// passes its row - if a diagonal holds as many tracklets as the lanes end per step:
//     (tracklets per task) / stagger = lanes / life      =>      stagger = (tracklets per task) * life / lanes
// with `life` the row steps a lane spends on a tracklet in that kernel.  The tracklets per task are known on
// the device only (k_order_* read the count); life is a property of the detector (how long tracks are in rows),
// not of the occupancy: the values below are the ones that were fastest on central Pb-Pb-like events of the
// 159-row geometry (a sweep; they are 1.0 - 1.4 times the mean steps per tracklet the device counters give:
// 26, 53, 73 and 37).  Only speed depends on them.
#ifndef TPC_LIFE_CHAIN
#define TPC_LIFE_CHAIN 37.8f
#endif
#ifndef TPC_LIFE_UP
#define TPC_LIFE_UP 70.8f
#endif
#ifndef TPC_LIFE_REFIT
#define TPC_LIFE_REFIT 74.6f
#endif
#ifndef TPC_LIFE_FINISH
#define TPC_LIFE_FINISH 51.8f
#endif
__host__ __device__ constexpr float order_life_of(int kind) {
  return kind == 0 ? TPC_LIFE_CHAIN : kind == 1 ? TPC_LIFE_UP : kind == 2 ? TPC_LIFE_REFIT : TPC_LIFE_FINISH;
}
constexpr uint32_t kStaggerMax = 512;  // stagger in 1/256 rows per task, at most 2 rows: bounds the diagonals
__host__ __device__ inline uint32_t order_keys(uint32_t n_rows, uint32_t n_tasks) {
  return n_rows + (uint32_t)(((uint64_t)n_tasks * kStaggerMax) >> 8) + 1u;
}
// stagger (1/256 rows per task) of kernel `kind` run by `lanes` lanes on n_trk tracklets
__device__ __forceinline__ uint32_t order_stagger(const Ctx& c, int kind, uint32_t lanes, uint32_t n_trk) {
  const float per_task = (float)n_trk / (float)(c.n_tasks ? c.n_tasks : 1u);
  const float s = per_task * order_life_of(kind) * 256.0f / (float)(lanes ? lanes : 1u);
  return (uint32_t)fminf(fmaxf(s, 1.0f), (float)kStaggerMax);
}
// trk_key holds task * n_rows + row (< 2^31, like every (task,row) index); the diagonal of that entry
__device__ __forceinline__ uint32_t order_diagonal(const Ctx& c, uint32_t key, uint32_t stagger) {
  const uint32_t n_rows = (uint32_t)c.n_rows, task = key / n_rows, row = key - task * n_rows;
  // The last n_rows / stagger tasks share one offset, so that the diagonals stay as long as they were down to the
  // last one (a diagonal of staggered tasks alone would thin out, the queue would run ahead of the lanes, and the
  // device would wait for the long tracklets of the last task).
  const uint32_t n_last = (n_rows * 256u) / stagger;
  const uint32_t n_stag = c.n_tasks > n_last ? c.n_tasks - n_last : 0u;
  return row + (uint32_t)(((uint64_t)min(task, n_stag) * stagger) >> 8);
}
// Called by the kernel in front of an a5 kernel when it has finished tracklet t: where its next pass begins
// (tr = task * n_rows + row, row counted from the end of the sector where that pass begins).
__device__ __forceinline__ void order_note(const Ctx& c, uint32_t t, uint32_t tr) { c.trk_key[t] = tr; }

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ uint32_t bins_base(const Ctx& c, uint32_t tr, uint32_t row_lo) {
  return kBinsPerCluster * row_lo + tr * kBinPad;
}

// Monotone clamped bin coordinate; the float is clamped before the conversion (SPEC 0).
__device__ __forceinline__ int bin_coord(float v, float v0, float inv, int n) {
  return (int)fminf(fmaxf((v - v0) * inv, 0.0f), (float)(n - 1));
}

// task*n_rows + row of idx h: last tr with row_off[tr] <= h
__device__ __forceinline__ uint32_t find_tr(const Ctx& c, uint32_t h) {
  uint32_t lo = 0u, hi = c.n_tr;  // row_off[lo] <= h < row_off[hi]
  while (hi - lo > 1u) {
    const uint32_t mid = (lo + hi) >> 1;
    if (c.row_off[mid] <= h) lo = mid; else hi = mid;
  }
  return lo;
}

// ---------------------------------------------------------------------------
// Ordered compaction across blocks: single-pass chained scan with decoupled
// look-back.  Tiles are numbered by a ticket taken when the block starts, so a
// tile only ever waits for tiles that are already running or finished.
// One 64-bit word per tile: bits 63..62 = 0 empty / 1 aggregate / 2 inclusive
// prefix, bits 61..0 the value.  Called by the 32 lanes of warp 0.
// ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long* p) {
  return *reinterpret_cast<const volatile unsigned long long*>(p);
}
__device__ __forceinline__ void st_volatile_u64(unsigned long long* p, unsigned long long v) {
  *reinterpret_cast<volatile unsigned long long*>(p) = v;
}

__device__ __forceinline__ unsigned long long lookback_exclusive(unsigned long long* st, uint32_t tile,
                                                                 unsigned long long agg) {
  const unsigned long long kAgg = 1ull << 62, kPre = 2ull << 62, kMask = (1ull << 62) - 1;
  const int lane = threadIdx.x & 31;
  if (tile == 0) {
    if (lane == 0) st_volatile_u64(&st[0], kPre | agg);
    return 0ull;
  }
  if (lane == 0) st_volatile_u64(&st[tile], kAgg | agg);
  unsigned long long excl = 0ull;
  long long j = (long long)tile - 1;
  while (true) {
    const long long idx = j - lane;
    const unsigned long long v = idx >= 0 ? ld_volatile_u64(&st[idx]) : kPre;
    const unsigned flag = (unsigned)(v >> 62);
    const unsigned ready = __ballot_sync(0xffffffffu, flag != 0u);
    const unsigned is_pre = __ballot_sync(0xffffffffu, flag == 2u);
    const int first_pre = is_pre ? (__ffs(is_pre) - 1) : 32;
    const unsigned need = first_pre >= 31 ? 0xffffffffu : ((2u << first_pre) - 1u);
    if ((ready & need) != need) continue;  // a predecessor has not published yet: read again
    unsigned long long contrib = (lane <= first_pre) ? (v & kMask) : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, o);
    excl += contrib;
    if (first_pre < 32) break;
    j -= 32;
  }
  if (lane == 0) st_volatile_u64(&st[tile], kPre | (excl + agg));
  return excl;
}

// Exclusive scan of one uint32 per thread over the block (blockDim.x <= 1024, multiple of 32).
// Returns the exclusive prefix; *total receives the block sum.  s_warp: shared [33].
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* s_warp, uint32_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
  uint32_t incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = lane < n_warps ? s_warp[lane] : 0u;
    uint32_t wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, wi, o);
      if (lane >= o) wi += t;
    }
    if (lane < n_warps) s_warp[lane] = wi - w;
    if (lane == 31) s_warp[32] = wi;
  }
  __syncthreads();
  const uint32_t r = s_warp[warp] + incl - v;
  *total = s_warp[32];
  __syncthreads();  // s_warp may be reused by the caller
  return r;
}

}  // namespace tpc
