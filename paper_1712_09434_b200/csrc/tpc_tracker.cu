// Host side of the C ABI in include/tpc_tracker.h: tables (docs/ARITH_SPEC.md
// section 1), workspace carving and the launch sequence a1..a7.  No host
// synchronisation and no allocation on the tpc_track_batch path.
//
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -fmad=false
//        -prec-div=true -prec-sqrt=true -ftz=false --shared -Xcompiler -fPIC
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/tpc_tracker.h"
#include "device_common.cuh"
#include "stage_its.cuh"
#include "stage_merge.cuh"
#include "stage_neighbours.cuh"
#include "stage_output.cuh"
#include "stage_slice.cuh"
#include "stage_tracklet.cuh"
#include "stage_transform.cuh"
#include "stages_ca.cuh"

using namespace tpc;

struct tpc_tracker {
  int32_t n_sectors = 0, n_rows = 0;
  float z_max = 0.f, bz = 0.f;
  tpc_params prm{};
  float a = 0.f, sy2 = 0.f, sz2 = 0.f, wy = 0.f, wz = 0.f, smax2 = 0.f;
  int32_t n_half = 1;        // SPEC 9 tables: sectors per side, cos and sin of the sector pitch
  float merge_ca = 1.f, merge_sa = 0.f;
  float* d_tables = nullptr;               // [6][n_rows]: X, ymax, dx_up, dx_dn, ratio_up, ratio_dn
  unsigned long long* d_counters = nullptr;  // [CN_COUNT]
  bool counters_on = false;
  bool debug_sync = false;  // TPC_DEBUG_SYNC=1: synchronise after every stage and name the stage that failed
  // persistent tracklet kernels (chain, up, refit, finish): [kernel][counters off/on] -> blocks that fit the device at once
  int n_sm = 0;
  int merge_grid = 0;  // persistent refit of the merger: blocks the device holds at once
  size_t trk_smem[4] = {0, 0, 0, 0};
  int trk_grid[4][2] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
  // stage timing: ring of TPC_STAGE_RING calls x (TPC_N_STAGES + 1) events, created on first use
  bool timing_on = false;
  // tpc_track_batch_host: one stream per chunk (+ events, pinned headers), created on first use
  std::vector<cudaStream_t> host_streams;
  std::vector<cudaEvent_t> host_events;
  uint32_t* host_headers = nullptr;
  // tpc_host_submit / tpc_host_collect: two batches in flight
  struct PipeSlot { bool busy = false; tpc_tracks d{}; uint32_t tcap = 0, hcap = 0; uint64_t up = 0; cudaEvent_t in = nullptr, done = nullptr; };
  PipeSlot pipe[2];
  uint32_t* pipe_headers = nullptr;  // pinned, 4 words per slot
  std::vector<cudaEvent_t> ev;
  uint32_t timed_calls = 0;
  std::string err;
};

namespace {

thread_local std::string g_create_error;

int fail(tpc_tracker* t, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  if (t) t->err = buf; else g_create_error = buf;
  return code;
}

constexpr size_t kAlign = 256;
size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

uint32_t resolve_max_tracklets(const tpc_tracker* t, uint32_t n, uint32_t max_tracklets) {
  if (max_tracklets) return max_tracklets;
  const uint32_t m = (uint32_t)(t->prm.min_seed_hits > 0 ? t->prm.min_seed_hits : 1);
  return n / m + 1u;  // chains are vertex disjoint and hold >= min_seed_hits clusters each (S2, S3)
}

// tpc_track_batch_host: tracklet slots of all chunks together.  Every chunk gets min(max_tracklets, what its
// clusters can seed at most), so a chunk never overflows while the whole batch would have fitted.
uint32_t host_total_tracklets(const tpc_tracker* t, uint32_t n, uint32_t max_tracklets, uint32_t chunks) {
  const uint64_t worst = (uint64_t)resolve_max_tracklets(t, n, 0u) + chunks;
  const uint64_t want = max_tracklets ? (uint64_t)max_tracklets * chunks : worst;
  return (uint32_t)(want < worst ? want : worst);
}

// Offsets of every workspace array, in bytes.
struct Carve {
  size_t yz, gid, bins, rowinfo, tile_tr, link_up, link_dn, clean_up, trk_seed, trk_hits, trk_rec, trk_meta, zero_begin,
      scan_seed, scan_out, tickets, n_tracklets, trk_task_off, trk_kept, order_cnt, zero_end, out_trk, out_rows, trk_perm, trk_key, total;
  uint32_t seed_tiles, out_tiles;
};

Carve carve(uint32_t n_rows, uint32_t n, uint32_t n_tasks, uint32_t T) {
  Carve c{};
  const size_t n_tr = (size_t)n_tasks * n_rows;
  const size_t n4 = ((size_t)n + kSeedItems - 1) / kSeedItems * kSeedItems + kSeedItems;  // k_seeds reads whole groups of kSeedItems
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes); return o; };
  c.yz = take(n4 * sizeof(float2));
  c.gid = take(n4 * sizeof(uint32_t));
  c.bins = take(((size_t)kBinsPerCluster * n + n_tr * kBinPad + 16) * sizeof(uint32_t));  // + slack of the 16-byte aligned bulk copies
  c.rowinfo = take((n_tr + 1) * sizeof(RowInfo));
  c.tile_tr = take((((size_t)n + kSeedTile - 1) / kSeedTile + 1) * sizeof(uint32_t));
  c.link_up = take(n4 * sizeof(int32_t));
  c.link_dn = take(n4 * sizeof(int32_t));
  c.clean_up = take(n4 * sizeof(int32_t));
  c.trk_seed = take((size_t)T * kSeedU4 * sizeof(uint4));
  c.trk_hits = take((size_t)T * map_stride((int)n_rows) * sizeof(uint32_t));
  c.trk_rec = take((size_t)T * kRecFloat4 * sizeof(float4));
  c.trk_meta = take((size_t)T * sizeof(uint4));
  c.seed_tiles = (uint32_t)(((size_t)n + kSeedTile - 1) / kSeedTile);
  if (c.seed_tiles == 0) c.seed_tiles = 1;
  c.out_tiles = (uint32_t)(((size_t)T + kOutThreads - 1) / kOutThreads);
  if (c.out_tiles == 0) c.out_tiles = 1;
  c.zero_begin = off;  // everything from here to zero_end is cleared by one memset per call
  c.scan_seed = take((size_t)c.seed_tiles * sizeof(unsigned long long));
  c.scan_out = take((size_t)c.out_tiles * sizeof(unsigned long long));
  c.tickets = take(8 * sizeof(uint32_t));
  c.n_tracklets = take(sizeof(uint32_t));
  c.trk_task_off = take(((size_t)n_tasks + 2) * sizeof(uint32_t));
  c.trk_kept = take((size_t)T * sizeof(uint32_t));
  c.order_cnt = take((size_t)8 * order_keys(n_rows, n_tasks) * sizeof(uint32_t));
  c.zero_end = off;
  c.out_trk = take((size_t)T * sizeof(uint32_t));
  c.out_rows = take((size_t)T * sizeof(uint32_t));
  c.trk_perm = take((size_t)T * sizeof(uint32_t));
  c.trk_key = take((size_t)T * sizeof(uint32_t));
  c.total = off;
  return c;
}

void default_params(tpc_params* p) {  // SPEC 8
  p->sigma_y = 0.1f; p->sigma_z = 0.15f;
  p->nf_hy = 2.0f; p->nf_hz = 1.5f; p->nf_chi2_max = 75.0f;
  p->grid_bin_min = 2.0f; p->grid_bin_max = 20.0f;
  p->max_sinphi = 0.95f;
  p->c0_sinphi = 1.0f; p->c0_dzds = 1.0f; p->c0_qpt = 100.0f;
  p->accept_k2 = 16.0f; p->search_max = 3.0f;
  p->turn_cov_scale = 100.0f;
  p->min_seed_hits = 5; p->max_row_gap = 4; p->min_track_hits = 10;
  p->nf_z_projection = 1;
}

Ctx make_ctx(const tpc_tracker* t, const tpc_clusters* in, const tpc_tracks* out, char* ws, const Carve& cv,
             uint32_t T) {
  Ctx c{};
  c.n_sectors = t->n_sectors; c.n_rows = t->n_rows;
  const size_t nr = (size_t)t->n_rows;
  c.X = t->d_tables; c.ymax = t->d_tables + nr; c.dx_up = t->d_tables + 2 * nr; c.dx_dn = t->d_tables + 3 * nr;
  c.ratio_up = t->d_tables + 4 * nr; c.ratio_dn = t->d_tables + 5 * nr;
  c.z_max = t->z_max;
  c.a = t->a; c.sy2 = t->sy2; c.sz2 = t->sz2; c.wy = t->wy; c.wz = t->wz; c.smax2 = t->smax2;
  c.prm = t->prm;
  c.y = in->y; c.z = in->z; c.row_off = in->row_offsets;
  c.n = in->n_clusters; c.n_tasks = in->n_tasks; c.n_tr = in->n_tasks * (uint32_t)t->n_rows;
  c.yz = (float2*)(ws + cv.yz); c.gid = (uint32_t*)(ws + cv.gid); c.bins = (uint32_t*)(ws + cv.bins);
  c.rowinfo = (RowInfo*)(ws + cv.rowinfo); c.tile_tr = (uint32_t*)(ws + cv.tile_tr);
  c.link_up = (int32_t*)(ws + cv.link_up); c.link_dn = (int32_t*)(ws + cv.link_dn);
  c.clean_up = (int32_t*)(ws + cv.clean_up);
  c.trk_seed = (uint4*)(ws + cv.trk_seed);
  c.trk_hits = (uint32_t*)(ws + cv.trk_hits); c.trk_rec = (float4*)(ws + cv.trk_rec);
  c.trk_meta = (uint4*)(ws + cv.trk_meta); c.trk_task_off = (uint32_t*)(ws + cv.trk_task_off);
  c.trk_kept = (uint32_t*)(ws + cv.trk_kept);
  c.trk_perm = (uint32_t*)(ws + cv.trk_perm); c.trk_key = (uint32_t*)(ws + cv.trk_key); c.order_cnt = (uint32_t*)(ws + cv.order_cnt);
  c.out_trk = (uint32_t*)(ws + cv.out_trk); c.out_rows = (uint32_t*)(ws + cv.out_rows);
  c.scan_seed = (unsigned long long*)(ws + cv.scan_seed); c.scan_out = (unsigned long long*)(ws + cv.scan_out);
  c.tickets = (uint32_t*)(ws + cv.tickets); c.n_tracklets = (uint32_t*)(ws + cv.n_tracklets);
  c.max_tracklets = T;
  c.counters = t->counters_on ? t->d_counters : nullptr;
  c.out = *out;
  return c;
}

}  // namespace

extern "C" {

void tpc_default_params(tpc_params* out) {
  if (out) default_params(out);
}

int tpc_tracker_create(const tpc_geometry* g, float bz_kgauss, const tpc_params* params, tpc_tracker** out) {
  if (!g || !out) return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_tracker_create: geometry and out must not be NULL");
  *out = nullptr;
  if (g->n_sectors < 1 || g->n_rows < 3 || g->n_rows > kMaxRows || !g->row_x)
    return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_tracker_create: need n_sectors >= 1, 3 <= n_rows <= %d, row_x",
                kMaxRows);
  for (int r = 0; r < g->n_rows; ++r)
    if (!(g->row_x[r] > 0.f) || (r > 0 && !(g->row_x[r] > g->row_x[r - 1])))
      return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_tracker_create: row_x must be positive and strictly increasing");
  if (!(g->tan_half_angle > 0.f) || !(g->z_max > 0.f))
    return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_tracker_create: tan_half_angle and z_max must be positive");
  tpc_tracker* t = new (std::nothrow) tpc_tracker();
  if (!t) return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_tracker_create: out of host memory");
  if (params) t->prm = *params; else default_params(&t->prm);
  const tpc_params& p = t->prm;
  if (!(p.sigma_y > 0.f) || !(p.sigma_z > 0.f) || !(p.grid_bin_min > 0.f) || !(p.grid_bin_max >= p.grid_bin_min) ||
      p.min_seed_hits < 2 || p.min_track_hits < 1 || p.max_row_gap < 0) {
    delete t;
    return fail(nullptr, TPC_ERR_ARGUMENT,
                "tpc_tracker_create: need sigma > 0, 0 < grid_bin_min <= grid_bin_max, min_seed_hits >= 2, "
                "min_track_hits >= 1, max_row_gap >= 0");
  }
  t->n_sectors = g->n_sectors; t->n_rows = g->n_rows; t->z_max = g->z_max; t->bz = bz_kgauss;
  {
    const char* dbg = getenv("TPC_DEBUG_SYNC");
    t->debug_sync = dbg && dbg[0] == '1';
  }
  const int n = g->n_rows;
  std::vector<float> tab((size_t)6 * n, 0.f);
  float *X = tab.data(), *ymax = X + n, *dx_up = X + 2 * n, *dx_dn = X + 3 * n, *ratio_up = X + 4 * n,
        *ratio_dn = X + 5 * n;
  for (int r = 0; r < n; ++r) X[r] = g->row_x[r];
  for (int r = 0; r < n; ++r) ymax[r] = X[r] * g->tan_half_angle + 1.0f;                    // T1
  const bool proj = p.nf_z_projection != 0;  // SPEC 11: no projection of z in time-frame mode
  for (int r = 0; r + 1 < n; ++r) { dx_up[r] = X[r + 1] - X[r]; ratio_up[r] = proj ? X[r + 1] / X[r] : 1.0f; }  // T2 T4
  for (int r = 1; r < n; ++r) { dx_dn[r] = X[r] - X[r - 1]; ratio_dn[r] = proj ? X[r - 1] / X[r] : 1.0f; }      // T3 T5
  t->a = -0.000299792458f * bz_kgauss;                                                       // T6
  t->sy2 = p.sigma_y * p.sigma_y; t->sz2 = p.sigma_z * p.sigma_z;                            // T7
  t->wy = 1.0f / t->sy2; t->wz = 1.0f / t->sz2;
  t->smax2 = p.search_max * p.search_max;                                                    // T8
  t->n_half = g->n_sectors >= 2 ? g->n_sectors / 2 : 1;                                      // SPEC 9 tables
  {
    const double alpha = 2.0 * 3.14159265358979323846 / (double)t->n_half;
    t->merge_ca = (float)cos(alpha);
    t->merge_sa = (float)sin(alpha);
  }
  cudaError_t e = cudaMalloc(&t->d_tables, tab.size() * sizeof(float));
  if (e == cudaSuccess) e = cudaMalloc(&t->d_counters, CN_COUNT * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMemcpy(t->d_tables, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemset(t->d_counters, 0, CN_COUNT * sizeof(unsigned long long));
  if (e != cudaSuccess) {
    const int rc = fail(nullptr, TPC_ERR_CUDA, "tpc_tracker_create: CUDA: %s (no CPU fallback exists)",
                        cudaGetErrorString(e));
    if (t->d_tables) cudaFree(t->d_tables);
    if (t->d_counters) cudaFree(t->d_counters);
    delete t;
    cudaGetLastError();
    return rc;
  }
#ifdef TPC_L2_FETCH
  cudaDeviceSetLimit(cudaLimitMaxL2FetchGranularity, TPC_L2_FETCH);
#endif
  // launch shape of the persistent tracklet constructor: as many blocks as the device holds at once
  int dev = 0, n_sm = 0;
  e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute((const void*)k_neighbours<false, kNfList>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)nf_smem_bytes(kNfList));
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute((const void*)k_neighbours<true, kNfList>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)nf_smem_bytes(kNfList));
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute((const void*)k_neighbours<false, kNfListDense>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)nf_smem_bytes(kNfListDense));
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute((const void*)k_neighbours<true, kNfListDense>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)nf_smem_bytes(kNfListDense));
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute((const void*)k_resolve, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(kResolveChunk * sizeof(unsigned long long)));
  t->n_sm = n_sm;
  if (e == cudaSuccess) {
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)k_merge_refit, kMergeThreads,
                                                      (size_t)t->n_rows * sizeof(float));
    t->merge_grid = (per_sm > 0 ? per_sm : 1) * n_sm;
  }
  const int trk_slot16[4] = {kChainSlot16, kRecSlot16, kRecSlot16, kFinishSlot16};
  for (int k = 0; k < 4; ++k) t->trk_smem[k] = trk_smem_bytes(t->n_rows, trk_slot16[k]);
  const void* trk_fn[4][2] = {{(const void*)k_trk_chain<false>, (const void*)k_trk_chain<true>},
                               {(const void*)k_trk_up<false>, (const void*)k_trk_up<true>},
                               {(const void*)k_trk_refit<false>, (const void*)k_trk_refit<true>},
                               {(const void*)k_trk_finish<false>, (const void*)k_trk_finish<true>}};
  for (int k = 0; k < 4; ++k)
    for (int cnt = 0; cnt < 2 && e == cudaSuccess; ++cnt) {
      int per_sm = 0;
      e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, trk_fn[k][cnt], kTrackletThreads, t->trk_smem[k]);
      t->trk_grid[k][cnt] = (per_sm > 0 ? per_sm : 1) * n_sm;
    }
  if (e != cudaSuccess) {
    const int rc = fail(nullptr, TPC_ERR_CUDA, "tpc_tracker_create: CUDA: %s", cudaGetErrorString(e));
    cudaFree(t->d_tables);
    cudaFree(t->d_counters);
    delete t;
    cudaGetLastError();
    return rc;
  }
  *out = t;
  return TPC_OK;
}

void tpc_tracker_destroy(tpc_tracker* t) {
  if (!t) return;
  for (cudaEvent_t e : t->ev) cudaEventDestroy(e);
  for (cudaStream_t x : t->host_streams) cudaStreamDestroy(x);
  for (cudaEvent_t x : t->host_events) cudaEventDestroy(x);
  if (t->host_headers) cudaFreeHost(t->host_headers);
  if (t->pipe_headers) cudaFreeHost(t->pipe_headers);
  for (auto& p : t->pipe) { if (p.in) cudaEventDestroy(p.in); if (p.done) cudaEventDestroy(p.done); }
  if (t->d_tables) cudaFree(t->d_tables);
  if (t->d_counters) cudaFree(t->d_counters);
  delete t;
}

size_t tpc_workspace_bytes(const tpc_tracker* t, uint32_t max_clusters, uint32_t max_tasks, uint32_t max_tracklets) {
  if (!t) return 0;
  const uint32_t T = resolve_max_tracklets(t, max_clusters, max_tracklets);
  return carve((uint32_t)t->n_rows, max_clusters, max_tasks, T).total;
}

int tpc_launches_per_batch(const tpc_tracker*) { return 23; }  // a1, a2, a3, a4, a5 (4 kernels, each behind the 3 of its queue order), K7 (2), a6+a7, a5 (4 kernels), K7 (2), a6+a7

void tpc_tracker_enable_counters(tpc_tracker* t, int on) {
  if (t) t->counters_on = on != 0;
}

void tpc_tracker_enable_stage_timing(tpc_tracker* t, int on) {
  if (!t) return;
  t->timing_on = on != 0;
  t->timed_calls = 0;
}

const char* tpc_stage_name(int stage) {
  static const char* const names[TPC_N_STAGES] = {"grid_build", "neighbour_finder", "cleaner", "start_hits",
                                                  "tracklet_chain_fit", "tracklet_up_pass", "tracklet_refit",
                                                  "tracklet_down_finish", "ownership", "selector_output"};
  return stage >= 0 && stage < TPC_N_STAGES ? names[stage] : nullptr;
}

int tpc_read_stage_ms(tpc_tracker* t, void* cuda_stream, float* out_ms, uint32_t* n_calls) {
  if (!t || !out_ms) return TPC_ERR_ARGUMENT;
  cudaError_t e = cudaStreamSynchronize((cudaStream_t)cuda_stream);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_read_stage_ms: CUDA: %s", cudaGetErrorString(e));
  const uint32_t n = t->timed_calls < TPC_STAGE_RING ? t->timed_calls : TPC_STAGE_RING;
  double sum[TPC_N_STAGES] = {0};
  for (uint32_t k = 0; k < n; ++k) {
    const uint32_t slot = (t->timed_calls - 1 - k) % TPC_STAGE_RING;
    const cudaEvent_t* ev = t->ev.data() + (size_t)slot * (TPC_N_STAGES + 1);
    for (int i = 0; i < TPC_N_STAGES; ++i) {
      float ms = 0.f;
      e = cudaEventElapsedTime(&ms, ev[i], ev[i + 1]);
      if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_read_stage_ms: CUDA: %s", cudaGetErrorString(e));
      sum[i] += ms;
    }
  }
  for (int i = 0; i < TPC_N_STAGES; ++i) out_ms[i] = n ? (float)(sum[i] / n) : 0.f;
  if (n_calls) *n_calls = n;
  return TPC_OK;
}

int tpc_read_counters(tpc_tracker* t, void* cuda_stream, uint64_t* out) {
  if (!t || !out) return TPC_ERR_ARGUMENT;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaMemcpyAsync(out, t->d_counters, CN_COUNT * sizeof(uint64_t), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_read_counters: CUDA: %s", cudaGetErrorString(e));
  return TPC_OK;
}

int tpc_track_batch(tpc_tracker* t, const tpc_clusters* in, tpc_tracks* out, void* workspace, size_t workspace_bytes,
                    uint32_t max_tracklets, void* cuda_stream) {
  if (!t) return TPC_ERR_ARGUMENT;
  if (!in || !out) return fail(t, TPC_ERR_ARGUMENT, "tpc_track_batch: clusters and tracks must not be NULL");
  if (!in->row_offsets || (in->n_clusters && (!in->y || !in->z)))
    return fail(t, TPC_ERR_ARGUMENT, "tpc_track_batch: y, z, row_offsets must not be NULL");
  if (in->n_clusters >= 0x80000000u) return fail(t, TPC_ERR_ARGUMENT, "tpc_track_batch: n_clusters must be < 2^31");
  if ((uint64_t)in->n_tasks * (uint64_t)t->n_rows >= 0x7FFFFFFFull)
    return fail(t, TPC_ERR_ARGUMENT, "tpc_track_batch: n_tasks*n_rows must be < 2^31");
  if (!out->header || !out->track_task || !out->track_hit_begin || !out->track_nhits || !out->track_ndf ||
      !out->track_x || !out->track_par || !out->track_cov || !out->track_chi2 || !out->hit_cluster)
    return fail(t, TPC_ERR_ARGUMENT, "tpc_track_batch: every track_* output and hit_cluster must not be NULL");
  const uint32_t T = resolve_max_tracklets(t, in->n_clusters, max_tracklets);
  const Carve cv = carve((uint32_t)t->n_rows, in->n_clusters, in->n_tasks, T);
  if (!workspace || workspace_bytes < cv.total)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_track_batch: workspace of %zu bytes, need %zu", workspace_bytes, cv.total);
  if (((uintptr_t)workspace & (kAlign - 1)) != 0)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_track_batch: workspace must be %zu-byte aligned", kAlign);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  const Ctx c = make_ctx(t, in, out, ws, cv, T);
  cudaError_t e = cudaMemsetAsync(ws + cv.zero_begin, 0, cv.zero_end - cv.zero_begin, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(out->header, 0, 4 * sizeof(uint32_t), s);
  if (e == cudaSuccess && t->counters_on) e = cudaMemsetAsync(t->d_counters, 0, CN_COUNT * sizeof(uint64_t), s);
  if (e == cudaSuccess && out->dbg_n_start_hits) e = cudaMemsetAsync(out->dbg_n_start_hits, 0, sizeof(uint32_t), s);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_track_batch: CUDA memset: %s", cudaGetErrorString(e));
  const bool cnt = t->counters_on;
  cudaEvent_t* ev = nullptr;  // stage marks of this call (nullptr: timing off)
  if (t->timing_on) {
    if (t->ev.empty()) {
      t->ev.resize((size_t)TPC_STAGE_RING * (TPC_N_STAGES + 1), nullptr);
      for (cudaEvent_t& x : t->ev)
        if (cudaEventCreate(&x) != cudaSuccess) {
          for (cudaEvent_t& y : t->ev) if (y) cudaEventDestroy(y);
          t->ev.clear();
          return fail(t, TPC_ERR_CUDA, "tpc_track_batch: cudaEventCreate failed");
        }
    }
    ev = t->ev.data() + (size_t)(t->timed_calls % TPC_STAGE_RING) * (TPC_N_STAGES + 1);
    ++t->timed_calls;
  }
  int stage = 0, bad_stage = -1;
  cudaError_t bad = cudaSuccess;
  auto mark = [&]() {
    if (ev) cudaEventRecord(ev[stage], s);
    if (t->debug_sync && bad == cudaSuccess && stage > 0) {
      bad = cudaStreamSynchronize(s);
      if (bad != cudaSuccess) bad_stage = stage - 1;
    }
    ++stage;
  };
  mark();
  if (c.n_tr > 0) {
    if (cnt) k_grid_build<true><<<c.n_tr, kGridThreads, 0, s>>>(c);                         // a1
    else k_grid_build<false><<<c.n_tr, kGridThreads, 0, s>>>(c);
  }
  mark();
  if (c.n_tr > 0) {
    // deeper candidate lists where the rows are dense (more than kNfDenseRow clusters per row on average)
    const bool dense = (uint64_t)c.n > (uint64_t)kNfDenseRow * c.n_tr;
    if (dense) {
      if (cnt) k_neighbours<true, kNfListDense><<<c.n_tr, kNfThreads, nf_smem_bytes(kNfListDense), s>>>(c);   // a2
      else k_neighbours<false, kNfListDense><<<c.n_tr, kNfThreads, nf_smem_bytes(kNfListDense), s>>>(c);
    } else {
      if (cnt) k_neighbours<true, kNfList><<<c.n_tr, kNfThreads, nf_smem_bytes(kNfList), s>>>(c);             // a2
      else k_neighbours<false, kNfList><<<c.n_tr, kNfThreads, nf_smem_bytes(kNfList), s>>>(c);
    }
  }
  mark();
  if (c.n > 0) {
    k_clean<<<(c.n + kCleanThreads * kCleanItems - 1) / (kCleanThreads * kCleanItems), kCleanThreads, 0, s>>>(c);  // a3
  }
  mark();
  if (cnt) k_seeds<true><<<cv.seed_tiles, kSeedThreads, 0, s>>>(c);                         // a4
  else k_seeds<false><<<cv.seed_tiles, kSeedThreads, 0, s>>>(c);
  mark();
  // a5: four persistent kernels, each with as many blocks as the device holds at once and its own queue order
  const int og = 4 * t->n_sm;
#define TPC_ORDER(KIND)                                                                                \
  {                                                                                                    \
    const uint32_t lanes = (uint32_t)t->trk_grid[KIND][cnt ? 1 : 0] * (uint32_t)kTrackletThreads;      \
    k_order_count<<<og, kOrderThreads, 0, s>>>(c, KIND, lanes);                                        \
    k_order_scan<<<1, 1024, 0, s>>>(c, KIND);                                                          \
    k_order_fill<<<og, kOrderThreads, 0, s>>>(c, KIND, lanes);                                         \
  }
  TPC_ORDER(0)
  if (cnt) k_trk_chain<true><<<t->trk_grid[0][1], kTrackletThreads, t->trk_smem[0], s>>>(c);
  else k_trk_chain<false><<<t->trk_grid[0][0], kTrackletThreads, t->trk_smem[0], s>>>(c);
  mark();
  TPC_ORDER(1)
  if (cnt) k_trk_up<true><<<t->trk_grid[1][1], kTrackletThreads, t->trk_smem[1], s>>>(c);
  else k_trk_up<false><<<t->trk_grid[1][0], kTrackletThreads, t->trk_smem[1], s>>>(c);
  mark();
  TPC_ORDER(2)
  if (cnt) k_trk_refit<true><<<t->trk_grid[2][1], kTrackletThreads, t->trk_smem[2], s>>>(c);
  else k_trk_refit<false><<<t->trk_grid[2][0], kTrackletThreads, t->trk_smem[2], s>>>(c);
  mark();
  TPC_ORDER(3)
#undef TPC_ORDER
  if (cnt) k_trk_finish<true><<<t->trk_grid[3][1], kTrackletThreads, t->trk_smem[3], s>>>(c);
  else k_trk_finish<false><<<t->trk_grid[3][0], kTrackletThreads, t->trk_smem[3], s>>>(c);
  mark();
  if (out->dbg_tracklet_capacity &&  // the row maps before the ownership kernel removes the hits a tracklet loses
      (out->dbg_tracklet_start || out->dbg_tracklet_nhits || out->dbg_tracklet_map || out->dbg_tracklet_par))
    k_debug_tracklets<<<(out->dbg_tracklet_capacity + 127) / 128, 128, 0, s>>>(c);
  if (c.n > 0) {                                                                            // K7 + L1
    k_task_offsets<<<2 * t->n_sm, 256, 0, s>>>(c);
    k_resolve<<<(c.n + kResolveChunk - 1) / kResolveChunk, kResolveThreads, kResolveChunk * sizeof(unsigned long long), s>>>(c);
  }
  mark();
  k_select_output<<<cv.out_tiles < 16u * (uint32_t)t->n_sm ? cv.out_tiles : 16u * (uint32_t)t->n_sm, kOutThreads, 0, s>>>(c);                          // a6 + a7
  mark();
  if (c.n > 0 && (out->dbg_link_up || out->dbg_link_dn || out->dbg_clean_up || out->dbg_clean_dn ||
                  out->dbg_start_hits))
    k_debug_links<<<(c.n + 255) / 256, 256, 0, s>>>(c);
  if (bad != cudaSuccess)
    return fail(t, TPC_ERR_CUDA, "tpc_track_batch: stage %s: %s", tpc_stage_name(bad_stage), cudaGetErrorString(bad));
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_track_batch: CUDA launch: %s", cudaGetErrorString(e));
  return TPC_OK;
}

// ---- host-buffer variant -------------------------------------------------------
// The batch is cut into up to kHostChunks runs of whole sector tasks (tasks are independent, PAPER.md L138,
// L127) and three streams - copies in, kernels, copies out - are used: the host->device copy of chunk k+1 and the
// device->host copy of chunk k-1 overlap the kernels of chunk k.  Every chunk is one tpc_track_batch call on its slice of the inputs; a small
// kernel rebases its row offsets before, and one shifts its task numbers, hit ranges and cluster indices to
// those of the whole batch after.  Chunks are visited in task order, so the result is the one call's result.
namespace {
constexpr uint32_t kHostChunks = 4;
constexpr uint32_t kHostChunkMinClusters = 1u << 20;  // smaller batches go through as one chunk

__global__ void k_rebase_offsets(uint32_t* ro, uint32_t n, uint32_t base) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) ro[i] -= base;
}
__global__ void k_shift_chunk(uint32_t* track_task, uint32_t* track_hit_begin, uint32_t n_tracks, uint32_t* hit_cluster,
                              uint32_t n_hits, uint32_t task0, uint32_t hit0, uint32_t gid0) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_tracks) { track_task[i] += task0; track_hit_begin[i] += hit0; }
  if (i < n_hits) hit_cluster[i] += gid0;
}

struct HostCarve {
  size_t y, z, row_off, header, track_task, track_hit_begin, track_nhits, track_ndf, track_x, track_par, track_cov,
      track_chi2, hit_cluster, inner, total;
  uint32_t tcap_dev, hcap_dev;
};
HostCarve host_carve(const tpc_tracker* t, uint32_t n, uint32_t n_tasks, uint32_t T, uint32_t tcap, uint32_t hcap) {
  HostCarve h{};
  const uint32_t mh = (uint32_t)(t->prm.min_track_hits > 0 ? t->prm.min_track_hits : 1);
  // device-side capacities: every chunk gets min(caller's capacity, what its clusters can produce at most)
  const uint64_t tc = (uint64_t)n / mh + kHostChunks, hc = (uint64_t)n + kHostChunks;
  h.tcap_dev = (uint32_t)(tc < (uint64_t)tcap * kHostChunks ? tc : (uint64_t)tcap * kHostChunks);
  h.hcap_dev = (uint32_t)(hc < (uint64_t)hcap * kHostChunks ? hc : (uint64_t)hcap * kHostChunks);
  if (h.tcap_dev < tcap) h.tcap_dev = tcap;
  if (h.hcap_dev < hcap) h.hcap_dev = hcap;
  const size_t tcd = h.tcap_dev, hcd = h.hcap_dev;
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes); return o; };
  h.y = take((size_t)n * 4); h.z = take((size_t)n * 4);
  h.row_off = take(((size_t)n_tasks * t->n_rows + kHostChunks) * 4 + kHostChunks * kAlign);
  h.header = take(16 * kHostChunks);
  h.track_task = take(tcd * 4); h.track_hit_begin = take(tcd * 4);
  h.track_nhits = take(tcd * 4); h.track_ndf = take(tcd * 4); h.track_x = take(tcd * 4);
  h.track_par = take(tcd * 20); h.track_cov = take(tcd * 60); h.track_chi2 = take(tcd * 4);
  h.hit_cluster = take(hcd * 4);
  h.inner = off;
  // the chunks' workspaces together: linear in clusters, tasks and tracklets, plus alignment slack per chunk
  h.total = off + carve((uint32_t)t->n_rows, n, n_tasks, T).total + (size_t)kHostChunks * 64 * 1024;
  return h;
}
}  // namespace

namespace { int ensure_host_streams(tpc_tracker* t); }

size_t tpc_host_workspace_bytes(const tpc_tracker* t, uint32_t max_clusters, uint32_t max_tasks, uint32_t max_tracklets,
                                uint32_t track_capacity, uint32_t hit_capacity) {
  if (!t) return 0;
  const uint32_t T = host_total_tracklets(t, max_clusters, max_tracklets, kHostChunks);
  return host_carve(t, max_clusters, max_tasks, T, track_capacity, hit_capacity).total;
}

int tpc_track_batch_host(tpc_tracker* t, const tpc_clusters* in, tpc_tracks* out, void* workspace, size_t workspace_bytes,
                         uint32_t max_tracklets, void* cuda_stream, uint64_t* h2d_bytes, uint64_t* d2h_bytes) {
  if (!t) return TPC_ERR_ARGUMENT;
  if (!in || !out) return fail(t, TPC_ERR_ARGUMENT, "tpc_track_batch_host: clusters and tracks must not be NULL");
  if (!in->row_offsets || (in->n_clusters && (!in->y || !in->z)) || !out->header)
    return fail(t, TPC_ERR_ARGUMENT, "tpc_track_batch_host: y, z, row_offsets, header must not be NULL");
  if (out->dbg_link_up || out->dbg_link_dn || out->dbg_clean_up || out->dbg_clean_dn || out->dbg_start_hits ||
      out->dbg_tracklet_start || out->dbg_tracklet_nhits || out->dbg_tracklet_map || out->dbg_tracklet_par)
    return fail(t, TPC_ERR_ARGUMENT, "tpc_track_batch_host: dbg_* outputs are not supported on host buffers");
  const uint32_t n = in->n_clusters, tcap = out->track_capacity, hcap = out->hit_capacity;
  const uint32_t n_rows = (uint32_t)t->n_rows;
  const uint32_t T_all = host_total_tracklets(t, n, max_tracklets, kHostChunks);
  const HostCarve h = host_carve(t, n, in->n_tasks, T_all, tcap, hcap);
  if (!workspace || workspace_bytes < h.total)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_track_batch_host: workspace of %zu bytes, need %zu", workspace_bytes, h.total);
  if (((uintptr_t)workspace & (kAlign - 1)) != 0)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_track_batch_host: workspace must be %zu-byte aligned", kAlign);
  cudaStream_t s_user = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  const uint32_t* ro = in->row_offsets;
  if (ro[(size_t)in->n_tasks * n_rows] != n)
    return fail(t, TPC_ERR_ARGUMENT, "tpc_track_batch_host: row_offsets must end at n_clusters");
  // chunk boundaries: whole tasks; a small first chunk (the kernels start early) and a middle-sized last one (its
  // copy-back is the tail) measured best on config 3 with the four-kernel tracklet constructor, whose persistent
  // kernels cost about 0.3 ms per extra chunk: 18.1 ms against 18.8 ms with cuts at 12 / 45 / 80 %
  static const double cut[] = {0.0, 0.15, 0.55, 1.0};
  constexpr uint32_t kCuts = sizeof(cut) / sizeof(cut[0]) - 1;
  static_assert(kCuts <= kHostChunks, "streams, events and headers are sized for kHostChunks chunks");
  uint32_t n_chunks = (n >= kHostChunkMinClusters && in->n_tasks >= kCuts) ? kCuts : 1u;
  uint32_t task_b[kHostChunks + 1];
  task_b[0] = 0u;
  for (uint32_t k = 1; k < n_chunks; ++k) {
    const uint64_t want = (uint64_t)((double)n * cut[k]);
    uint32_t lo = task_b[k - 1], hi = in->n_tasks;  // first task whose clusters start at or after `want`
    while (lo < hi) {
      const uint32_t mid = lo + (hi - lo) / 2;
      if (ro[(size_t)mid * n_rows] < want) lo = mid + 1; else hi = mid;
    }
    task_b[k] = lo;
  }
  task_b[n_chunks] = in->n_tasks;
  // streams and events of the chunks, created on first use
  cudaError_t e = cudaSuccess;
  {
    const int rc0 = ensure_host_streams(t);
    if (rc0 != TPC_OK) return rc0;
  }
  const bool timing = t->timing_on, counters = t->counters_on;
  t->timing_on = false; t->counters_on = false;  // per-stage marks and counters describe one tpc_track_batch call
  uint64_t up = 0, down = 0;
  e = cudaEventRecord(t->host_events[kHostChunks], s_user);  // the chunks start after the caller's stream got here
  struct Chunk { uint32_t n, idx0, task0, n_tasks, T, tcap, hcap, t0, h0; tpc_tracks d; } ch[kHostChunks];
  size_t inner_off = h.inner, ro_off = h.row_off;
  uint32_t t_used = 0, h_used = 0;
  const uint32_t mh = (uint32_t)(t->prm.min_track_hits > 0 ? t->prm.min_track_hits : 1);
  int rc = TPC_OK;
  // three streams: copies in, kernels, copies out.  The kernels of the chunks run one after the other - run side by
  // side, two persistent tracklet constructors slow each other down more than the overlap gains (measured:
  // 16.5 ms against 14.6 ms for the two halves of config 3).
  cudaStream_t s_in = t->host_streams[0], s_cmp = t->host_streams[1], s_out = t->host_streams[2];
  if (e == cudaSuccess) e = cudaStreamWaitEvent(s_in, t->host_events[kHostChunks], 0);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(s_cmp, t->host_events[kHostChunks], 0);
  for (uint32_t k = 0; k < n_chunks && e == cudaSuccess && rc == TPC_OK; ++k) {
    Chunk& c = ch[k];
    cudaStream_t s = s_cmp;
    c.task0 = task_b[k]; c.n_tasks = task_b[k + 1] - task_b[k];
    c.idx0 = ro[(size_t)c.task0 * n_rows];
    c.n = ro[(size_t)task_b[k + 1] * n_rows] - c.idx0;
    c.T = resolve_max_tracklets(t, c.n, 0u);
    if (max_tracklets && max_tracklets < c.T) c.T = max_tracklets;
    c.tcap = c.n / mh + 1u < tcap ? c.n / mh + 1u : tcap;
    c.hcap = c.n + 1u < hcap ? c.n + 1u : hcap;
    c.t0 = t_used; c.h0 = h_used;
    t_used += c.tcap; h_used += c.hcap;
    const size_t n_off = (size_t)c.n_tasks * n_rows + 1;
    uint32_t* d_ro = (uint32_t*)(ws + ro_off);
    ro_off = align_up(ro_off + n_off * 4);
    auto h2d = [&](void* dst, const void* src, size_t bytes) {
      if (e == cudaSuccess && bytes) { e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, s_in); up += bytes; }
    };
    h2d(ws + h.y + (size_t)c.idx0 * 4, in->y + c.idx0, (size_t)c.n * 4);
    h2d(ws + h.z + (size_t)c.idx0 * 4, in->z + c.idx0, (size_t)c.n * 4);
    h2d(d_ro, ro + (size_t)c.task0 * n_rows, n_off * 4);
    if (e == cudaSuccess) e = cudaEventRecord(t->host_events[kHostChunks + 1 + k], s_in);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_cmp, t->host_events[kHostChunks + 1 + k], 0);
    if (e != cudaSuccess) break;
    if (c.idx0) k_rebase_offsets<<<(unsigned)((n_off + 255) / 256), 256, 0, s>>>(d_ro, (uint32_t)n_off, c.idx0);
    tpc_clusters din{};
    din.y = (const float*)(ws + h.y) + c.idx0; din.z = (const float*)(ws + h.z) + c.idx0;  // x, charge: not read (R18, R23)
    din.row_offsets = d_ro; din.n_clusters = c.n; din.n_tasks = c.n_tasks;
    tpc_tracks& d = c.d;
    d = tpc_tracks{};
    d.track_capacity = c.tcap; d.hit_capacity = c.hcap;
    d.header = (uint32_t*)(ws + h.header) + 4 * k;
    d.track_task = (uint32_t*)(ws + h.track_task) + c.t0; d.track_hit_begin = (uint32_t*)(ws + h.track_hit_begin) + c.t0;
    d.track_nhits = (uint32_t*)(ws + h.track_nhits) + c.t0; d.track_ndf = (int32_t*)(ws + h.track_ndf) + c.t0;
    d.track_x = (float*)(ws + h.track_x) + c.t0; d.track_chi2 = (float*)(ws + h.track_chi2) + c.t0;
    // SoA columns of a chunk are c.tcap apart, packed one chunk after the other
    d.track_par = (float*)(ws + h.track_par) + (size_t)5 * c.t0; d.track_cov = (float*)(ws + h.track_cov) + (size_t)15 * c.t0;
    d.hit_cluster = (uint32_t*)(ws + h.hit_cluster) + c.h0;
    const size_t need = carve(n_rows, c.n, c.n_tasks, c.T).total;
    if (inner_off + need > workspace_bytes) { rc = fail(t, TPC_ERR_WORKSPACE, "tpc_track_batch_host: workspace too small for chunk %u", k); break; }
    rc = tpc_track_batch(t, &din, &d, ws + inner_off, need, c.T, s);
    inner_off = align_up(inner_off + need);
    if (rc != TPC_OK) break;
    e = cudaMemcpyAsync(t->host_headers + 4 * k, d.header, 16, cudaMemcpyDeviceToHost, s);
    down += 16;
    if (e == cudaSuccess) e = cudaEventRecord(t->host_events[k], s);
  }
  // collect the chunks in task order
  uint32_t tracks_off = 0, hits_off = 0, status = 0, tracklets = 0;
  uint64_t tracks_all = 0, hits_all = 0;
  for (uint32_t k = 0; k < n_chunks && e == cudaSuccess && rc == TPC_OK; ++k) {
    Chunk& c = ch[k];
    cudaStream_t s = s_out;
    e = cudaEventSynchronize(t->host_events[k]);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_out, t->host_events[k], 0);
    if (e != cudaSuccess) break;
    const uint32_t* hh = t->host_headers + 4 * k;
    status |= hh[2]; tracklets += hh[3];
    tracks_all += hh[0]; hits_all += hh[1];
    const uint32_t nt_dev = hh[0] < c.tcap ? hh[0] : c.tcap, nh_dev = hh[1] < c.hcap ? hh[1] : c.hcap;
    uint32_t nt = nt_dev, nh = nh_dev;
    if ((uint64_t)tracks_off + nt > tcap) { nt = tcap - tracks_off; status |= TPC_STATUS_TRACK_OVERFLOW; }
    if ((uint64_t)hits_off + nh > hcap) { nh = hcap - hits_off; status |= TPC_STATUS_HIT_OVERFLOW; }
    const uint32_t m = nt_dev > nh_dev ? nt_dev : nh_dev;
    if (m && (c.task0 || hits_off || c.idx0))
      k_shift_chunk<<<(m + 255) / 256, 256, 0, s>>>(c.d.track_task, c.d.track_hit_begin, nt_dev, c.d.hit_cluster, nh_dev,
                                                    c.task0, hits_off, c.idx0);
    auto d2h = [&](void* dst, const void* src, size_t bytes) {
      if (e == cudaSuccess && dst && bytes) { e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, s); down += bytes; }
    };
    d2h(out->track_task ? out->track_task + tracks_off : nullptr, c.d.track_task, (size_t)nt * 4);
    d2h(out->track_hit_begin ? out->track_hit_begin + tracks_off : nullptr, c.d.track_hit_begin, (size_t)nt * 4);
    d2h(out->track_nhits ? out->track_nhits + tracks_off : nullptr, c.d.track_nhits, (size_t)nt * 4);
    d2h(out->track_ndf ? out->track_ndf + tracks_off : nullptr, c.d.track_ndf, (size_t)nt * 4);
    d2h(out->track_x ? out->track_x + tracks_off : nullptr, c.d.track_x, (size_t)nt * 4);
    d2h(out->track_chi2 ? out->track_chi2 + tracks_off : nullptr, c.d.track_chi2, (size_t)nt * 4);
    for (int j = 0; j < 5 && out->track_par; ++j)
      d2h(out->track_par + (size_t)j * tcap + tracks_off, c.d.track_par + (size_t)j * c.tcap, (size_t)nt * 4);
    for (int j = 0; j < 15 && out->track_cov; ++j)
      d2h(out->track_cov + (size_t)j * tcap + tracks_off, c.d.track_cov + (size_t)j * c.tcap, (size_t)nt * 4);
    d2h(out->hit_cluster ? out->hit_cluster + hits_off : nullptr, c.d.hit_cluster, (size_t)nh * 4);
    tracks_off += nt; hits_off += nh;
  }
  for (uint32_t k = 0; k < 3; ++k) {
    const cudaError_t e2 = cudaStreamSynchronize(t->host_streams[k]);
    if (e == cudaSuccess) e = e2;
  }
  t->timing_on = timing; t->counters_on = counters;
  if (rc != TPC_OK) return rc;
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_track_batch_host: CUDA: %s", cudaGetErrorString(e));
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_track_batch_host: CUDA launch: %s", cudaGetErrorString(e));
  out->header[0] = (uint32_t)(tracks_all > 0xFFFFFFFFull ? 0xFFFFFFFFull : tracks_all);
  out->header[1] = (uint32_t)(hits_all > 0xFFFFFFFFull ? 0xFFFFFFFFull : hits_all);
  out->header[2] = status;
  out->header[3] = tracklets;
  if (h2d_bytes) *h2d_bytes = up;
  if (d2h_bytes) *d2h_bytes = down;
  return TPC_OK;
}

// ---- pipelined host entry point: two batches in flight ---------------------------------------------
// submit(slot) queues the upload, the path and the download of the header of one batch on the tracker's own
// streams (copies in / kernels / copies out) and returns; collect(slot) waits for that batch, then copies its
// tracks and hits to the caller's host arrays.  With submit(k + 1) issued before collect(k), the upload of batch
// k + 1 and the download of batch k run under the kernels of their neighbours: in the steady state a batch costs
// what its kernels cost.  One chunk per batch (the persistent tracklet kernels cost 0.3 ms per extra chunk).
namespace {
int ensure_host_streams(tpc_tracker* t) {
  cudaError_t e = cudaSuccess;
  if (t->host_streams.empty()) {
    t->host_streams.resize(kHostChunks, nullptr);
    t->host_events.resize(2 * kHostChunks + 1, nullptr);
    for (auto& x : t->host_streams) if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&x, cudaStreamNonBlocking);
    for (auto& x : t->host_events) if (e == cudaSuccess) e = cudaEventCreateWithFlags(&x, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&t->host_headers, 16 * kHostChunks, cudaHostAllocDefault);
    if (e != cudaSuccess) {
      for (auto& x : t->host_streams) if (x) cudaStreamDestroy(x);
      for (auto& x : t->host_events) if (x) cudaEventDestroy(x);
      if (t->host_headers) cudaFreeHost(t->host_headers);
      t->host_streams.clear(); t->host_events.clear(); t->host_headers = nullptr;
      return fail(t, TPC_ERR_CUDA, "host streams: CUDA: %s", cudaGetErrorString(e));
    }
  }
  if (!t->pipe_headers) {
    e = cudaHostAlloc((void**)&t->pipe_headers, 2 * 16, cudaHostAllocDefault);
    for (auto& p : t->pipe) {
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p.in, cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p.done, cudaEventDisableTiming);
    }
    if (e != cudaSuccess) {
      for (auto& p : t->pipe) { if (p.in) cudaEventDestroy(p.in); if (p.done) cudaEventDestroy(p.done); p.in = p.done = nullptr; }
      if (t->pipe_headers) cudaFreeHost(t->pipe_headers);
      t->pipe_headers = nullptr;
      return fail(t, TPC_ERR_CUDA, "host pipeline: CUDA: %s", cudaGetErrorString(e));
    }
  }
  return TPC_OK;
}
}  // namespace

int tpc_host_submit(tpc_tracker* t, int slot, const tpc_clusters* in, uint32_t track_capacity, uint32_t hit_capacity,
                    void* workspace, size_t workspace_bytes, uint32_t max_tracklets) {
  if (!t) return TPC_ERR_ARGUMENT;
  if (slot < 0 || slot > 1) return fail(t, TPC_ERR_ARGUMENT, "tpc_host_submit: slot must be 0 or 1");
  if (!in || !in->row_offsets || (in->n_clusters && (!in->y || !in->z)))
    return fail(t, TPC_ERR_ARGUMENT, "tpc_host_submit: y, z, row_offsets must not be NULL");
  tpc_tracker::PipeSlot& ps = t->pipe[slot];
  if (ps.busy) return fail(t, TPC_ERR_ARGUMENT, "tpc_host_submit: slot %d has not been collected", slot);
  const uint32_t n = in->n_clusters, n_rows = (uint32_t)t->n_rows;
  if (in->row_offsets[(size_t)in->n_tasks * n_rows] != n)
    return fail(t, TPC_ERR_ARGUMENT, "tpc_host_submit: row_offsets must end at n_clusters");
  const uint32_t T_all = host_total_tracklets(t, n, max_tracklets, kHostChunks);
  const HostCarve h = host_carve(t, n, in->n_tasks, T_all, track_capacity, hit_capacity);
  if (!workspace || workspace_bytes < h.total)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_host_submit: workspace of %zu bytes, need %zu (tpc_host_workspace_bytes)", workspace_bytes, h.total);
  if (((uintptr_t)workspace & (kAlign - 1)) != 0)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_host_submit: workspace must be %zu-byte aligned", kAlign);
  int rc = ensure_host_streams(t);
  if (rc != TPC_OK) return rc;
  cudaStream_t s_in = t->host_streams[0], s_cmp = t->host_streams[1];
  char* ws = (char*)workspace;
  const size_t n_off = (size_t)in->n_tasks * n_rows + 1;
  cudaError_t e = cudaSuccess;
  uint64_t up = 0;
  auto h2d = [&](void* dst, const void* src, size_t bytes) {
    if (e == cudaSuccess && bytes) { e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, s_in); up += bytes; }
  };
  h2d(ws + h.y, in->y, (size_t)n * 4);
  h2d(ws + h.z, in->z, (size_t)n * 4);
  h2d(ws + h.row_off, in->row_offsets, n_off * 4);
  if (e == cudaSuccess) e = cudaEventRecord(ps.in, s_in);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(s_cmp, ps.in, 0);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_host_submit: CUDA: %s", cudaGetErrorString(e));
  tpc_clusters din{};
  din.y = (const float*)(ws + h.y); din.z = (const float*)(ws + h.z);
  din.row_offsets = (const uint32_t*)(ws + h.row_off); din.n_clusters = n; din.n_tasks = in->n_tasks;
  const uint32_t mh = (uint32_t)(t->prm.min_track_hits > 0 ? t->prm.min_track_hits : 1);
  tpc_tracks& d = ps.d;
  d = tpc_tracks{};
  ps.tcap = n / mh + 1u < track_capacity ? n / mh + 1u : track_capacity;
  ps.hcap = n + 1u < hit_capacity ? n + 1u : hit_capacity;
  d.track_capacity = ps.tcap; d.hit_capacity = ps.hcap;
  d.header = (uint32_t*)(ws + h.header);
  d.track_task = (uint32_t*)(ws + h.track_task); d.track_hit_begin = (uint32_t*)(ws + h.track_hit_begin);
  d.track_nhits = (uint32_t*)(ws + h.track_nhits); d.track_ndf = (int32_t*)(ws + h.track_ndf);
  d.track_x = (float*)(ws + h.track_x); d.track_chi2 = (float*)(ws + h.track_chi2);
  d.track_par = (float*)(ws + h.track_par); d.track_cov = (float*)(ws + h.track_cov);
  d.hit_cluster = (uint32_t*)(ws + h.hit_cluster);
  uint32_t T = resolve_max_tracklets(t, n, 0u);
  if (max_tracklets && max_tracklets < T) T = max_tracklets;
  const size_t need = carve(n_rows, n, in->n_tasks, T).total;
  if (h.inner + need > workspace_bytes) return fail(t, TPC_ERR_WORKSPACE, "tpc_host_submit: workspace too small");
  const bool timing = t->timing_on, counters = t->counters_on;
  t->timing_on = false; t->counters_on = false;
  rc = tpc_track_batch(t, &din, &d, ws + h.inner, need, T, s_cmp);
  t->timing_on = timing; t->counters_on = counters;
  if (rc != TPC_OK) return rc;
  e = cudaMemcpyAsync(t->pipe_headers + 4 * slot, d.header, 16, cudaMemcpyDeviceToHost, s_cmp);
  if (e == cudaSuccess) e = cudaEventRecord(ps.done, s_cmp);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_host_submit: CUDA: %s", cudaGetErrorString(e));
  ps.up = up;
  ps.busy = true;
  return TPC_OK;
}

int tpc_host_collect(tpc_tracker* t, int slot, tpc_tracks* out, uint64_t* h2d_bytes, uint64_t* d2h_bytes) {
  if (!t) return TPC_ERR_ARGUMENT;
  if (slot < 0 || slot > 1 || !out || !out->header) return fail(t, TPC_ERR_ARGUMENT, "tpc_host_collect: slot 0 or 1, tracks and header must not be NULL");
  tpc_tracker::PipeSlot& ps = t->pipe[slot];
  if (!ps.busy) return fail(t, TPC_ERR_ARGUMENT, "tpc_host_collect: nothing was submitted in slot %d", slot);
  ps.busy = false;
  cudaStream_t s_out = t->host_streams[2];
  cudaError_t e = cudaEventSynchronize(ps.done);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(s_out, ps.done, 0);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_host_collect: CUDA: %s", cudaGetErrorString(e));
  const uint32_t* hh = t->pipe_headers + 4 * slot;
  const uint32_t tcap = out->track_capacity, hcap = out->hit_capacity;
  uint32_t status = hh[2];
  uint32_t nt = hh[0] < ps.tcap ? hh[0] : ps.tcap, nh = hh[1] < ps.hcap ? hh[1] : ps.hcap;
  if (nt > tcap) { nt = tcap; status |= TPC_STATUS_TRACK_OVERFLOW; }
  if (nh > hcap) { nh = hcap; status |= TPC_STATUS_HIT_OVERFLOW; }
  uint64_t down = 16;
  const tpc_tracks& d = ps.d;
  auto d2h = [&](void* dst, const void* src, size_t bytes) {
    if (e == cudaSuccess && dst && bytes) { e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, s_out); down += bytes; }
  };
  d2h(out->track_task, d.track_task, (size_t)nt * 4);
  d2h(out->track_hit_begin, d.track_hit_begin, (size_t)nt * 4);
  d2h(out->track_nhits, d.track_nhits, (size_t)nt * 4);
  d2h(out->track_ndf, d.track_ndf, (size_t)nt * 4);
  d2h(out->track_x, d.track_x, (size_t)nt * 4);
  d2h(out->track_chi2, d.track_chi2, (size_t)nt * 4);
  for (int j = 0; j < 5 && out->track_par; ++j) d2h(out->track_par + (size_t)j * tcap, d.track_par + (size_t)j * ps.tcap, (size_t)nt * 4);
  for (int j = 0; j < 15 && out->track_cov; ++j) d2h(out->track_cov + (size_t)j * tcap, d.track_cov + (size_t)j * ps.tcap, (size_t)nt * 4);
  d2h(out->hit_cluster, d.hit_cluster, (size_t)nh * 4);
  const cudaError_t e2 = cudaStreamSynchronize(s_out);
  if (e == cudaSuccess) e = e2;
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_host_collect: CUDA: %s", cudaGetErrorString(e));
  out->header[0] = hh[0]; out->header[1] = hh[1]; out->header[2] = status; out->header[3] = hh[3];
  if (h2d_bytes) *h2d_bytes = ps.up;
  if (d2h_bytes) *d2h_bytes = down;
  return TPC_OK;
}

// ---- sector-segment merger + refit (SPEC 9) ------------------------------------------------------
namespace {
struct MergeCarve {
  size_t ends, row_start, row_list, best_out, best_chi, zero_begin, row_cnt, row_fill, scan, ticket, zero_end, ones_begin,
      key_in, ones_end, total;
  uint32_t tiles;
};
MergeCarve merge_carve(uint32_t cap, uint32_t n_tasks, uint32_t n_rows) {
  MergeCarve m{};
  const size_t n_tr = (size_t)n_tasks * n_rows + 2;
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes); return o; };
  m.ends = take((size_t)cap * kEndFloats * sizeof(float));
  m.row_start = take(n_tr * sizeof(uint32_t));
  m.row_list = take((size_t)cap * sizeof(uint32_t));
  m.best_out = take((size_t)cap * sizeof(int32_t));
  m.best_chi = take((size_t)cap * sizeof(float));
  m.tiles = (cap + kMergeThreads - 1) / kMergeThreads;
  if (m.tiles == 0) m.tiles = 1;
  m.zero_begin = off;  // cleared with one memset per call
  m.row_cnt = take(n_tr * sizeof(uint32_t));
  m.row_fill = take(n_tr * sizeof(uint32_t));
  m.scan = take((size_t)m.tiles * sizeof(unsigned long long));
  m.ticket = take(2 * sizeof(uint32_t));
  m.zero_end = off;
  m.ones_begin = off;  // set to all ones per call
  m.key_in = take((size_t)cap * sizeof(unsigned long long));
  m.ones_end = off;
  m.total = off;
  return m;
}
__global__ void k_merge_guard(const Ctx c, const MergeCtx m) {  // the tracker's status decides whether anything runs
  if (c.out.header[2] != 0u) atomicOr(&m.out.header[2], TPC_MERGE_STATUS_INPUT_OVERFLOW);
  else if (c.out.header[0] > m.out.capacity) atomicOr(&m.out.header[2], TPC_MERGE_STATUS_CAPACITY);
}
}  // namespace

void tpc_default_merge_params(tpc_merge_params* out) {
  if (out) { out->merge_chi2_max = 50.0f; out->merge_max_row_gap = 8; out->n_slices = 1; }
}

size_t tpc_merge_workspace_bytes(const tpc_tracker* t, uint32_t track_capacity, uint32_t max_tasks) {
  if (!t) return 0;
  return merge_carve(track_capacity, max_tasks, (uint32_t)t->n_rows).total;
}

int tpc_merge_refit(tpc_tracker* t, const tpc_clusters* in, const tpc_tracks* tracks, const tpc_merge_params* params,
                    tpc_merged* merged, void* workspace, size_t workspace_bytes, uint32_t max_tracklets,
                    void* merge_workspace, size_t merge_workspace_bytes, void* cuda_stream) {
  if (!t) return TPC_ERR_ARGUMENT;
  if (!in || !tracks || !merged) return fail(t, TPC_ERR_ARGUMENT, "tpc_merge_refit: clusters, tracks and merged must not be NULL");
  if (!merged->header || !merged->seg_next || !merged->seg_prev || !merged->merged_first || !merged->merged_nseg ||
      !merged->merged_nhits || !merged->merged_nfit || !merged->merged_sector || !merged->merged_ndf ||
      !merged->merged_x || !merged->merged_par || !merged->merged_cov || !merged->merged_chi2)
    return fail(t, TPC_ERR_ARGUMENT, "tpc_merge_refit: every array of tpc_merged must not be NULL");
  if (!tracks->header || !tracks->track_task || !tracks->track_hit_begin || !tracks->track_nhits || !tracks->track_ndf ||
      !tracks->track_x || !tracks->track_par || !tracks->track_cov || !tracks->track_chi2 || !tracks->hit_cluster)
    return fail(t, TPC_ERR_ARGUMENT, "tpc_merge_refit: tracks must be the complete output of tpc_track_batch");
  tpc_merge_params mp;
  if (params) mp = *params; else tpc_default_merge_params(&mp);
  if (!(mp.merge_chi2_max >= 0.f) || mp.merge_max_row_gap < 0 || mp.n_slices < 1)
    return fail(t, TPC_ERR_ARGUMENT, "tpc_merge_refit: need merge_chi2_max >= 0, merge_max_row_gap >= 0, n_slices >= 1");
  const uint32_t T = resolve_max_tracklets(t, in->n_clusters, max_tracklets);
  const Carve cv = carve((uint32_t)t->n_rows, in->n_clusters, in->n_tasks, T);
  if (!workspace || workspace_bytes < cv.total)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_merge_refit: workspace of %zu bytes, the tracker's call needed %zu", workspace_bytes, cv.total);
  const uint32_t cap = tracks->track_capacity;
  const MergeCarve mc = merge_carve(cap, in->n_tasks, (uint32_t)t->n_rows);
  if (!merge_workspace || merge_workspace_bytes < mc.total)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_merge_refit: merge workspace of %zu bytes, need %zu", merge_workspace_bytes, mc.total);
  if ((((uintptr_t)workspace | (uintptr_t)merge_workspace) & (kAlign - 1)) != 0)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_merge_refit: workspaces must be %zu-byte aligned", kAlign);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const Ctx c = make_ctx(t, in, tracks, (char*)workspace, cv, T);
  char* mw = (char*)merge_workspace;
  MergeCtx m{};
  m.out = *merged;
  m.chi2_max = mp.merge_chi2_max; m.max_row_gap = mp.merge_max_row_gap; m.n_slices = mp.n_slices;
  m.n_half = t->n_half; m.ca = t->merge_ca; m.sa = t->merge_sa;
  m.ends = (float4*)(mw + mc.ends);
  m.row_cnt = (uint32_t*)(mw + mc.row_cnt); m.row_start = (uint32_t*)(mw + mc.row_start);
  m.row_fill = (uint32_t*)(mw + mc.row_fill); m.row_list = (uint32_t*)(mw + mc.row_list);
  m.best_out = (int32_t*)(mw + mc.best_out); m.best_chi = (float*)(mw + mc.best_chi);
  m.key_in = (unsigned long long*)(mw + mc.key_in);
  m.scan = (unsigned long long*)(mw + mc.scan); m.ticket = (uint32_t*)(mw + mc.ticket);
  cudaError_t e = cudaMemsetAsync(mw + mc.zero_begin, 0, mc.zero_end - mc.zero_begin, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(mw + mc.ones_begin, 0xFF, mc.ones_end - mc.ones_begin, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(merged->header, 0, 4 * sizeof(uint32_t), s);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_merge_refit: CUDA memset: %s", cudaGetErrorString(e));
  const uint32_t blocks = mc.tiles;
  k_merge_guard<<<1, 1, 0, s>>>(c, m);
  if (cap > 0) {
    k_merge_ends<<<blocks, kMergeThreads, 0, s>>>(c, m);                                   // G1
    k_merge_row_scan<<<1, 1024, 0, s>>>(c, m);
    k_merge_row_fill<<<blocks, kMergeThreads, 0, s>>>(c, m);
    k_merge_match<<<blocks, kMergeThreads, 0, s>>>(c, m);                                  // G2..G5
    k_merge_link<<<blocks, kMergeThreads, 0, s>>>(c, m);                                   // G6
    k_merge_heads<<<blocks, kMergeThreads, 0, s>>>(c, m);                                  // G7
    k_merge_refit<<<t->merge_grid, kMergeThreads, (size_t)t->n_rows * sizeof(float), s>>>(c, m);  // F1..F3
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_merge_refit: CUDA launch: %s", cudaGetErrorString(e));
  return TPC_OK;
}

// ---- cluster transformation (SPEC 10) --------------------------------------------------------------
struct tpc_transform {
  TransformCtx c{};
  float* d_tables = nullptr;  // pitch, centre, ky [n_rows] each, then the map
  std::string err;
};

int tpc_transform_create(const tpc_geometry* g, const tpc_calibration* cal, tpc_transform** out) {
  if (!g || !cal || !out) return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_transform_create: geometry, calibration and out must not be NULL");
  *out = nullptr;
  if (g->n_sectors < 1 || g->n_rows < 1 || g->n_rows > kMaxRows || !cal->pad_pitch || !cal->n_pads || !cal->map ||
      cal->map_ny < 2 || cal->map_nz < 2 || !(cal->t_max > 0.f) || !(g->z_max > 0.f))
    return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_transform_create: need tables, map_ny >= 2, map_nz >= 2, t_max > 0");
  for (int r = 0; r < g->n_rows; ++r)
    if (cal->n_pads[r] < 2) return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_transform_create: n_pads must be >= 2 in every row");
  tpc_transform* t = new (std::nothrow) tpc_transform();
  if (!t) return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_transform_create: out of host memory");
  const int n = g->n_rows;
  const size_t n_map = (size_t)g->n_sectors * n * cal->map_nz * cal->map_ny * 2;
  const size_t map_off = ((size_t)3 * n + 3) & ~(size_t)3;  // the kernel reads the map as float2 / 16-byte groups
  std::vector<float> tab(map_off + n_map);
  for (int r = 0; r < n; ++r) {
    tab[r] = cal->pad_pitch[r];
    tab[n + r] = 0.5f * (float)(cal->n_pads[r] - 1);                              // X1
    tab[2 * n + r] = (float)(cal->map_ny - 1) / (float)(cal->n_pads[r] - 1);      // X3 ky
  }
  memcpy(tab.data() + map_off, cal->map, n_map * sizeof(float));
  cudaError_t e = cudaMalloc(&t->d_tables, tab.size() * sizeof(float));
  if (e == cudaSuccess) e = cudaMemcpy(t->d_tables, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    const int rc = fail(nullptr, TPC_ERR_CUDA, "tpc_transform_create: CUDA: %s (no CPU fallback exists)", cudaGetErrorString(e));
    if (t->d_tables) cudaFree(t->d_tables);
    delete t;
    cudaGetLastError();
    return rc;
  }
  TransformCtx& c = t->c;
  c.n_sectors = g->n_sectors; c.n_rows = n; c.my = cal->map_ny; c.mz = cal->map_nz;
  c.z_max = g->z_max; c.t0 = cal->t0; c.v_drift = cal->v_drift;
  c.kz = (float)(cal->map_nz - 1) / cal->t_max;                                   // X3 kz
  c.pitch = t->d_tables; c.centre = t->d_tables + n; c.ky = t->d_tables + 2 * n; c.map = t->d_tables + map_off;
  *out = t;
  return TPC_OK;
}

void tpc_transform_destroy(tpc_transform* t) {
  if (!t) return;
  if (t->d_tables) cudaFree(t->d_tables);
  delete t;
}

int tpc_transform_clusters(tpc_transform* t, const float* pad, const float* time, const uint32_t* row_offsets,
                           uint32_t n_clusters, uint32_t n_tasks, float* y, float* z, void* cuda_stream) {
  if (!t) return TPC_ERR_ARGUMENT;
  auto bad = [&](const char* msg) { t->err = msg; return TPC_ERR_ARGUMENT; };
  if (!row_offsets || (n_clusters && (!pad || !time || !y || !z))) return bad("tpc_transform_clusters: pad, time, row_offsets, y, z must not be NULL");
  if ((((uintptr_t)pad | (uintptr_t)time | (uintptr_t)y | (uintptr_t)z) & 15u) != 0) return bad("tpc_transform_clusters: pad, time, y, z must be 16-byte aligned");
  if ((uint64_t)n_tasks * (uint64_t)t->c.n_rows >= 0x7FFFFFFFull) return bad("tpc_transform_clusters: n_tasks*n_rows must be < 2^31");
  if (n_clusters == 0) return TPC_OK;
  TransformCtx c = t->c;
  c.pad = pad; c.time = time; c.row_off = row_offsets; c.n = n_clusters; c.n_tr = n_tasks * (uint32_t)c.n_rows;
  c.y = y; c.z = z;
  k_transform<<<(n_clusters + kXfChunk - 1) / kXfChunk, kXfThreads, 0, (cudaStream_t)cuda_stream>>>(c);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { t->err = std::string("tpc_transform_clusters: CUDA launch: ") + cudaGetErrorString(e); return TPC_ERR_CUDA; }
  return TPC_OK;
}

const char* tpc_transform_last_error(const tpc_transform* t) { return t ? t->err.c_str() : g_create_error.c_str(); }

// ---- frame slicer (SPEC 11, SLICE) ------------------------------------------------------------------
size_t tpc_slice_workspace_bytes(uint32_t n_tasks_in, int32_t n_rows, int32_t n_slices) {
  if (n_rows < 1 || n_slices < 1) return 0;
  return align_up(((size_t)n_tasks_in * (size_t)n_rows * (size_t)n_slices + 2) * sizeof(uint32_t));
}

int tpc_slice_frames(const float* y, const float* zeta, const uint32_t* row_offsets_in, uint32_t n_clusters,
                     uint32_t n_tasks_in, int32_t n_sectors, int32_t n_rows, float slice_len, int32_t n_slices,
                     float* y_out, float* z_out, uint32_t* src_index, uint32_t* row_offsets_out, void* workspace,
                     size_t workspace_bytes, void* cuda_stream) {
  if (!row_offsets_in || !row_offsets_out || !workspace || (n_clusters && (!y || !zeta || !y_out || !z_out || !src_index)))
    return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_slice_frames: NULL argument");
  if (n_sectors < 1 || n_rows < 1 || n_slices < 1 || n_slices > kMaxSlices || !(slice_len > 0.f) || n_tasks_in % (uint32_t)n_sectors != 0u)
    return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_slice_frames: need n_sectors, n_rows >= 1, 1 <= n_slices <= %d, slice_len > 0, whole frames", kMaxSlices);
  if ((uint64_t)n_tasks_in * (uint64_t)n_rows * (uint64_t)n_slices >= 0x7FFFFFFFull)
    return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_slice_frames: n_tasks_in*n_rows*n_slices must be < 2^31");
  if (workspace_bytes < tpc_slice_workspace_bytes(n_tasks_in, n_rows, n_slices))
    return fail(nullptr, TPC_ERR_WORKSPACE, "tpc_slice_frames: workspace too small");
  SliceCtx c{};
  c.y = y; c.z = zeta; c.row_off_in = row_offsets_in; c.n = n_clusters; c.n_tr_in = n_tasks_in * (uint32_t)n_rows;
  c.n_sectors = n_sectors; c.n_rows = n_rows; c.n_slices = n_slices;
  c.inv_len = 1.0f / slice_len;
  c.y_out = y_out; c.z_out = z_out; c.src_index = src_index; c.row_off_out = row_offsets_out;
  c.counts = (uint32_t*)workspace;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const unsigned blocks = (c.n_tr_in + kSliceThreads / 32 - 1) / (kSliceThreads / 32);
  if (blocks) k_slice_count<<<blocks, kSliceThreads, 0, s>>>(c);
  k_slice_scan<<<1, 1024, 0, s>>>(c);
  if (blocks) k_slice_scatter<<<blocks, kSliceThreads, 0, s>>>(c);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(nullptr, TPC_ERR_CUDA, "tpc_slice_frames: CUDA launch: %s", cudaGetErrorString(e));
  return TPC_OK;
}

// ---- frame slicer without caller scratch (include/tpc_tracker.h: tpc_slice_frames_static) -------------------
// The counts of the output rows live in this array.  In host code its NAME is a host-side stand-in, not a
// device address: the kernels get the address cudaGetSymbolAddress returns for the current device, resolved
// once per device (tpc_slice_static_setup) and kept in g_slice_static_ptr.
static __device__ __align__(256) uint32_t g_slice_static_counts[TPC_SLICE_STATIC_MAX_ENTRIES];
namespace {
constexpr int kSliceStaticMaxDevices = 64;
uint32_t* g_slice_static_ptr[kSliceStaticMaxDevices] = {nullptr};
std::mutex g_slice_static_mutex;

// Device address of g_slice_static_counts on the current device, or nullptr (error text set).
uint32_t* slice_static_address() {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    fail(nullptr, TPC_ERR_CUDA, "tpc_slice_static_setup: cudaGetDevice: %s", cudaGetErrorString(e));
    return nullptr;
  }
  if (dev < 0 || dev >= kSliceStaticMaxDevices) {
    fail(nullptr, TPC_ERR_ARGUMENT, "tpc_slice_static_setup: device %d, at most %d are supported", dev, kSliceStaticMaxDevices);
    return nullptr;
  }
  std::lock_guard<std::mutex> lock(g_slice_static_mutex);
  if (!g_slice_static_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_slice_static_counts);
    if (e != cudaSuccess || !p) {
      fail(nullptr, TPC_ERR_CUDA, "tpc_slice_static_setup: cudaGetSymbolAddress on device %d: %s", dev,
           cudaGetErrorString(e));
      cudaGetLastError();
      return nullptr;
    }
    g_slice_static_ptr[dev] = (uint32_t*)p;
  }
  return g_slice_static_ptr[dev];
}
}  // namespace

int tpc_slice_static_setup(void) { return slice_static_address() ? TPC_OK : TPC_ERR_CUDA; }

int tpc_slice_frames_static(const float* y, const float* zeta, const uint32_t* row_offsets_in, uint32_t n_clusters,
                            uint32_t n_tasks_in, int32_t n_sectors, int32_t n_rows, float slice_len, int32_t n_slices,
                            float* y_out, float* z_out, uint32_t* src_index, uint32_t* row_offsets_out,
                            void* cuda_stream) {
  if (!row_offsets_in || !row_offsets_out || (n_clusters && (!y || !zeta || !y_out || !z_out || !src_index)))
    return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_slice_frames_static: NULL argument");
  if (n_sectors < 1 || n_rows < 1 || n_slices < 1 || n_slices > kMaxSlices || !(slice_len > 0.f) || n_tasks_in % (uint32_t)n_sectors != 0u)
    return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_slice_frames_static: need n_sectors, n_rows >= 1, 1 <= n_slices <= %d, slice_len > 0, whole frames", kMaxSlices);
  const uint64_t entries = (uint64_t)n_tasks_in * (uint64_t)n_rows * (uint64_t)n_slices + 2u;
  if (entries > (uint64_t)TPC_SLICE_STATIC_MAX_ENTRIES)
    return fail(nullptr, TPC_ERR_WORKSPACE,
                "tpc_slice_frames_static: n_tasks_in*n_rows*n_slices + 2 = %llu entries of scratch, the static array "
                "holds %u: slice fewer frames per call or use tpc_slice_frames with a workspace",
                (unsigned long long)entries, (unsigned)TPC_SLICE_STATIC_MAX_ENTRIES);
  uint32_t* counts = slice_static_address();
  if (!counts) return TPC_ERR_CUDA;
  SliceCtx c{};
  c.y = y; c.z = zeta; c.row_off_in = row_offsets_in; c.n = n_clusters; c.n_tr_in = n_tasks_in * (uint32_t)n_rows;
  c.n_sectors = n_sectors; c.n_rows = n_rows; c.n_slices = n_slices;
  c.inv_len = 1.0f / slice_len;
  c.y_out = y_out; c.z_out = z_out; c.src_index = src_index; c.row_off_out = row_offsets_out;
  c.counts = counts;  // every entry a call reads is written by its k_slice_count first: nothing to clear
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const unsigned blocks = (c.n_tr_in + kSliceThreads / 32 - 1) / (kSliceThreads / 32);
  if (blocks) k_slice_count<<<blocks, kSliceThreads, 0, s>>>(c);
  k_slice_scan<<<1, 1024, 0, s>>>(c);
  if (blocks) k_slice_scatter<<<blocks, kSliceThreads, 0, s>>>(c);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(nullptr, TPC_ERR_CUDA, "tpc_slice_frames_static: CUDA launch: %s", cudaGetErrorString(e));
  return TPC_OK;
}

// ---- ITS standalone tracker (SPEC 12) -----------------------------------------------------------------
struct tpc_its_tracker {
  ItsCtx c{};
  std::string err;
};
namespace {
struct ItsCarve { size_t best1, best0, tl_a, tl_b, tl_ev, recs, zero_begin, scan_tl, scan_out, tickets, n_tracklets, zero_end, total; uint32_t max_tl, tiles_n, tiles_tl; };
ItsCarve its_carve(uint32_t n, uint32_t) {
  ItsCarve v{};
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes); return o; };
  v.max_tl = n / 2u + 1u;  // a tracklet holds two clusters
  v.tiles_n = (n + kItsThreads - 1) / kItsThreads; if (v.tiles_n == 0) v.tiles_n = 1;
  v.tiles_tl = (v.max_tl + kItsThreads - 1) / kItsThreads;
  v.best1 = take((size_t)(n + 1) * 4); v.best0 = take((size_t)(n + 1) * 4);
  v.tl_a = take((size_t)v.max_tl * 4); v.tl_b = take((size_t)v.max_tl * 4); v.tl_ev = take((size_t)v.max_tl * 4);
  v.recs = take((size_t)v.max_tl * sizeof(ItsRec));
  v.zero_begin = off;
  v.scan_tl = take((size_t)v.tiles_n * 8); v.scan_out = take((size_t)v.tiles_tl * 8);
  v.tickets = take(2 * 4); v.n_tracklets = take(4);
  v.zero_end = off;
  v.total = off;
  return v;
}
}  // namespace

void tpc_its_default_params(tpc_its_params* p) {
  if (!p) return;
  p->max_sinphi_pair = 0.03f; p->max_dtan = 0.02f; p->sig_sinphi = 0.002f; p->sig_tan = 0.004f;
  p->sig_vtx_xy = 0.01f; p->sig_vtx_z = 0.01f; p->chi2_max = 30.0f; p->max_dx = 2.0f;
  p->c0_sinphi = 1.0f; p->c0_dzds = 1.0f; p->c0_qpt = 100.0f; p->turn_cov_scale = 100.0f; p->max_sinphi = 0.95f;
  p->min_clusters = 4;
}

int tpc_its_create(const tpc_its_geometry* g, float bz_kgauss, const tpc_its_params* params, tpc_its_tracker** out) {
  if (!g || !out) return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_its_create: geometry and out must not be NULL");
  *out = nullptr;
  for (int l = 0; l < 6; ++l)
    if (!(g->R[l] > 0.f) || (l && !(g->R[l] > g->R[l - 1])) || !(g->sig_rphi[l] > 0.f) || !(g->sig_z[l] > 0.f) || !(g->xx0[l] >= 0.f))
      return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_its_create: radii must grow, errors must be positive, material >= 0");
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaFree(nullptr) != cudaSuccess) {
    cudaGetLastError();
    return fail(nullptr, TPC_ERR_CUDA, "tpc_its_create: no CUDA device (no CPU fallback exists)");
  }
  tpc_its_tracker* t = new (std::nothrow) tpc_its_tracker();
  if (!t) return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_its_create: out of host memory");
  ItsCtx& c = t->c;
  if (params) c.prm = *params; else tpc_its_default_params(&c.prm);
  const tpc_its_params& p = c.prm;
  if (!(p.sig_sinphi > 0.f) || !(p.sig_tan > 0.f) || !(p.sig_vtx_xy > 0.f) || !(p.sig_vtx_z > 0.f) || p.min_clusters < 2) {
    delete t;
    return fail(nullptr, TPC_ERR_ARGUMENT, "tpc_its_create: need positive sigmas and min_clusters >= 2");
  }
  for (int l = 0; l < 6; ++l) {
    c.R[l] = g->R[l];
    c.sr2[l] = g->sig_rphi[l] * g->sig_rphi[l];
    c.sz2[l] = g->sig_z[l] * g->sig_z[l];
    c.ms2[l] = (0.0136f * 0.0136f) * g->xx0[l];
  }
  c.a = -0.000299792458f * bz_kgauss;
  c.wphi = 1.0f / (p.sig_sinphi * p.sig_sinphi); c.wtan = 1.0f / (p.sig_tan * p.sig_tan);
  c.svxy2 = p.sig_vtx_xy * p.sig_vtx_xy; c.svz2 = p.sig_vtx_z * p.sig_vtx_z;
  *out = t;
  return TPC_OK;
}

void tpc_its_destroy(tpc_its_tracker* t) { delete t; }

size_t tpc_its_workspace_bytes(const tpc_its_tracker* t, uint32_t max_clusters, uint32_t max_events) {
  return t ? its_carve(max_clusters, max_events).total : 0;
}

int tpc_its_track_batch(tpc_its_tracker* t, const float* x, const float* y, const float* z, const uint32_t* layer_offsets,
                        const float* vertex, uint32_t n_clusters, uint32_t n_events, tpc_its_tracks* tracks, void* workspace,
                        size_t workspace_bytes, void* cuda_stream) {
  if (!t) return TPC_ERR_ARGUMENT;
  auto bad = [&](int code, const char* msg) { t->err = msg; return code; };
  if (!layer_offsets || !tracks || (n_events && !vertex) || (n_clusters && (!x || !y || !z)))
    return bad(TPC_ERR_ARGUMENT, "tpc_its_track_batch: NULL argument");
  if (!tracks->header || !tracks->event || !tracks->cluster || !tracks->n_clusters || !tracks->frame || !tracks->out_state ||
      !tracks->in_state || !tracks->out_ndf || !tracks->in_ndf)
    return bad(TPC_ERR_ARGUMENT, "tpc_its_track_batch: every array of tpc_its_tracks must not be NULL");
  if (n_clusters >= 0x7FFFFFFFu || (uint64_t)n_events * 6u >= 0x7FFFFFFFull) return bad(TPC_ERR_ARGUMENT, "tpc_its_track_batch: too many clusters or events");
  const ItsCarve v = its_carve(n_clusters, n_events);
  if (!workspace || workspace_bytes < v.total) return bad(TPC_ERR_WORKSPACE, "tpc_its_track_batch: workspace too small (tpc_its_workspace_bytes)");
  if (((uintptr_t)workspace & (kAlign - 1)) != 0) return bad(TPC_ERR_WORKSPACE, "tpc_its_track_batch: workspace must be 256-byte aligned");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  ItsCtx c = t->c;
  c.x = x; c.y = y; c.z = z; c.lo = layer_offsets; c.vtx = vertex; c.n = n_clusters; c.n_events = n_events;
  c.max_tracklets = v.max_tl;
  c.best1 = (int32_t*)(ws + v.best1); c.best0 = (int32_t*)(ws + v.best0);
  c.tl_a = (uint32_t*)(ws + v.tl_a); c.tl_b = (uint32_t*)(ws + v.tl_b); c.tl_ev = (uint32_t*)(ws + v.tl_ev);
  c.recs = (ItsRec*)(ws + v.recs);
  c.scan_tl = (unsigned long long*)(ws + v.scan_tl); c.scan_out = (unsigned long long*)(ws + v.scan_out);
  c.tickets = (uint32_t*)(ws + v.tickets); c.n_tracklets = (uint32_t*)(ws + v.n_tracklets);
  c.out = *tracks;
  cudaError_t e = cudaMemsetAsync(ws + v.zero_begin, 0, v.zero_end - v.zero_begin, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(tracks->header, 0, 16, s);
  if (e != cudaSuccess) return bad(TPC_ERR_CUDA, "tpc_its_track_batch: CUDA memset failed");
  if (n_clusters > 0 && n_events > 0) {
    k_its_pairs<<<dim3(kItsBlocksPerEvent, n_events, 2), kItsThreads, 0, s>>>(c);
    k_its_tracklets<<<v.tiles_n, kItsThreads, 0, s>>>(c);
    k_its_follow<<<(v.max_tl + kItsThreads / 32 - 1) / (kItsThreads / 32), kItsThreads, 0, s>>>(c);
    k_its_output<<<v.tiles_tl, kItsThreads, 0, s>>>(c);
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) { t->err = std::string("tpc_its_track_batch: CUDA launch: ") + cudaGetErrorString(e); return TPC_ERR_CUDA; }
  return TPC_OK;
}

const char* tpc_its_last_error(const tpc_its_tracker* t) { return t ? t->err.c_str() : g_create_error.c_str(); }

const char* tpc_last_error(const tpc_tracker* t) { return t ? t->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
