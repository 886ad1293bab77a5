// Host side of the C ABI in include/tpc_tracker.h: tables (docs/ARITH_SPEC.md
// section 1), workspace carving and the launch sequence a1..a7.  No host
// synchronisation and no allocation on the tpc_track_batch path.
//
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -fmad=false
//        -prec-div=true -prec-sqrt=true -ftz=false --shared -Xcompiler -fPIC
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/tpc_tracker.h"
#include "device_common.cuh"
#include "stage_neighbours.cuh"
#include "stage_output.cuh"
#include "stage_tracklet.cuh"
#include "stages_ca.cuh"

using namespace tpc;

struct tpc_tracker {
  int32_t n_sectors = 0, n_rows = 0;
  float z_max = 0.f, bz = 0.f;
  tpc_params prm{};
  float a = 0.f, sy2 = 0.f, sz2 = 0.f, wy = 0.f, wz = 0.f, smax2 = 0.f;
  float* d_tables = nullptr;               // [6][n_rows]: X, ymax, dx_up, dx_dn, ratio_up, ratio_dn
  unsigned long long* d_counters = nullptr;  // [CN_COUNT]
  bool counters_on = false;
  // persistent tracklet kernel: [counters off/on] -> blocks that fit the device at once
  size_t trk_smem = 0;
  int trk_grid[2] = {0, 0};
  // stage timing: ring of TPC_STAGE_RING calls x (TPC_N_STAGES + 1) events, created on first use
  bool timing_on = false;
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

// Offsets of every workspace array, in bytes.
struct Carve {
  size_t yz, gid, bins, rowinfo, link_up, link_dn, clean_up, owner, trk_seed, trk_hits, trk_rec, zero_begin,
      scan_seed, scan_out, tickets, n_tracklets, zero_end, total;
  uint32_t seed_tiles, out_tiles;
};

Carve carve(uint32_t n_rows, uint32_t n, uint32_t n_tasks, uint32_t T) {
  Carve c{};
  const size_t n_tr = (size_t)n_tasks * n_rows;
  const size_t n4 = ((size_t)n + 3) / 4 * 4 + 4;  // k_seeds reads in groups of 4
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes); return o; };
  c.yz = take(n4 * sizeof(float2));
  c.gid = take(n4 * sizeof(uint32_t));
  c.bins = take(((size_t)kBinsPerCluster * n + n_tr * kBinPad + 16) * sizeof(uint32_t));  // + slack of the 16-byte aligned bulk copies
  c.rowinfo = take((n_tr + 1) * sizeof(RowInfo));
  c.link_up = take(n4 * sizeof(int32_t));
  c.link_dn = take(n4 * sizeof(int32_t));
  c.clean_up = take(n4 * sizeof(int32_t));
  c.owner = take(n4 * sizeof(unsigned long long));
  c.trk_seed = take((size_t)T * kSeedU4 * sizeof(uint4));
  c.trk_hits = take((size_t)T * map_stride((int)n_rows) * sizeof(uint32_t));
  c.trk_rec = take((size_t)T * kRecFloat4 * sizeof(float4));
  c.seed_tiles = (uint32_t)(((size_t)n + kSeedTile - 1) / kSeedTile);
  if (c.seed_tiles == 0) c.seed_tiles = 1;
  c.out_tiles = (uint32_t)(((size_t)T + kOutThreads - 1) / kOutThreads);
  if (c.out_tiles == 0) c.out_tiles = 1;
  c.zero_begin = off;  // everything from here to zero_end is cleared by one memset per call
  c.scan_seed = take((size_t)c.seed_tiles * sizeof(unsigned long long));
  c.scan_out = take((size_t)c.out_tiles * sizeof(unsigned long long));
  c.tickets = take(8 * sizeof(uint32_t));
  c.n_tracklets = take(sizeof(uint32_t));
  c.zero_end = off;
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
  c.rowinfo = (RowInfo*)(ws + cv.rowinfo);
  c.link_up = (int32_t*)(ws + cv.link_up); c.link_dn = (int32_t*)(ws + cv.link_dn);
  c.clean_up = (int32_t*)(ws + cv.clean_up); c.owner = (unsigned long long*)(ws + cv.owner);
  c.trk_seed = (uint4*)(ws + cv.trk_seed);
  c.trk_hits = (uint32_t*)(ws + cv.trk_hits); c.trk_rec = (float4*)(ws + cv.trk_rec);
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
  const int n = g->n_rows;
  std::vector<float> tab((size_t)6 * n, 0.f);
  float *X = tab.data(), *ymax = X + n, *dx_up = X + 2 * n, *dx_dn = X + 3 * n, *ratio_up = X + 4 * n,
        *ratio_dn = X + 5 * n;
  for (int r = 0; r < n; ++r) X[r] = g->row_x[r];
  for (int r = 0; r < n; ++r) ymax[r] = X[r] * g->tan_half_angle + 1.0f;                    // T1
  for (int r = 0; r + 1 < n; ++r) { dx_up[r] = X[r + 1] - X[r]; ratio_up[r] = X[r + 1] / X[r]; }  // T2 T4
  for (int r = 1; r < n; ++r) { dx_dn[r] = X[r] - X[r - 1]; ratio_dn[r] = X[r - 1] / X[r]; }      // T3 T5
  t->a = -0.000299792458f * bz_kgauss;                                                       // T6
  t->sy2 = p.sigma_y * p.sigma_y; t->sz2 = p.sigma_z * p.sigma_z;                            // T7
  t->wy = 1.0f / t->sy2; t->wz = 1.0f / t->sz2;
  t->smax2 = p.search_max * p.search_max;                                                    // T8
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
  // launch shape of the persistent tracklet constructor: as many blocks as the device holds at once
  int dev = 0, n_sm = 0;
  e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute((const void*)k_neighbours<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)kNfSmemBytes);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute((const void*)k_neighbours<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)kNfSmemBytes);
  t->trk_smem = (size_t)t->n_rows * sizeof(float);
  for (int cnt = 0; cnt < 2 && e == cudaSuccess; ++cnt) {
    const void* fn = cnt ? (const void*)k_tracklets<true> : (const void*)k_tracklets<false>;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, kTrackletThreads, t->trk_smem);
    t->trk_grid[cnt] = (per_sm > 0 ? per_sm : 1) * n_sm;
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
  if (t->d_tables) cudaFree(t->d_tables);
  if (t->d_counters) cudaFree(t->d_counters);
  delete t;
}

size_t tpc_workspace_bytes(const tpc_tracker* t, uint32_t max_clusters, uint32_t max_tasks, uint32_t max_tracklets) {
  if (!t) return 0;
  const uint32_t T = resolve_max_tracklets(t, max_clusters, max_tracklets);
  return carve((uint32_t)t->n_rows, max_clusters, max_tasks, T).total;
}

int tpc_launches_per_batch(const tpc_tracker*) { return 6; }  // a1, a2, a3, a4, a5, a6+a7

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
                                                  "tracklet_constructor", "selector_output"};
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
      t->ev.resize((size_t)TPC_STAGE_RING * (TPC_N_STAGES + 1));
      for (cudaEvent_t& x : t->ev)
        if (cudaEventCreate(&x) != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_track_batch: cudaEventCreate failed");
    }
    ev = t->ev.data() + (size_t)(t->timed_calls % TPC_STAGE_RING) * (TPC_N_STAGES + 1);
    ++t->timed_calls;
  }
  int stage = 0;
  auto mark = [&]() { if (ev) cudaEventRecord(ev[stage], s); ++stage; };
  mark();
  if (c.n_tr > 0) {
    if (cnt) k_grid_build<true><<<c.n_tr, kGridThreads, 0, s>>>(c);                         // a1
    else k_grid_build<false><<<c.n_tr, kGridThreads, 0, s>>>(c);
  }
  mark();
  if (c.n_tr > 0) {
    if (cnt) k_neighbours<true><<<c.n_tr, kNfThreads, kNfSmemBytes, s>>>(c);                // a2
    else k_neighbours<false><<<c.n_tr, kNfThreads, kNfSmemBytes, s>>>(c);
  }
  mark();
  if (c.n > 0) {
    k_clean<<<(c.n + kCleanThreads - 1) / kCleanThreads, kCleanThreads, 0, s>>>(c);         // a3
  }
  mark();
  if (cnt) k_seeds<true><<<cv.seed_tiles, kSeedThreads, 0, s>>>(c);                         // a4
  else k_seeds<false><<<cv.seed_tiles, kSeedThreads, 0, s>>>(c);
  mark();
  // a5: persistent, as many blocks as the device holds at once
  if (cnt) k_tracklets<true><<<t->trk_grid[1], kTrackletThreads, t->trk_smem, s>>>(c);
  else k_tracklets<false><<<t->trk_grid[0], kTrackletThreads, t->trk_smem, s>>>(c);
  mark();
  const size_t keep_smem = (size_t)kOutThreads * ((size_t)(t->n_rows + 31) / 32) * sizeof(uint32_t);
  k_select_output<<<cv.out_tiles, kOutThreads, keep_smem, s>>>(c);                          // a6 + a7
  mark();
  if (c.n > 0 && (out->dbg_link_up || out->dbg_link_dn || out->dbg_clean_up || out->dbg_clean_dn ||
                  out->dbg_start_hits))
    k_debug_links<<<(c.n + 255) / 256, 256, 0, s>>>(c);
  if (out->dbg_tracklet_capacity &&
      (out->dbg_tracklet_start || out->dbg_tracklet_nhits || out->dbg_tracklet_map || out->dbg_tracklet_par))
    k_debug_tracklets<<<(out->dbg_tracklet_capacity + 127) / 128, 128, 0, s>>>(c);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_track_batch: CUDA launch: %s", cudaGetErrorString(e));
  return TPC_OK;
}

// ---- host-buffer variant -------------------------------------------------------
namespace {
struct HostCarve {
  size_t y, z, row_off, header, track_task, track_hit_begin, track_nhits, track_ndf, track_x, track_par, track_cov,
      track_chi2, hit_cluster, inner, total;
};
HostCarve host_carve(const tpc_tracker* t, uint32_t n, uint32_t n_tasks, uint32_t T, uint32_t tcap, uint32_t hcap) {
  HostCarve h{};
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align_up(off + bytes); return o; };
  h.y = take((size_t)n * 4); h.z = take((size_t)n * 4);
  h.row_off = take(((size_t)n_tasks * t->n_rows + 1) * 4);
  h.header = take(16);
  h.track_task = take((size_t)tcap * 4); h.track_hit_begin = take((size_t)tcap * 4);
  h.track_nhits = take((size_t)tcap * 4); h.track_ndf = take((size_t)tcap * 4); h.track_x = take((size_t)tcap * 4);
  h.track_par = take((size_t)tcap * 20); h.track_cov = take((size_t)tcap * 60); h.track_chi2 = take((size_t)tcap * 4);
  h.hit_cluster = take((size_t)hcap * 4);
  h.inner = off;
  h.total = off + carve((uint32_t)t->n_rows, n, n_tasks, T).total;
  return h;
}
}  // namespace

size_t tpc_host_workspace_bytes(const tpc_tracker* t, uint32_t max_clusters, uint32_t max_tasks, uint32_t max_tracklets,
                                uint32_t track_capacity, uint32_t hit_capacity) {
  if (!t) return 0;
  const uint32_t T = resolve_max_tracklets(t, max_clusters, max_tracklets);
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
  const uint32_t T = resolve_max_tracklets(t, n, max_tracklets);
  const HostCarve h = host_carve(t, n, in->n_tasks, T, tcap, hcap);
  if (!workspace || workspace_bytes < h.total)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_track_batch_host: workspace of %zu bytes, need %zu", workspace_bytes, h.total);
  if (((uintptr_t)workspace & (kAlign - 1)) != 0)
    return fail(t, TPC_ERR_WORKSPACE, "tpc_track_batch_host: workspace must be %zu-byte aligned", kAlign);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  const size_t n_off = (size_t)in->n_tasks * t->n_rows + 1;
  uint64_t up = 0, down = 0;
  cudaError_t e = cudaSuccess;
  auto h2d = [&](size_t off, const void* src, size_t bytes) {
    if (e == cudaSuccess && bytes) { e = cudaMemcpyAsync(ws + off, src, bytes, cudaMemcpyHostToDevice, s); up += bytes; }
  };
  h2d(h.y, in->y, (size_t)n * 4);
  h2d(h.z, in->z, (size_t)n * 4);
  h2d(h.row_off, in->row_offsets, n_off * 4);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_track_batch_host: CUDA H2D: %s", cudaGetErrorString(e));
  tpc_clusters din = *in;
  din.x = nullptr; din.charge = nullptr;  // not read (R18, R23), so not copied either
  din.y = (const float*)(ws + h.y); din.z = (const float*)(ws + h.z);
  din.row_offsets = (const uint32_t*)(ws + h.row_off);
  tpc_tracks dout{};
  dout.track_capacity = tcap; dout.hit_capacity = hcap;
  dout.header = (uint32_t*)(ws + h.header);
  dout.track_task = (uint32_t*)(ws + h.track_task); dout.track_hit_begin = (uint32_t*)(ws + h.track_hit_begin);
  dout.track_nhits = (uint32_t*)(ws + h.track_nhits); dout.track_ndf = (int32_t*)(ws + h.track_ndf);
  dout.track_x = (float*)(ws + h.track_x); dout.track_par = (float*)(ws + h.track_par);
  dout.track_cov = (float*)(ws + h.track_cov); dout.track_chi2 = (float*)(ws + h.track_chi2);
  dout.hit_cluster = (uint32_t*)(ws + h.hit_cluster);
  const int rc = tpc_track_batch(t, &din, &dout, ws + h.inner, workspace_bytes - h.inner, T, cuda_stream);
  if (rc != TPC_OK) return rc;
  e = cudaMemcpyAsync(out->header, dout.header, 16, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_track_batch_host: CUDA: %s", cudaGetErrorString(e));
  down += 16;
  const uint32_t nt = out->header[0] < tcap ? out->header[0] : tcap;
  const uint32_t nh = out->header[1] < hcap ? out->header[1] : hcap;
  auto d2h = [&](void* dst, const void* src, size_t bytes) {
    if (e == cudaSuccess && dst && bytes) { e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, s); down += bytes; }
  };
  d2h(out->track_task, dout.track_task, (size_t)nt * 4);
  d2h(out->track_hit_begin, dout.track_hit_begin, (size_t)nt * 4);
  d2h(out->track_nhits, dout.track_nhits, (size_t)nt * 4);
  d2h(out->track_ndf, dout.track_ndf, (size_t)nt * 4);
  d2h(out->track_x, dout.track_x, (size_t)nt * 4);
  d2h(out->track_chi2, dout.track_chi2, (size_t)nt * 4);
  for (int j = 0; j < 5 && out->track_par; ++j)
    d2h(out->track_par + (size_t)j * tcap, dout.track_par + (size_t)j * tcap, (size_t)nt * 4);
  for (int j = 0; j < 15 && out->track_cov; ++j)
    d2h(out->track_cov + (size_t)j * tcap, dout.track_cov + (size_t)j * tcap, (size_t)nt * 4);
  d2h(out->hit_cluster, dout.hit_cluster, (size_t)nh * 4);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, "tpc_track_batch_host: CUDA D2H: %s", cudaGetErrorString(e));
  if (h2d_bytes) *h2d_bytes = up;
  if (d2h_bytes) *d2h_bytes = down;
  return TPC_OK;
}

const char* tpc_last_error(const tpc_tracker* t) { return t ? t->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
