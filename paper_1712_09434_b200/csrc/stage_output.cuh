// a6 tracklet selector + a7 output compaction (docs/ARITH_SPEC.md section 7, L1..L4),
// and the untimed debug kernels that translate internal idx to gid.
#pragma once
#include "device_common.cuh"
#include "stage_tracklet.cuh"

namespace tpc {

constexpr int kOutThreads = 128;

// One thread per tracklet.  Pass 1 counts the hits the tracklet still owns (L1);
// the block then takes its place in the output with an ordered chained scan over
// (tracks, hits) packed as tracks<<32 | hits; pass 2 writes the track and its
// hits as gids in ascending row order (L3).  Output order = tracklet order.
__global__ void __launch_bounds__(kOutThreads) k_select_output(const Ctx c) {
  __shared__ uint32_t s_warp[33];
  __shared__ uint32_t s_tile;
  __shared__ unsigned long long s_prefix;
  if (threadIdx.x == 0) s_tile = atomicAdd(&c.tickets[1], 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t n_trk = *c.n_tracklets;
  // the grid covers max_tracklets; tiles past the last tracklet have nothing to add and nobody waits for them
  const uint32_t last_tile = n_trk > 0u ? (n_trk - 1u) / kOutThreads : 0u;
  if (tile > last_tile) return;
  const uint32_t t = tile * kOutThreads + threadIdx.x;
  const uint32_t T = c.max_tracklets;
  const int n_rows = c.n_rows;
  int first_row = 0, last_row = -1;
  uint32_t kept = 0u;
  unsigned long long key = 0ull;
  if (t < n_trk) {
    const int n_hits = c.trk_rows[2u * T + t];
    if (n_hits >= c.prm.min_track_hits) {                              // K6
      first_row = c.trk_rows[t];
      last_row = c.trk_rows[T + t];
      key = ((unsigned long long)(uint32_t)n_hits << 32) |
            (unsigned long long)(0xFFFFFFFFu - c.gid[c.trk_start[t]]);
      for (int r = first_row; r <= last_row; ++r) {
        const int32_t m = c.trk_map[map_index(t, r, n_rows)];
        if (m >= 0 && c.owner[m] == key) ++kept;                       // L1
      }
    }
  }
  const bool is_track = kept >= (uint32_t)c.prm.min_track_hits && kept > 0u;  // L2
  const uint32_t my_hits = is_track ? kept : 0u;
  uint32_t tot_tracks, tot_hits;
  const uint32_t ex_tracks = block_exclusive_scan(is_track ? 1u : 0u, s_warp, &tot_tracks);
  const uint32_t ex_hits = block_exclusive_scan(my_hits, s_warp, &tot_hits);
  const unsigned long long agg = ((unsigned long long)tot_tracks << 32) | (unsigned long long)tot_hits;
  if (threadIdx.x < 32) {
    const unsigned long long p = lookback_exclusive(c.scan_out, tile, agg);
    if (threadIdx.x == 0) s_prefix = p;
  }
  __syncthreads();
  const unsigned long long prefix = s_prefix;
  if (is_track) {
    const uint32_t slot = (uint32_t)(prefix >> 32) + ex_tracks;
    const uint32_t hb = (uint32_t)(prefix & 0xFFFFFFFFull) + ex_hits;
    const tpc_tracks& o = c.out;
    if (slot >= o.track_capacity) {
      atomicOr(&o.header[2], TPC_STATUS_TRACK_OVERFLOW);
    } else {
      const size_t cap = o.track_capacity;
      o.track_task[slot] = c.trk_tr[t] / (uint32_t)n_rows;
      o.track_hit_begin[slot] = hb;
      o.track_nhits[slot] = kept;
      o.track_ndf[slot] = c.trk_ndf[t];
      const float* st = c.trk_state + t;
      o.track_x[slot] = st[0];
#pragma unroll
      for (int j = 0; j < 5; ++j) o.track_par[(size_t)j * cap + slot] = st[(size_t)(1 + j) * T];
#pragma unroll
      for (int j = 0; j < 15; ++j) o.track_cov[(size_t)j * cap + slot] = st[(size_t)(6 + j) * T];
      o.track_chi2[slot] = st[(size_t)21 * T];
      if ((unsigned long long)hb + kept > (unsigned long long)o.hit_capacity) {
        atomicOr(&o.header[2], TPC_STATUS_HIT_OVERFLOW);
      } else {
        uint32_t w = hb;
        for (int r = first_row; r <= last_row; ++r) {
          const int32_t m = c.trk_map[map_index(t, r, n_rows)];
          if (m >= 0 && c.owner[m] == key) o.hit_cluster[w++] = c.gid[m];
        }
      }
    }
  }
  if (threadIdx.x == 0 && tile == last_tile) {  // the last tile knows the totals
    const unsigned long long all = prefix + agg;
    c.out.header[0] = (uint32_t)(all >> 32);
    c.out.header[1] = (uint32_t)(all & 0xFFFFFFFFull);
  }
}

// ---------------------------------------------------------------------------
// debug (untimed): links and cleaned links as gids indexed by gid; start hits
// (S1) as an unordered gid list; tracklets before selection.
// ---------------------------------------------------------------------------
__global__ void k_debug_links(const Ctx c) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= c.n) return;
  const uint32_t g = c.gid[i];
  const int32_t u = c.link_up[i], d = c.link_dn[i];
  const int32_t cu = (u >= 0 && c.link_dn[u] == (int32_t)i) ? u : -1;
  const int32_t cd = (d >= 0 && c.link_up[d] == (int32_t)i) ? d : -1;
  const tpc_tracks& o = c.out;
  if (o.dbg_link_up) o.dbg_link_up[g] = u >= 0 ? (int32_t)c.gid[u] : -1;
  if (o.dbg_link_dn) o.dbg_link_dn[g] = d >= 0 ? (int32_t)c.gid[d] : -1;
  if (o.dbg_clean_up) o.dbg_clean_up[g] = cu >= 0 ? (int32_t)c.gid[cu] : -1;
  if (o.dbg_clean_dn) o.dbg_clean_dn[g] = cd >= 0 ? (int32_t)c.gid[cd] : -1;
  if (o.dbg_start_hits && o.dbg_n_start_hits && cu >= 0 && cd < 0)
    o.dbg_start_hits[atomicAdd(o.dbg_n_start_hits, 1u)] = g;
}

__global__ void k_debug_tracklets(const Ctx c) {
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t n_trk = *c.n_tracklets;
  const tpc_tracks& o = c.out;
  if (t >= n_trk || t >= o.dbg_tracklet_capacity) return;
  const uint32_t T = c.max_tracklets;
  const int n_rows = c.n_rows;
  if (o.dbg_tracklet_start) o.dbg_tracklet_start[t] = c.gid[c.trk_start[t]];
  if (o.dbg_tracklet_nhits) o.dbg_tracklet_nhits[t] = (uint32_t)c.trk_rows[2u * T + t];
  if (o.dbg_tracklet_par)
    for (int j = 0; j < 5; ++j) o.dbg_tracklet_par[(size_t)t * 5 + j] = c.trk_state[(size_t)(1 + j) * T + t];
  if (o.dbg_tracklet_map) {
    const int first_row = c.trk_rows[t], last_row = c.trk_rows[T + t];
    for (int r = 0; r < n_rows; ++r) {
      int32_t m = -1;
      if (r >= first_row && r <= last_row) m = c.trk_map[map_index(t, r, n_rows)];
      o.dbg_tracklet_map[(size_t)t * n_rows + r] = m >= 0 ? (int32_t)c.gid[m] : -1;
    }
  }
}

}  // namespace tpc
