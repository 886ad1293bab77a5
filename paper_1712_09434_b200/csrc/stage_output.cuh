// K7 ownership + a6 tracklet selector + a7 output compaction (docs/ARITH_SPEC.md sections 6 (K7) and 7, L1..L4),
// and the untimed debug kernels that translate internal idx to gid.
#pragma once
#include "device_common.cuh"
#include "stage_tracklet.cuh"

namespace tpc {

// ---------------------------------------------------------------------------
// K7 + L1: who owns a cluster.  owner[h] = max over the kept tracklets that hold h of
// (nHits, ~gid(h0)), and a tracklet keeps h iff it is that owner.  The ownership words never exist in
// global memory: the clusters are cut into chunks of kResolveChunk consecutive idx, one block per chunk
// holds the chunk's ownership words in shared memory.  Pass 1 walks the row maps of the tracklets of the
// task(s) the chunk lies in - only the rows the chunk covers - and takes atomicMax (shared-memory
// atomics) of
//     key = nHits << 53 | (2^27 - 1 - (gid(h0) - first gid of the task)) << 26 | tracklet index in the task
// which orders like (nHits, ~gid(h0)) because a start hit has one tracklet, and names the winner.
// Pass 2 walks the chunk's CLUSTERS: the winner's map entry gets kOwnedBit and its count of kept hits
// goes up by one.  After this kernel a tracklet keeps exactly the flagged entries of its map (L1).
// (Global 64-bit atomicMax per hit - 139 M of them on config 3, each a DRAM read-modify-write because
// the three or four tracklets that share a cluster end far apart in time - cost more than the whole
// down pass; shared memory takes that traffic away.)
// A task with 2^27 clusters or more (fifty times the whole config-3 batch in one sector) does not fit
// the key: its tracklets keep nothing and TPC_STATUS_TASK_TOO_LARGE is set.
// ---------------------------------------------------------------------------
#ifndef TPC_RESOLVE_THREADS
#define TPC_RESOLVE_THREADS 256
#endif
constexpr int kResolveThreads = TPC_RESOLVE_THREADS;
#ifndef TPC_RESOLVE_CHUNK
#define TPC_RESOLVE_CHUNK 4096
#endif
constexpr uint32_t kResolveChunk = TPC_RESOLVE_CHUNK;  // clusters per block: 32 KB of ownership words (2048: 1.05 ms, 4096: 0.84 ms, 8192: 1.00 ms)
#ifndef TPC_RESOLVE_BATCH
#define TPC_RESOLVE_BATCH 4
#endif
constexpr int kResolveBatch = TPC_RESOLVE_BATCH;  // (tracklet, four rows) groups a thread has in flight (2: 0.92, 4: 0.84, 8: 1.24 ms)
constexpr int kResolveRows = 512;                 // row offsets of the chunk kept in shared memory
constexpr uint32_t kKeyGidBits = 27, kKeyTrkBits = 26;

// first tracklet of every task: tracklets are in idx order of their start hits, so a task's are consecutive
__global__ void k_task_offsets(const Ctx c) {
  const uint32_t n_trk = *c.n_tracklets, n_rows = (uint32_t)c.n_rows;
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < n_trk; t += gridDim.x * blockDim.x) {
    const uint32_t task = c.trk_seed[(size_t)t * kSeedU4].y / n_rows;
    const uint32_t from = t ? c.trk_seed[(size_t)(t - 1u) * kSeedU4].y / n_rows + 1u : 0u;
    for (uint32_t k = from; k <= task; ++k) c.trk_task_off[k] = t;
    if (t == n_trk - 1u)
      for (uint32_t k = task + 1u; k <= c.n_tasks; ++k) c.trk_task_off[k] = n_trk;
  }
}

__global__ void __launch_bounds__(kResolveThreads) k_resolve(const Ctx c) {
  extern __shared__ unsigned long long s_owner[];  // [kResolveChunk]
  __shared__ uint32_t s_rowoff[kResolveRows + 1];
  const uint32_t i0 = blockIdx.x * kResolveChunk;
  const uint32_t i1 = min(i0 + kResolveChunk, c.n), span = i1 - i0;
  const int tid = (int)threadIdx.x, n_rows = c.n_rows;
  for (uint32_t i = tid; i < kResolveChunk; i += kResolveThreads) s_owner[i] = 0ull;
  // (task,row) of the first and of the last cluster of the chunk: k_grid_build noted the row of every
  // kSeedTileIdx-th idx (Ctx::tile_tr), so the last one is searched for among the few rows up to the next chunk's first
  static_assert(kResolveChunk % kSeedTileIdx == 0u, "Ctx::tile_tr holds the row of every chunk start");
  const uint32_t tr_a = c.tile_tr[i0 / kSeedTileIdx];
  uint32_t tr_b;
  {
    uint32_t lo = tr_a, hi = i1 < c.n ? c.tile_tr[i1 / kSeedTileIdx] + 1u : c.n_tr;  // row_off[lo] <= i1 - 1 < row_off[hi]
    while (hi - lo > 1u) {
      const uint32_t mid = (lo + hi) >> 1;
      if (c.row_off[mid] <= i1 - 1u) lo = mid; else hi = mid;
    }
    tr_b = lo;
  }
  const uint32_t task_a = tr_a / (uint32_t)n_rows, task_b = tr_b / (uint32_t)n_rows;
  const bool rows_staged = tr_b - tr_a < (uint32_t)kResolveRows;
  if (rows_staged)
    for (uint32_t j = tid; j <= tr_b - tr_a + 1u; j += kResolveThreads) s_rowoff[j] = c.row_off[tr_a + j];
  const int min_hits = c.prm.min_track_hits;
  const size_t stride = map_stride(n_rows);
  __syncthreads();
  // pass 1 (K7): for every tracklet of every task of the chunk, the rows the chunk covers, read four rows at a time
  // (16-byte groups of the row map: a map row starts at a multiple of 640 bytes); the (tracklet, group) pairs are
  // taken group fastest, thread tid the pairs tid, tid + 256, ...; (tt, gg) is stepped without a division
  for (uint32_t k = task_a; k <= task_b; ++k) {
    const uint32_t t0 = c.trk_task_off[k], nt = c.trk_task_off[k + 1u] - t0;
    const uint32_t gid_lo = c.row_off[k * (uint32_t)n_rows], gid_hi = c.row_off[(k + 1u) * (uint32_t)n_rows];
    if (gid_hi - gid_lo >= (1u << kKeyGidBits)) {
      if (tid == 0) atomicOr(&c.out.header[2], TPC_STATUS_TASK_TOO_LARGE);
      continue;
    }
    const uint32_t ra = k == task_a ? tr_a - k * (uint32_t)n_rows : 0u;
    const uint32_t rb = k == task_b ? tr_b - k * (uint32_t)n_rows : (uint32_t)n_rows - 1u;
    const uint32_t g0 = ra >> 2, G = (rb >> 2) - g0 + 1u, step_t = kResolveThreads / G, step_g = kResolveThreads % G;
    uint32_t tt = (uint32_t)tid / G, gg = (uint32_t)tid % G;
    while (__any_sync(0xffffffffu, tt < nt)) {
      uint4 m[kResolveBatch], e[kResolveBatch];
      uint32_t ts[kResolveBatch], rs[kResolveBatch];
#pragma unroll
      for (int j = 0; j < kResolveBatch; ++j) {  // meta and four map entries together (entries outside the
        ts[j] = tt; rs[j] = 4u * (g0 + gg);      // tracklet's rows are read and ignored)
        const bool in = tt < nt;
        m[j] = in ? __ldg(&c.trk_meta[t0 + tt]) : make_uint4(0u, 0u, 0u, 0u);
        e[j] = in ? *reinterpret_cast<const uint4*>(c.trk_hits + (size_t)(t0 + tt) * stride + rs[j])
                  : make_uint4(kNoHit, kNoHit, kNoHit, kNoHit);
        tt += step_t; gg += step_g;
        if (gg >= G) { gg -= G; ++tt; }
      }
#pragma unroll
      for (int j = 0; j < kResolveBatch; ++j) {
        if ((int)m[j].x < min_hits) continue;
        const uint32_t first = max(m[j].y & 0xFFFFu, ra), last = min(m[j].y >> 16, rb);
        const unsigned long long key = ((unsigned long long)m[j].x << (kKeyGidBits + kKeyTrkBits)) |
                                       ((unsigned long long)(((1u << kKeyGidBits) - 1u) - (m[j].z - gid_lo)) << kKeyTrkBits) |
                                       (unsigned long long)ts[j];
        const uint32_t idx[4] = {e[j].x, e[j].y, e[j].z, e[j].w};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const uint32_t r = rs[j] + (uint32_t)q, off = idx[q] - i0;  // idx < i0 wraps to a large number
          // (the 64-bit shared-memory atomicMax is a compare-and-swap loop: a claim that cannot win skips it)
          if (r >= first && r <= last && idx[q] != kNoHit && off < span && s_owner[off] < key) atomicMax(&s_owner[off], key);
        }
      }
    }
  }
  __syncthreads();
  // pass 2 (L1): every owned cluster of the chunk marks its entry in the winner's map; row by row, so that the
  // (task,row) of a cluster is known without a search
  for (uint32_t tr = tr_a; tr <= tr_b; ++tr) {
    const uint32_t r_lo = rows_staged ? s_rowoff[tr - tr_a] : c.row_off[tr];
    const uint32_t r_hi = rows_staged ? s_rowoff[tr - tr_a + 1u] : c.row_off[tr + 1u];
    const uint32_t a = max(r_lo, i0), b = min(r_hi, i1);
    if (a >= b) continue;
    const uint32_t task = tr / (uint32_t)n_rows, row = tr - task * (uint32_t)n_rows;
    const uint32_t t_first = c.trk_task_off[task];
    for (uint32_t h = a + (uint32_t)tid; h < b; h += kResolveThreads) {
      const unsigned long long key = s_owner[h - i0];
      if (key == 0ull) continue;
      const uint32_t t = t_first + (uint32_t)(key & ((1ull << kKeyTrkBits) - 1ull));
      c.trk_hits[(size_t)t * stride + row] = h | kOwnedBit;
      atomicAdd(&c.trk_kept[t], 1u);
    }
  }
}

#ifndef TPC_OUT_THREADS
#define TPC_OUT_THREADS 128
#endif
constexpr int kOutThreads = TPC_OUT_THREADS;  // = tracklets per tile; 4 warps x 32 tracklets
constexpr int kOutChunks = 5;     // 32-row chunks of a row map read per round (159 rows = 5 chunks)

// a6 (L2) + a7.  One tile = 128 consecutive tracklets; k_resolve has counted the hits every tracklet keeps
// (L1) and flagged exactly those in its row map.  The tile takes its place in the output with an ordered
// chained scan over (tracks, hits) packed as tracks<<32 | hits; then every warp writes its surviving
// tracks one by one - the record as SoA columns and the kept hits as gids in ascending row order (L3).
// Output order = tracklet order.
__global__ void __launch_bounds__(kOutThreads) k_select_output(const Ctx c) {
  __shared__ uint32_t s_warp[33];
  __shared__ uint32_t s_tile;
  __shared__ unsigned long long s_prefix;
  constexpr unsigned FULL = 0xffffffffu;
  const uint32_t n_trk = *c.n_tracklets;
  const uint32_t last_tile = n_trk > 0u ? (n_trk - 1u) / kOutThreads : 0u;
  // The host does not know how many tracklets were built, only their bound: it launches a fixed number of
  // blocks and every block takes tiles by ticket until they run out.  A tile only waits (look-back) for tiles
  // with smaller tickets, which are held by running blocks.
  for (;;) {
  __syncthreads();  // s_tile, s_prefix, s_warp of the previous tile are no longer read
  if (threadIdx.x == 0) s_tile = atomicAdd(&c.tickets[1], 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  if (tile > last_tile) return;
  const int n_rows = c.n_rows;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t t_warp = tile * kOutThreads + warp * 32;
  const int min_hits = c.prm.min_track_hits;
  // lane j holds what it needs of tracklet t_warp + j
  int my_first = 0, my_last = -1;
  uint32_t my_kept = 0u;
  if (t_warp + lane < n_trk) {
    const uint4 m = __ldg(&c.trk_meta[t_warp + lane]);
    my_first = (int)(m.y & 0xFFFFu); my_last = (int)(m.y >> 16);
    my_kept = c.trk_kept[t_warp + lane];
  }
  const bool is_track = my_kept >= (uint32_t)min_hits && my_kept > 0u;  // L2
  const uint32_t my_hits = is_track ? my_kept : 0u;
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
  const uint32_t my_slot = (uint32_t)(prefix >> 32) + ex_tracks;
  const uint32_t my_hb = (uint32_t)(prefix & 0xFFFFFFFFull) + ex_hits;
  const tpc_tracks& o = c.out;
  const size_t cap = o.track_capacity;
  unsigned status = 0u;
  const unsigned tracks_here = __ballot_sync(FULL, is_track);
  // The warp writes its tracks one after the other; what the NEXT track needs first - its record and the first
  // kOutChunks x 32 rows of its map - is requested before the current one's gid gathers and stores, so a track costs
  // one round trip of latency instead of two.
  float v_nx = 0.0f;
  uint32_t e_nx[kOutChunks];
  auto request = [&](int j) {  // loads of track t_warp + j into v_nx / e_nx
    const uint32_t t = t_warp + (uint32_t)j;
    const int first = __shfl_sync(FULL, my_first, j), last = __shfl_sync(FULL, my_last, j);
    v_nx = lane < 28 ? reinterpret_cast<const float*>(c.trk_rec + (size_t)t * kRecFloat4)[lane] : 0.0f;
    const uint32_t* map = c.trk_hits + (size_t)t * map_stride(n_rows);
#pragma unroll
    for (int q = 0; q < kOutChunks; ++q) {
      const int r = first + 32 * q + lane;
      e_nx[q] = r <= last ? map[r] : kNoHit;
    }
  };
  if (tracks_here) request(__ffs(tracks_here) - 1);
  for (unsigned rest = tracks_here; rest; rest &= rest - 1u) {
    const int j = __ffs(rest) - 1;
    const uint32_t t = t_warp + j;
    const uint32_t slot = __shfl_sync(FULL, my_slot, j), hb = __shfl_sync(FULL, my_hb, j);
    const uint32_t kept = __shfl_sync(FULL, my_kept, j);
    const int first = __shfl_sync(FULL, my_first, j), last = __shfl_sync(FULL, my_last, j);
    const float v = v_nx;  // record -> SoA columns: lanes 0..22 carry x, p[5], c[15], chi2, ndf
    uint32_t e_cur[kOutChunks];
#pragma unroll
    for (int q = 0; q < kOutChunks; ++q) e_cur[q] = e_nx[q];
    const unsigned after = rest & (rest - 1u);
    if (after) request(__ffs(after) - 1);
    if (slot >= o.track_capacity) { status |= TPC_STATUS_TRACK_OVERFLOW; continue; }
    if (lane == 0) {
      o.track_x[slot] = v;
      o.track_task[slot] = c.trk_seed[(size_t)t * kSeedU4].y / (uint32_t)n_rows;
      o.track_hit_begin[slot] = hb;
      o.track_nhits[slot] = kept;
    } else if (lane <= 5) o.track_par[(size_t)(lane - 1) * cap + slot] = v;
    else if (lane <= 20) o.track_cov[(size_t)(lane - 6) * cap + slot] = v;
    else if (lane == 21) o.track_chi2[slot] = v;
    else if (lane == 22) o.track_ndf[slot] = __float_as_int(v);
    if ((unsigned long long)hb + kept > (unsigned long long)o.hit_capacity) { status |= TPC_STATUS_HIT_OVERFLOW; continue; }
    const uint32_t* map = c.trk_hits + (size_t)t * map_stride(n_rows);
    uint32_t w = hb;
    int kept_first = -1, kept_last = -1;  // rows of the first and last kept hit (for the merger)
    // the map loads of kOutChunks chunks together, then their gid gathers, then the stores
    for (int rb0 = first; rb0 <= last; rb0 += 32 * kOutChunks) {
      uint32_t idx[kOutChunks], g[kOutChunks];
#pragma unroll
      for (int q = 0; q < kOutChunks; ++q) {  // kept (L1): the entry carries kOwnedBit
        const int r = rb0 + 32 * q + lane;
        const uint32_t e = rb0 == first ? e_cur[q] : (r <= last ? map[r] : kNoHit);
        idx[q] = (e != kNoHit && (e & kOwnedBit)) ? (e & ~kOwnedBit) : kNoHit;
      }
#pragma unroll
      for (int q = 0; q < kOutChunks; ++q) g[q] = idx[q] != kNoHit ? c.gid[idx[q]] : 0u;
#pragma unroll
      for (int q = 0; q < kOutChunks; ++q) {
        const unsigned mask = __ballot_sync(FULL, idx[q] != kNoHit);
        if (idx[q] != kNoHit) o.hit_cluster[w + __popc(mask & ((1u << lane) - 1u))] = g[q];
        w += __popc(mask);
        if (mask) {
          if (kept_first < 0) kept_first = rb0 + 32 * q + __ffs(mask) - 1;
          kept_last = rb0 + 32 * q + 31 - __clz(mask);
        }
      }
    }
    if (lane == 0) {
      c.out_trk[slot] = t;
      c.out_rows[slot] = (uint32_t)kept_first | ((uint32_t)kept_last << 16);
    }
  }
  if (status && lane == 0) atomicOr(&o.header[2], status);
  if (threadIdx.x == 0 && tile == last_tile) {  // the last tile knows the totals
    const unsigned long long all = prefix + agg;
    c.out.header[0] = (uint32_t)(all >> 32);
    c.out.header[1] = (uint32_t)(all & 0xFFFFFFFFull);
  }
  }  // next tile
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
  const int n_rows = c.n_rows;
  const float* rec = reinterpret_cast<const float*>(c.trk_rec + (size_t)t * kRecFloat4);
  const int n_hits = __float_as_int(rec[23]);
  if (o.dbg_tracklet_start) o.dbg_tracklet_start[t] = c.trk_seed[(size_t)t * kSeedU4 + 2].z;
  if (o.dbg_tracklet_nhits) o.dbg_tracklet_nhits[t] = (uint32_t)n_hits;
  if (o.dbg_tracklet_par)
    for (int j = 0; j < 5; ++j) o.dbg_tracklet_par[(size_t)t * 5 + j] = rec[1 + j];
  if (o.dbg_tracklet_map) {
    const int first = __float_as_int(rec[24]), last = __float_as_int(rec[25]);
    for (int r = 0; r < n_rows; ++r) {
      const uint32_t m = (r >= first && r <= last) ? c.trk_hits[(size_t)t * map_stride(n_rows) + r] : kNoHit;
      o.dbg_tracklet_map[(size_t)t * n_rows + r] = m != kNoHit ? (int32_t)c.gid[m] : -1;
    }
  }
}

}  // namespace tpc
