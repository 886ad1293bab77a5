// Cellular-Automaton stages of the TPC sector tracker (PAPER.md L121, L123:
// "1 GPU thread handles 1 cluster" in the CA phase):
//   a1 k_grid_build   - per (task,row) counting sort of the clusters into a y-z grid (SPEC 2)
//   (a2, the neighbour finder, is in stage_neighbours.cuh)
//   a3 k_clean        - keep a link iff reciprocated (SPEC 4, C1; C2 is evaluated where needed)
//   a4 k_seeds        - start hits with a chain of >= min_seed_hits, compacted in idx order (S1..S3)
#pragma once
#include "device_common.cuh"

namespace tpc {

// ---------------------------------------------------------------------------
// a1  grid build.  One block per (task,row).  The grid is acceleration only
// (SPEC 2): every later search applies the exact test to a superset, so the bin
// size and the extent of the grid (the bounding box of the row's clusters) are this implementation's own choice.  The clusters of a row are
// rewritten as float2 (y,z) in bin order ("idx" order) with idx -> gid beside;
// inside a bin they are ordered by gid so that idx order, and with it the order
// of start hits, tracklets and output tracks, is the same on every run.
// ---------------------------------------------------------------------------
#ifndef TPC_GRID_THREADS
#define TPC_GRID_THREADS 96  // with 5 clusters per thread in registers: 64: 0.62 ms, 96: 0.54, 128: 0.61, 160 (3 kept): 0.59, 192: 0.64 (a row of a central event: 444 clusters)
#endif
constexpr int kGridThreads = TPC_GRID_THREADS;
#ifndef TPC_GRID_KEEP
#define TPC_GRID_KEEP 5
#endif
constexpr int kGridKeep = TPC_GRID_KEEP;  // clusters per thread kept in registers between the passes of k_grid_build

// Grid of a row with n clusters inside the box [ylo, yhi] x [zlo, zhi]: kBinsPerCluster bins per cluster.
__device__ __forceinline__ RowInfo make_row_info(const Ctx& c, uint32_t tr, uint32_t lo, uint32_t n, float ylo,
                                                 float yhi, float zlo, float zhi) {
  const float W = fmaxf(yhi - ylo, 0.0f), L = fmaxf(zhi - zlo, 0.0f);
  float B = sqrtf((W * L) / (float)(kBinsPerCluster * (n > 0u ? n : 1u)));
  B = fminf(fmaxf(B, c.prm.grid_bin_min), c.prm.grid_bin_max);
  RowInfo g;
  int ny = 1, nz = 1;
  // The box is finite (the caller clamps every coordinate to +-kCoordClamp), so a few dozen coarsening steps
  // always end; the iteration bound only guards against parameters that make B non-finite: then one bin.
  for (int it = 0; it < 96; ++it) {
    g.inv = 1.0f / B;
    ny = (int)fminf(fmaxf(W * g.inv, 0.0f), 65000.0f) + 1;
    nz = (int)fminf(fmaxf(L * g.inv, 0.0f), 65000.0f) + 1;
    const long long nb = (long long)ny * nz;
    if (nb + 1 <= (long long)kBinsPerCluster * n + kBinPad && nb <= (long long)kMaxBinsPerRow) break;
    B = B * 1.25f;  // too many bins for the slot of this row: coarser grid
    if (it == 95) { ny = 1; nz = 1; g.inv = 0.0f; }
  }
  g.y0 = ylo; g.z0 = zlo;
  g.ny_nz = (uint32_t)ny | ((uint32_t)nz << 16);
  g.bins_off = bins_base(c, tr, lo);
  g.row_lo = lo;
  g.pad0 = 0u; g.pad1 = 0u;
  return g;
}

template <bool COUNT>
__global__ void __launch_bounds__(kGridThreads) k_grid_build(const Ctx c) {
  __shared__ __align__(16) uint32_t s_cnt[kMaxBinsPerRow + 4];  // + 1 end entry, padded to whole 16-byte groups
  __shared__ uint32_t s_part[kGridThreads];
  __shared__ float s_box[4][kGridThreads / 32];
  __shared__ uint32_t s_nlist;  // bins with two clusters or more, listed for the sort
  const uint32_t tr = blockIdx.x;
  const uint32_t lo = c.row_off[tr], hi = c.row_off[tr + 1], n = hi - lo;
  const int tid = threadIdx.x;
  // bounding box of the row's clusters
  const float kInf = __int_as_float(0x7f800000);
  float ylo = kInf, yhi = -kInf, zlo = kInf, zhi = -kInf;
  // The first kGridKeep clusters of a thread (all of them in a row of a central event) stay in registers for the
  // three passes over the row; what is beyond them is read again.
  float ky[kGridKeep], kz[kGridKeep];
#pragma unroll
  for (int k = 0; k < kGridKeep; ++k) {
    const uint32_t i = lo + (uint32_t)(tid + k * kGridThreads);
    ky[k] = i < hi ? c.y[i] : 0.0f;
    kz[k] = i < hi ? c.z[i] : 0.0f;
  }
  auto for_clusters = [&](auto&& body) {  // body(i, y, z) for the clusters lo + tid, lo + tid + kGridThreads, ...
#pragma unroll
    for (int k = 0; k < kGridKeep; ++k) {
      const uint32_t i = lo + (uint32_t)(tid + k * kGridThreads);
      if (i < hi) body(i, ky[k], kz[k]);
    }
    for (uint32_t i = lo + (uint32_t)(tid + kGridKeep * kGridThreads); i < hi; i += kGridThreads) body(i, c.y[i], c.z[i]);
  };
  for_clusters([&](uint32_t, float yr, float zr) {
    // non-finite coordinates (outside the contract, R27) must not make the box infinite: +-Inf is clamped, NaN
    // is dropped by fminf/fmaxf; such a cluster lands in an edge bin and never passes an exact window test
    const float y = fminf(fmaxf(yr, -kCoordClamp), kCoordClamp), z = fminf(fmaxf(zr, -kCoordClamp), kCoordClamp);
    ylo = fminf(ylo, y); yhi = fmaxf(yhi, y); zlo = fminf(zlo, z); zhi = fmaxf(zhi, z);
  });
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ylo = fminf(ylo, __shfl_xor_sync(0xffffffffu, ylo, o)); yhi = fmaxf(yhi, __shfl_xor_sync(0xffffffffu, yhi, o));
    zlo = fminf(zlo, __shfl_xor_sync(0xffffffffu, zlo, o)); zhi = fmaxf(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
  }
  if ((tid & 31) == 0) { s_box[0][tid >> 5] = ylo; s_box[1][tid >> 5] = yhi; s_box[2][tid >> 5] = zlo; s_box[3][tid >> 5] = zhi; }
  __syncthreads();
#pragma unroll
  for (int w = 0; w < kGridThreads / 32; ++w) {
    ylo = fminf(ylo, s_box[0][w]); yhi = fmaxf(yhi, s_box[1][w]); zlo = fminf(zlo, s_box[2][w]); zhi = fmaxf(zhi, s_box[3][w]);
  }
  if (n == 0u || !(ylo <= yhi) || !(zlo <= zhi)) { ylo = yhi = zlo = zhi = 0.0f; }  // empty row, or NaN only
  const RowInfo g = make_row_info(c, tr, lo, n, ylo, yhi, zlo, zhi);
  const int g_ny = info_ny(g), g_nz = info_nz(g);
  const int nb = g_ny * g_nz;
  const float y0 = g.y0, z0 = g.z0;
  if (tid == 0) {
    c.rowinfo[tr] = g;
    // the row that holds the first idx of every tile of the start-hit finder (a4)
    for (uint32_t k = (lo + kSeedTileIdx - 1u) / kSeedTileIdx; k * kSeedTileIdx < hi; ++k) c.tile_tr[k] = tr;
  }
  for (int b = 4 * tid; b <= nb; b += 4 * kGridThreads)  // 16 bytes per store (entries behind nb are scratch)
    *reinterpret_cast<uint4*>(&s_cnt[b]) = make_uint4(0u, 0u, 0u, 0u);
  if (tid == 0) s_nlist = 0u;
  __syncthreads();
  for_clusters([&](uint32_t, float y, float z) {
    const int bin = bin_coord(z, z0, g.inv, g_nz) * g_ny + bin_coord(y, y0, g.inv, g_ny);
    atomicAdd(&s_cnt[bin], 1u);
  });
  __syncthreads();
  // exclusive scan of s_cnt[0..nb): each thread owns a contiguous chunk
  const int chunk = (nb + kGridThreads - 1) / kGridThreads;
  const int b0 = min(tid * chunk, nb), b1 = min(b0 + chunk, nb);
  uint32_t sum = 0u;
  for (int b = b0; b < b1; ++b) sum += s_cnt[b];
  s_part[tid] = sum;
  __syncthreads();
  if (tid < 32) {  // scan of the 128 partial sums by one warp, 4 per lane
    uint32_t v[kGridThreads / 32], tot = 0u;
#pragma unroll
    for (int k = 0; k < kGridThreads / 32; ++k) { v[k] = s_part[tid * (kGridThreads / 32) + k]; tot += v[k]; }
    uint32_t incl = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
      if (tid >= o) incl += t;
    }
    uint32_t run = incl - tot;
#pragma unroll
    for (int k = 0; k < kGridThreads / 32; ++k) { s_part[tid * (kGridThreads / 32) + k] = run; run += v[k]; }
  }
  __syncthreads();
  uint32_t run = s_part[tid];
  for (int b = b0; b < b1; ++b) { const uint32_t t = s_cnt[b]; s_cnt[b] = run; run += t; }
  __syncthreads();
  uint32_t* gbins = c.bins + g.bins_off;
  // bins_off is even (kBinsPerCluster * row_lo + tr * kBinPad): two entries per 8-byte store
  static_assert(kBinsPerCluster % 2u == 0u && kBinPad % 2u == 0u, "8-byte stores of the bin table need an even bins_off");
  for (int b = 2 * tid; b < nb; b += 2 * kGridThreads) {
    const uint2 v = *reinterpret_cast<const uint2*>(&s_cnt[b]);
    if (b + 1 < nb) *reinterpret_cast<uint2*>(&gbins[b]) = make_uint2(lo + v.x, lo + v.y);
    else gbins[b] = lo + v.x;
  }
  if (tid == 0) gbins[nb] = hi;
  __syncthreads();
  // scatter; s_cnt[b] becomes the running end of bin b
  for_clusters([&](uint32_t i, float y, float z) {
    const int bin = bin_coord(z, z0, g.inv, g_nz) * g_ny + bin_coord(y, y0, g.inv, g_ny);
    const uint32_t pos = lo + atomicAdd(&s_cnt[bin], 1u);
    c.yz[pos] = make_float2(y, z);
    c.gid[pos] = i;
  });
  __syncthreads();
  // order every bin by gid.  Bins hold about half a cluster; those with 2..4 are sorted in registers - their gids
  // are read together, ordered by a 5-exchange network, and (y,z) is re-read from the input by gid - so that a bin
  // costs one round of loads instead of a chain of them; larger bins take the insertion sort.  One bin in eleven
  // needs it, so the bins are listed first (in the unused tail of s_cnt) and the threads sort the listed bins side by
  // side instead of each thread meeting one now and then among its own bins (4.6 of 32 lanes).
  auto sort_bin = [&](int b) {
    const uint32_t e = lo + s_cnt[b], s = lo + (b > 0 ? s_cnt[b - 1] : 0u);
    const uint32_t m = e - s;
    if (m <= 4u) {
      const uint32_t o0 = c.gid[s], o1 = c.gid[s + 1], o2 = m > 2u ? c.gid[s + 2] : 0xFFFFFFFFu;
      const uint32_t o3 = m > 3u ? c.gid[s + 3] : 0xFFFFFFFFu;
      uint32_t g0 = o0, g1 = o1, g2 = o2, g3 = o3, t;
#define TPC_CSWAP(a, b) t = min(a, b); b = max(a, b); a = t;
      TPC_CSWAP(g0, g1) TPC_CSWAP(g2, g3) TPC_CSWAP(g0, g2) TPC_CSWAP(g1, g3) TPC_CSWAP(g1, g2)
#undef TPC_CSWAP
      if (g0 != o0) { c.gid[s] = g0; c.yz[s] = make_float2(c.y[g0], c.z[g0]); }
      if (g1 != o1) { c.gid[s + 1] = g1; c.yz[s + 1] = make_float2(c.y[g1], c.z[g1]); }
      if (g2 != o2) { c.gid[s + 2] = g2; c.yz[s + 2] = make_float2(c.y[g2], c.z[g2]); }
      if (g3 != o3) { c.gid[s + 3] = g3; c.yz[s + 3] = make_float2(c.y[g3], c.z[g3]); }
      return;
    }
    for (uint32_t i = s + 1; i < e; ++i) {
      const uint32_t gi = c.gid[i];
      const float2 vi = c.yz[i];
      uint32_t j = i;
      while (j > s && c.gid[j - 1] > gi) { c.gid[j] = c.gid[j - 1]; c.yz[j] = c.yz[j - 1]; --j; }
      if (j != i) { c.gid[j] = gi; c.yz[j] = vi; }
    }
  };
  uint32_t* s_list = s_cnt + nb + 1;                     // s_cnt has kMaxBinsPerRow + 1 entries, nb + 1 are in use
  const uint32_t list_cap = kMaxBinsPerRow - (uint32_t)nb;
  for (int b = tid; b < nb; b += kGridThreads) {
    if (s_cnt[b] - (b > 0 ? s_cnt[b - 1] : 0u) < 2u) continue;
    const uint32_t k = atomicAdd(&s_nlist, 1u);
    if (k < list_cap) s_list[k] = (uint32_t)b;
    else sort_bin(b);                                    // no room in the list (a row close to kMaxBinsPerRow bins)
  }
  __syncthreads();
  for (uint32_t k = (uint32_t)tid, nl = min(s_nlist, list_cap); k < nl; k += kGridThreads) sort_bin((int)s_list[k]);
  if (COUNT && tid == 0) {
    atomicAdd(&c.counters[CN_BINS], (unsigned long long)nb);
    atomicAdd(&c.counters[CN_CLUSTERS], (unsigned long long)n);
  }
}

// ---------------------------------------------------------------------------
// a3  neighbour cleaner (SPEC 4, C1): clean_up[h] = up[h] iff dn[up[h]] == h.
// Four clusters per thread: one 16-byte load of the up-links, the four gathers of their down-links in
// flight together, one 16-byte store (the arrays are padded to whole groups, Carve).
// ---------------------------------------------------------------------------
constexpr int kCleanThreads = 256;
constexpr uint32_t kCleanItems = 4;

__global__ void __launch_bounds__(kCleanThreads) k_clean(const Ctx c) {
  const uint32_t i = (blockIdx.x * kCleanThreads + threadIdx.x) * kCleanItems;
  if (i >= c.n) return;
  const int4 u = *reinterpret_cast<const int4*>(c.link_up + i);
  const int32_t uu[4] = {u.x, u.y, u.z, u.w};
  int32_t back[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) back[k] = (i + (uint32_t)k < c.n && uu[k] >= 0) ? c.link_dn[uu[k]] : -2;
  int32_t r[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) r[k] = back[k] == (int32_t)(i + (uint32_t)k) ? uu[k] : -1;
  *reinterpret_cast<int4*>(c.clean_up + i) = make_int4(r[0], r[1], r[2], r[3]);
}

// ---------------------------------------------------------------------------
// a4  start hits (S1) whose chain has >= min_seed_hits hits (S2, S3), written
// in idx order as seed records (trk_seed).  Tile = kSeedThreads * kSeedItems idx.
// Three steps per tile: every thread tests its kSeedItems clusters for S1 (16-byte loads and the
// link gathers of C2 in flight together); the tile's start hits (about one cluster in twenty) are
// compacted in order into shared memory and each is walked by a thread of its own (S2: the four or
// five dependent link loads of a chain run side by side instead of up to four chains per thread one
// after the other); those with a long enough chain are compacted again, the tile takes its place in
// the output (chained scan with decoupled look-back), and the threads write the seed records.
// ---------------------------------------------------------------------------
#ifndef TPC_SEED_THREADS
#define TPC_SEED_THREADS 256
#endif
constexpr int kSeedThreads = TPC_SEED_THREADS;
constexpr int kSeedItems = TPC_SEED_ITEMS;  // clusters per thread: whole 16-byte groups
static_assert(kSeedItems % 4 == 0, "k_seeds reads the links in 16-byte groups");
#ifndef TPC_SEED_MINBLOCKS
#define TPC_SEED_MINBLOCKS 7  // 7 x 28.5 KB of shared memory per SM; (threads, items, blocks): (512, 4, 4) 0.43 ms, (256, 8, 7) 0.35 - more idx in flight per SM
#endif
constexpr uint32_t kSeedTile = kSeedThreads * kSeedItems;
static_assert(kSeedTile == kSeedTileIdx, "k_grid_build notes the row of every tile start");
constexpr int kSeedRows = 96;  // row offsets of the tile kept in shared memory (a tile of a central event spans 3 rows)

template <bool COUNT>
__global__ void __launch_bounds__(kSeedThreads, TPC_SEED_MINBLOCKS) k_seeds(const Ctx c) {
  __shared__ uint32_t s_warp[33];
  __shared__ uint32_t s_tile, s_tr;
  __shared__ unsigned long long s_prefix;
  __shared__ uint16_t s_cand[kSeedTile];        // start hits of the tile (idx - tile base), in idx order
  __shared__ int32_t s_h[3][kSeedTile];         // h1, h2, h3 of candidate j
  __shared__ uint32_t s_rowoff[kSeedRows + 1];  // row_off[s_tr + j]
  const int tid = (int)threadIdx.x;
  if (tid == 0) {
    s_tile = atomicAdd(&c.tickets[0], 1u);
    s_tr = c.tile_tr[s_tile];
  }
  __syncthreads();
  const uint32_t tile = s_tile, tile_base = tile * kSeedTile;
  const uint32_t tr_tile = s_tr;
  if (tid <= kSeedRows) s_rowoff[tid] = c.row_off[min(tr_tile + (uint32_t)tid, c.n_tr)];
  const uint32_t base = tile_base + (uint32_t)tid * kSeedItems;
  // S1: cleaned up-link present, cleaned down-link absent
  int32_t cu[kSeedItems], dn[kSeedItems];
#pragma unroll
  for (int g = 0; g < kSeedItems / 4; ++g) {
    int4 cu4 = make_int4(-1, -1, -1, -1), dn4 = make_int4(-1, -1, -1, -1);
    if (base < c.n) {  // arrays are padded to whole groups of kSeedItems
      cu4 = *reinterpret_cast<const int4*>(c.clean_up + base + 4 * g);
      dn4 = *reinterpret_cast<const int4*>(c.link_dn + base + 4 * g);
    }
    cu[4 * g] = cu4.x; cu[4 * g + 1] = cu4.y; cu[4 * g + 2] = cu4.z; cu[4 * g + 3] = cu4.w;
    dn[4 * g] = dn4.x; dn[4 * g + 1] = dn4.y; dn[4 * g + 2] = dn4.z; dn[4 * g + 3] = dn4.w;
  }
  int32_t back[kSeedItems];
#pragma unroll
  for (int k = 0; k < kSeedItems; ++k)  // (the padding behind the last cluster holds anything)
    back[k] = (base + k < c.n && cu[k] >= 0 && dn[k] >= 0) ? c.link_up[dn[k]] : -1;
  uint32_t s1 = 0u;
#pragma unroll
  for (int k = 0; k < kSeedItems; ++k)
    if (base + k < c.n && cu[k] >= 0 && !(dn[k] >= 0 && back[k] == (int32_t)(base + k))) s1 |= 1u << k;  // C2
  uint32_t n_cand;
  uint32_t at = block_exclusive_scan(__popc(s1), s_warp, &n_cand);
#pragma unroll
  for (int k = 0; k < kSeedItems; ++k)
    if (s1 & (1u << k)) {
      s_cand[at] = (uint16_t)(tid * kSeedItems + k);
      s_h[0][at] = cu[k];
      ++at;
    }
  __syncthreads();
  // S2, S3: one start hit per thread (loop: a tile can hold more start hits than threads)
  const int min_seed = c.prm.min_seed_hits;
  uint32_t keep = 0u;  // bit q: candidate tid + q*kSeedThreads has a long enough chain
  for (uint32_t j = (uint32_t)tid, q = 0u; j < n_cand; j += kSeedThreads, ++q) {
    const int32_t h1 = s_h[0][j];
    const int32_t h2 = c.clean_up[h1];
    int32_t h = h2 >= 0 ? c.clean_up[h2] : -1;  // h3
    s_h[1][j] = h2; s_h[2][j] = h;
    int len = 2 + (h2 >= 0 ? 1 : 0) + (h >= 0 ? 1 : 0);  // hits of the chain, counted up to min_seed_hits
    while (len < min_seed && h >= 0) {
      h = c.clean_up[h];
      if (h >= 0) ++len;
    }
    if (len >= min_seed) keep |= 1u << q;
  }
  // ordered compaction of the kept candidates: candidate order is j = tid + q*kSeedThreads, so the scan runs
  // once per q (one round for a tile with up to kSeedThreads start hits)
  uint32_t excl[kSeedItems], total = 0u;
  for (uint32_t q = 0u; q * kSeedThreads < n_cand || q == 0u; ++q) {
    uint32_t tq;
    excl[q] = total + block_exclusive_scan((keep >> q) & 1u, s_warp, &tq);
    total += tq;
  }
  if (tid < 32) {
    const unsigned long long p = lookback_exclusive(c.scan_seed, tile, (unsigned long long)total);
    if (tid == 0) s_prefix = p;
  }
  __syncthreads();
  const unsigned long long prefix = s_prefix;
  for (uint32_t j = (uint32_t)tid, q = 0u; j < n_cand; j += kSeedThreads, ++q) {
    if (!((keep >> q) & 1u)) continue;
    const unsigned long long pos = prefix + excl[q];
    if (pos >= c.max_tracklets) continue;
    const uint32_t h0 = tile_base + s_cand[j], h1 = (uint32_t)s_h[0][j];
    const int32_t h2 = s_h[1][j], h3 = s_h[2][j];
    uint32_t tr0;
    if (h0 < s_rowoff[kSeedRows]) {  // last of the staged rows with row_off <= h0
      int lo = 0, hi = kSeedRows;
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (s_rowoff[mid] <= h0) lo = mid; else hi = mid;
      }
      tr0 = tr_tile + (uint32_t)lo;
    } else {
      tr0 = find_tr(c, h0);
    }
    const float2 p0 = c.yz[h0], p1 = c.yz[h1];
    const float2 p2 = h2 >= 0 ? c.yz[h2] : make_float2(0.0f, 0.0f);
    const uint32_t g0 = c.gid[h0];
    uint4* rec = c.trk_seed + (size_t)pos * kSeedU4;
    order_note(c, (uint32_t)pos, tr0);  // queue order of the chain fit: from the row of the start hit upwards
    rec[0] = make_uint4(h0, tr0, h1, (uint32_t)h2);
    rec[1] = make_uint4(__float_as_uint(p0.x), __float_as_uint(p0.y), __float_as_uint(p1.x), __float_as_uint(p1.y));
    rec[2] = make_uint4(__float_as_uint(p2.x), __float_as_uint(p2.y), g0, (uint32_t)h3);
  }
  if (tid == 0 && tile == gridDim.x - 1) {  // the last tile knows the total
    const unsigned long long all = prefix + total;
    if (all > c.max_tracklets) atomicOr(&c.out.header[2], TPC_STATUS_TRACKLET_OVERFLOW);
    const uint32_t built = (uint32_t)(all > c.max_tracklets ? c.max_tracklets : all);
    *c.n_tracklets = built;
    c.out.header[3] = built;
    if (COUNT) atomicAdd(&c.counters[CN_TRACKLETS_BUILT], (unsigned long long)built);
  }
  if (COUNT) {
    const uint32_t n_s1 = __popc(s1);
    if (n_s1) atomicAdd(&c.counters[CN_START_HITS], (unsigned long long)n_s1);
  }
}

}  // namespace tpc
