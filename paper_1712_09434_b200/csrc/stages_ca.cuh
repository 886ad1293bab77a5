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
constexpr int kGridThreads = 128;

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
  __shared__ uint32_t s_cnt[kMaxBinsPerRow + 1];
  __shared__ uint32_t s_part[kGridThreads];
  __shared__ float s_box[4][kGridThreads / 32];
  const uint32_t tr = blockIdx.x;
  const uint32_t lo = c.row_off[tr], hi = c.row_off[tr + 1], n = hi - lo;
  const int tid = threadIdx.x;
  // bounding box of the row's clusters
  const float kInf = __int_as_float(0x7f800000);
  float ylo = kInf, yhi = -kInf, zlo = kInf, zhi = -kInf;
  for (uint32_t i = lo + tid; i < hi; i += kGridThreads) {
    // non-finite coordinates (outside the contract, R27) must not make the box infinite: +-Inf is clamped, NaN
    // is dropped by fminf/fmaxf; such a cluster lands in an edge bin and never passes an exact window test
    const float y = fminf(fmaxf(c.y[i], -kCoordClamp), kCoordClamp), z = fminf(fmaxf(c.z[i], -kCoordClamp), kCoordClamp);
    ylo = fminf(ylo, y); yhi = fmaxf(yhi, y); zlo = fminf(zlo, z); zhi = fmaxf(zhi, z);
  }
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
  if (tid == 0) c.rowinfo[tr] = g;
  for (int b = tid; b <= nb; b += kGridThreads) s_cnt[b] = 0u;
  __syncthreads();
  for (uint32_t i = lo + tid; i < hi; i += kGridThreads) {
    const int bin = bin_coord(c.z[i], z0, g.inv, g_nz) * g_ny + bin_coord(c.y[i], y0, g.inv, g_ny);
    atomicAdd(&s_cnt[bin], 1u);
  }
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
  for (int b = tid; b < nb; b += kGridThreads) gbins[b] = lo + s_cnt[b];
  if (tid == 0) gbins[nb] = hi;
  __syncthreads();
  // scatter; s_cnt[b] becomes the running end of bin b
  for (uint32_t i = lo + tid; i < hi; i += kGridThreads) {
    const float y = c.y[i], z = c.z[i];
    const int bin = bin_coord(z, z0, g.inv, g_nz) * g_ny + bin_coord(y, y0, g.inv, g_ny);
    const uint32_t pos = lo + atomicAdd(&s_cnt[bin], 1u);
    c.yz[pos] = make_float2(y, z);
    c.gid[pos] = i;
  }
  __syncthreads();
  // order every bin by gid.  Bins hold about half a cluster; those with 2..4 are sorted in registers - their gids
  // are read together, ordered by a 5-exchange network, and (y,z) is re-read from the input by gid - so that a bin
  // costs one round of loads instead of a chain of them; larger bins take the insertion sort.
  for (int b = tid; b < nb; b += kGridThreads) {
    const uint32_t e = lo + s_cnt[b], s = lo + (b > 0 ? s_cnt[b - 1] : 0u);
    const uint32_t m = e - s;
    if (m < 2u) continue;
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
      continue;
    }
    for (uint32_t i = s + 1; i < e; ++i) {
      const uint32_t gi = c.gid[i];
      const float2 vi = c.yz[i];
      uint32_t j = i;
      while (j > s && c.gid[j - 1] > gi) { c.gid[j] = c.gid[j - 1]; c.yz[j] = c.yz[j - 1]; --j; }
      if (j != i) { c.gid[j] = gi; c.yz[j] = vi; }
    }
  }
  if (COUNT && tid == 0) {
    atomicAdd(&c.counters[CN_BINS], (unsigned long long)nb);
    atomicAdd(&c.counters[CN_CLUSTERS], (unsigned long long)n);
  }
}

// ---------------------------------------------------------------------------
// a3  neighbour cleaner (SPEC 4, C1): clean_up[h] = up[h] iff dn[up[h]] == h.
// One thread per cluster.
// ---------------------------------------------------------------------------
constexpr int kCleanThreads = 256;

__global__ void __launch_bounds__(kCleanThreads) k_clean(const Ctx c) {
  const uint32_t i = blockIdx.x * kCleanThreads + threadIdx.x;
  if (i >= c.n) return;
  const int32_t u = c.link_up[i];
  c.clean_up[i] = (u >= 0 && c.link_dn[u] == (int32_t)i) ? u : -1;
}

// ---------------------------------------------------------------------------
// a4  start hits (S1) whose chain has >= min_seed_hits hits (S2, S3), written
// in idx order as seed records (trk_seed).  Tile = kSeedThreads * kSeedItems idx.
// ---------------------------------------------------------------------------
constexpr int kSeedThreads = 256;
constexpr int kSeedItems = 4;
constexpr uint32_t kSeedTile = kSeedThreads * kSeedItems;

template <bool COUNT>
__global__ void __launch_bounds__(kSeedThreads) k_seeds(const Ctx c) {
  __shared__ uint32_t s_warp[33];
  __shared__ uint32_t s_tile;
  __shared__ unsigned long long s_prefix;
  if (threadIdx.x == 0) s_tile = atomicAdd(&c.tickets[0], 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t base = tile * kSeedTile + threadIdx.x * kSeedItems;
  uint32_t flags = 0u, n_s1 = 0u;
  int32_t h1s[kSeedItems], h2s[kSeedItems], h3s[kSeedItems];
  // the four cleaned up-links and raw down-links of this thread: one 16-byte load each (arrays are padded)
  int4 cu4 = make_int4(-1, -1, -1, -1), dn4 = make_int4(-1, -1, -1, -1);
  if (base < c.n) {
    cu4 = *reinterpret_cast<const int4*>(c.clean_up + base);
    dn4 = *reinterpret_cast<const int4*>(c.link_dn + base);
  }
  const int32_t cu[kSeedItems] = {cu4.x, cu4.y, cu4.z, cu4.w}, dn[kSeedItems] = {dn4.x, dn4.y, dn4.z, dn4.w};
#pragma unroll
  for (int k = 0; k < kSeedItems; ++k) {
    const uint32_t i = base + k;
    h1s[k] = -1; h2s[k] = -1; h3s[k] = -1;
    if (i >= c.n) continue;
    const int32_t h1 = cu[k];
    if (h1 < 0) continue;
    const int32_t d = dn[k];
    if (d >= 0 && c.link_up[d] == (int32_t)i) continue;  // clean_dn[i] >= 0 (C2): not a start hit
    if (COUNT) ++n_s1;
    const int32_t h2 = c.clean_up[h1];
    int32_t h = h2 >= 0 ? c.clean_up[h2] : -1;           // h3
    h1s[k] = h1; h2s[k] = h2; h3s[k] = h;
    int len = 2 + (h2 >= 0 ? 1 : 0) + (h >= 0 ? 1 : 0);  // S2: hits of the chain, counted up to min_seed_hits
    while (len < c.prm.min_seed_hits && h >= 0) {
      h = c.clean_up[h];
      if (h >= 0) ++len;
    }
    if (len >= c.prm.min_seed_hits) flags |= 1u << k;
  }
  uint32_t total;
  const uint32_t excl = block_exclusive_scan(__popc(flags), s_warp, &total);
  if (threadIdx.x < 32) {
    const unsigned long long p = lookback_exclusive(c.scan_seed, tile, (unsigned long long)total);
    if (threadIdx.x == 0) s_prefix = p;
  }
  __syncthreads();
  const unsigned long long prefix = s_prefix;
  uint32_t pos = (uint32_t)prefix + excl;
#pragma unroll
  for (int k = 0; k < kSeedItems; ++k) {
    if (!(flags & (1u << k))) continue;
    if (pos < c.max_tracklets) {
      const uint32_t h0 = base + k, h1 = (uint32_t)h1s[k];
      const uint32_t tr0 = find_tr(c, h0);
      const float2 p0 = c.yz[h0], p1 = c.yz[h1];
      const float2 p2 = h2s[k] >= 0 ? c.yz[h2s[k]] : make_float2(0.0f, 0.0f);
      uint4* rec = c.trk_seed + (size_t)pos * kSeedU4;
      rec[0] = make_uint4(h0, tr0, h1, (uint32_t)h2s[k]);
      rec[1] = make_uint4(__float_as_uint(p0.x), __float_as_uint(p0.y), __float_as_uint(p1.x), __float_as_uint(p1.y));
      rec[2] = make_uint4(__float_as_uint(p2.x), __float_as_uint(p2.y), c.gid[h0], (uint32_t)h3s[k]);
    }
    ++pos;
  }
  if (threadIdx.x == 0 && tile == gridDim.x - 1) {  // the last tile knows the total
    const unsigned long long all = prefix + total;
    if (all > c.max_tracklets) atomicOr(&c.out.header[2], TPC_STATUS_TRACKLET_OVERFLOW);
    const uint32_t built = (uint32_t)(all > c.max_tracklets ? c.max_tracklets : all);
    *c.n_tracklets = built;
    c.out.header[3] = built;
    if (COUNT) atomicAdd(&c.counters[CN_TRACKLETS_BUILT], (unsigned long long)built);
  }
  if (COUNT && n_s1) atomicAdd(&c.counters[CN_START_HITS], (unsigned long long)n_s1);
}

}  // namespace tpc
