// Cellular-Automaton stages of the TPC sector tracker (PAPER.md L121, L123:
// "1 GPU thread handles 1 cluster" in the CA phase):
//   a1 k_grid_build   - per (task,row) counting sort of the clusters into a y-z grid (SPEC 2)
//   a2 k_neighbours   - best (up,down) pair by straight-line chi2 (SPEC 3, N1..N5)
//   a3 k_clean        - keep a link iff reciprocated (SPEC 4, C1; C2 is evaluated where needed)
//   a4 k_seeds        - start hits with a chain of >= min_seed_hits, compacted in idx order (S1..S3)
#pragma once
#include "device_common.cuh"

namespace tpc {

// ---------------------------------------------------------------------------
// a1  grid build.  One block per (task,row).  The grid is acceleration only
// (SPEC 2): every later search applies the exact test to a superset, so the bin
// size below is this implementation's own choice.  The clusters of a row are
// rewritten as float2 (y,z) in bin order ("idx" order) with idx -> gid beside;
// inside a bin they are ordered by gid so that idx order, and with it the order
// of start hits, tracklets and output tracks, is the same on every run.
// ---------------------------------------------------------------------------
constexpr int kGridThreads = 128;

__device__ __forceinline__ RowGrid make_row_grid(const Ctx& c, int row, uint32_t n) {
  const float W = 2.0f * c.ymax[row], L = c.z_max + 2.0f;
  float B = sqrtf((W * L) / (float)(n > 0u ? n : 1u));
  B = fminf(fmaxf(B, c.prm.grid_bin_min), c.prm.grid_bin_max);
  RowGrid g;
  while (true) {
    g.inv = 1.0f / B;
    g.ny = (int)(W * g.inv) + 1;
    g.nz = (int)(L * g.inv) + 1;
    const long long nb = (long long)g.ny * g.nz;
    if (nb + 1 <= (long long)n + kBinPad && nb <= (long long)kMaxBinsPerRow) break;
    B = B * 1.25f;  // too many bins for the slot of this row: coarser grid
  }
  g.pad = 0;
  return g;
}

template <bool COUNT>
__global__ void __launch_bounds__(kGridThreads) k_grid_build(const Ctx c) {
  __shared__ uint32_t s_cnt[kMaxBinsPerRow + 1];
  __shared__ uint32_t s_part[kGridThreads];
  const uint32_t tr = blockIdx.x;
  const int row = (int)(tr % (uint32_t)c.n_rows);
  const uint32_t task = tr / (uint32_t)c.n_rows;
  const uint32_t lo = c.row_off[tr], hi = c.row_off[tr + 1], n = hi - lo;
  const RowGrid g = make_row_grid(c, row, n);
  const int nb = g.ny * g.nz;
  const float y0 = -c.ymax[row], z0 = side_z0(c, task);
  const int tid = threadIdx.x;
  if (tid == 0) c.rowgrid[tr] = g;
  for (int b = tid; b <= nb; b += kGridThreads) s_cnt[b] = 0u;
  __syncthreads();
  for (uint32_t i = lo + tid; i < hi; i += kGridThreads) {
    const int bin = bin_coord(c.z[i], z0, g.inv, g.nz) * g.ny + bin_coord(c.y[i], y0, g.inv, g.ny);
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
  uint32_t* gbins = c.bins + bins_base(c, tr, lo);
  for (int b = tid; b < nb; b += kGridThreads) gbins[b] = lo + s_cnt[b];
  if (tid == 0) gbins[nb] = hi;
  __syncthreads();
  // scatter; s_cnt[b] becomes the running end of bin b
  for (uint32_t i = lo + tid; i < hi; i += kGridThreads) {
    const float y = c.y[i], z = c.z[i];
    const int bin = bin_coord(z, z0, g.inv, g.nz) * g.ny + bin_coord(y, y0, g.inv, g.ny);
    const uint32_t pos = lo + atomicAdd(&s_cnt[bin], 1u);
    c.yz[pos] = make_float2(y, z);
    c.gid[pos] = i;
  }
  __syncthreads();
  // order every bin by gid (bins hold about one cluster; insertion sort)
  for (int b = tid; b < nb; b += kGridThreads) {
    const uint32_t e = lo + s_cnt[b], s = lo + (b > 0 ? s_cnt[b - 1] : 0u);
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
// a2  neighbour finder (SPEC 3).  One block per (task,row); one thread per
// cluster of the row, in idx order so that the lanes of a warp look at the same
// few bins of rows r+1 and r-1.
// ---------------------------------------------------------------------------
constexpr int kNfThreads = 128;

struct Window {  // bin range of one search window in one row
  const uint32_t* bins;  // first bin of the row
  int ny, iy0, iy1, iz0, iz1;
};

__device__ __forceinline__ Window make_window(const Ctx& c, uint32_t tr, int row, float z0, float ylo, float yhi,
                                              float zlo, float zhi) {
  const RowGrid g = c.rowgrid[tr];
  const float y0 = -c.ymax[row];
  Window w;
  w.bins = c.bins + bins_base(c, tr, c.row_off[tr]);
  w.ny = g.ny;
  w.iy0 = bin_coord(ylo, y0, g.inv, g.ny);
  w.iy1 = bin_coord(yhi, y0, g.inv, g.ny);
  w.iz0 = bin_coord(zlo, z0, g.inv, g.nz);
  w.iz1 = bin_coord(zhi, z0, g.inv, g.nz);
  return w;
}

template <bool COUNT>
__global__ void __launch_bounds__(kNfThreads) k_neighbours(const Ctx c) {
  const uint32_t tr = blockIdx.x;
  const int row = (int)(tr % (uint32_t)c.n_rows);
  const uint32_t task = tr / (uint32_t)c.n_rows;
  const uint32_t lo = c.row_off[tr], hi = c.row_off[tr + 1];
  if (row == 0 || row == c.n_rows - 1) {  // SPEC 3: no links in the first and last row
    for (uint32_t i = lo + threadIdx.x; i < hi; i += kNfThreads) { c.link_up[i] = -1; c.link_dn[i] = -1; }
    return;
  }
  const float HY = c.prm.nf_hy, HZ = c.prm.nf_hz, CHI_MAX = c.prm.nf_chi2_max, M = kGridMargin;
  const float b = c.dx_dn[row], a_ = c.dx_up[row];                 // N4
  const float ratio_up = c.ratio_up[row], ratio_dn = c.ratio_dn[row];
  const float wy = c.wy, wz = c.wz;
  const float z0 = side_z0(c, task);
  unsigned long long n_pairs = 0ull;
  for (uint32_t i = lo + threadIdx.x; i < hi; i += kNfThreads) {
    const float2 h = c.yz[i];
    const float y = h.x, z = h.y;
    const float zu = z * ratio_up, zd = z * ratio_dn;              // N1
    const Window wu = make_window(c, tr + 1, row + 1, z0, (y - HY) - M, (y + HY) + M, (zu - HZ) - M, (zu + HZ) + M);
    const Window wd = make_window(c, tr - 1, row - 1, z0, (y - HY) - M, (y + HY) + M, (zd - HZ) - M, (zd + HZ) + M);
    bool have = false;
    float best = 0.0f;
    uint32_t bu = 0u, bd = 0u, bgu = 0u, bgd = 0u;  // idx and gid of the best pair
    for (int izu = wu.iz0; izu <= wu.iz1; ++izu) {
      const uint32_t u0 = wu.bins[izu * wu.ny + wu.iy0], u1 = wu.bins[izu * wu.ny + wu.iy1 + 1];
      for (uint32_t u = u0; u < u1; ++u) {
        const float2 pu = c.yz[u];
        if (!(fabsf(pu.x - y) <= HY && fabsf(pu.y - zu) <= HZ)) continue;   // N2
        const float ty = (pu.x - y) * b, tz = (pu.y - z) * b;
        for (int izd = wd.iz0; izd <= wd.iz1; ++izd) {
          const uint32_t d0 = wd.bins[izd * wd.ny + wd.iy0], d1 = wd.bins[izd * wd.ny + wd.iy1 + 1];
          for (uint32_t d = d0; d < d1; ++d) {
            const float2 pd = c.yz[d];
            if (!(fabsf(pd.x - y) <= HY && fabsf(pd.y - zd) <= HZ)) continue;  // N3
            const float dy = ty - ((y - pd.x) * a_);                          // N4
            const float dz = tz - ((z - pd.y) * a_);
            const float chi = ((dy * dy) * wy) + ((dz * dz) * wz);
            if (COUNT) ++n_pairs;
            if (!(chi < CHI_MAX)) continue;                                   // N5
            bool take = !have || chi < best;
            if (have && chi == best) {  // tie: lexicographic (gid_u, gid_d)
              const uint32_t gu = c.gid[u], gd = c.gid[d];
              take = gu < bgu || (gu == bgu && gd < bgd);
            }
            if (take) {
              have = true; best = chi; bu = u; bd = d;
              bgu = c.gid[u]; bgd = c.gid[d];
            }
          }
        }
      }
    }
    c.link_up[i] = have ? (int32_t)bu : -1;
    c.link_dn[i] = have ? (int32_t)bd : -1;
  }
  if (COUNT && n_pairs) atomicAdd(&c.counters[CN_NF_PAIRS], n_pairs);
}

// ---------------------------------------------------------------------------
// a3  neighbour cleaner (SPEC 4, C1): clean_up[h] = up[h] iff dn[up[h]] == h.
// One thread per cluster.  Also clears the ownership words of K7.
// ---------------------------------------------------------------------------
constexpr int kCleanThreads = 256;

__global__ void __launch_bounds__(kCleanThreads) k_clean(const Ctx c) {
  const uint32_t i = blockIdx.x * kCleanThreads + threadIdx.x;
  if (i >= c.n) return;
  const int32_t u = c.link_up[i];
  c.clean_up[i] = (u >= 0 && c.link_dn[u] == (int32_t)i) ? u : -1;
  c.owner[i] = 0ull;
}

// ---------------------------------------------------------------------------
// a4  start hits (S1) whose chain has >= min_seed_hits hits (S2, S3), written
// in idx order to trk_start / trk_tr.  Tile = kSeedThreads * kSeedItems idx.
// ---------------------------------------------------------------------------
constexpr int kSeedThreads = 256;
constexpr int kSeedItems = 4;
constexpr uint32_t kSeedTile = kSeedThreads * kSeedItems;

// task*n_rows + row of idx h: last tr with row_off[tr] <= h
__device__ __forceinline__ uint32_t find_tr(const Ctx& c, uint32_t h) {
  uint32_t lo = 0u, hi = c.n_tr;  // row_off[lo] <= h < row_off[hi]
  while (hi - lo > 1u) {
    const uint32_t mid = (lo + hi) >> 1;
    if (c.row_off[mid] <= h) lo = mid; else hi = mid;
  }
  return lo;
}

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
#pragma unroll
  for (int k = 0; k < kSeedItems; ++k) {
    const uint32_t i = base + k;
    if (i >= c.n) break;
    int32_t h = c.clean_up[i];
    if (h < 0) continue;
    const int32_t d = c.link_dn[i];
    if (d >= 0 && c.link_up[d] == (int32_t)i) continue;  // clean_dn[i] >= 0 (C2): not a start hit
    if (COUNT) ++n_s1;
    int len = 2;
    while (len < c.prm.min_seed_hits) {
      h = c.clean_up[h];
      if (h < 0) break;
      ++len;
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
      c.trk_start[pos] = base + k;
      c.trk_tr[pos] = find_tr(c, base + k);
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
