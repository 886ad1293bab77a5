// a2  neighbour finder (docs/ARITH_SPEC.md section 3, N1..N5; the
// Cellular-Automaton phase, one GPU thread per cluster).
//
// One block per (task,row).  The two neighbour rows r-1 and r+1 (their bin-sorted (y,z) pairs
// and their bin tables, both contiguous in memory) are staged in shared memory with two TMA 1-D
// bulk copies each (cp.async.bulk + mbarrier) when they fit; larger rows are read through L1.
// A thread first collects the down candidates that pass N3 into a short list in shared memory
// (stored as the products (y - y_d)*a_, (z - z_d)*a_ of N4), then walks its up window once and
// pairs every up candidate that passes N2 with the list.  Both window walks are single flat
// loops, so a warp runs max-over-lanes(candidates) iterations instead of the product of the
// nested trip counts.
#pragma once
#include "device_common.cuh"

namespace tpc {

constexpr int kNfThreads = 128;
constexpr int kNfList = 8;                    // down candidates a thread keeps; more -> nested fallback
constexpr uint32_t kNfStageBytes = 24 * 1024;  // staged neighbour rows (both) must fit in this
constexpr uint32_t kNfListBytes = kNfThreads * kNfList * 12;
constexpr uint32_t kNfSmemBytes = 16 + kNfListBytes + kNfStageBytes;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// TMA 1-D bulk copy global -> shared; size and both addresses are multiples of 16 bytes.
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}

// A neighbour row as the finder reads it: the staged copy or global memory.
struct RowView {
  const float2* yz;      // (y,z) of idx i at yz[i - yz_base]
  const uint32_t* bins;  // first idx of bin b at bins[b]; bins[ny*nz] = end of the row
  uint32_t yz_base;
  int ny, nz;
  float inv, y0;
};

// Calls f(idx, (y,z)) for every cluster whose bin overlaps the window; one flat loop.
template <class F>
__device__ __forceinline__ void for_window(const RowView& v, float z0, float ylo, float yhi, float zlo, float zhi,
                                           F&& f) {
  const int iy0 = bin_coord(ylo, v.y0, v.inv, v.ny), iy1 = bin_coord(yhi, v.y0, v.inv, v.ny);
  int iz = bin_coord(zlo, z0, v.inv, v.nz);
  const int iz1 = bin_coord(zhi, z0, v.inv, v.nz);
  const uint32_t* bp = v.bins + iz * v.ny;
  uint32_t i = bp[iy0], e = bp[iy1 + 1];
  while (true) {
    if (i >= e) {
      if (iz >= iz1) break;
      ++iz;
      bp += v.ny;
      i = bp[iy0];
      e = bp[iy1 + 1];
      continue;
    }
    f(i, v.yz[i - v.yz_base]);
    ++i;
  }
}

// lexicographic (chi, gid_u, gid_d) comparison of N5; the gids are only loaded on an exact chi tie
__device__ __forceinline__ bool nf_better(const Ctx& c, bool have, float chi, float best, uint32_t u, uint32_t d,
                                          uint32_t bu, uint32_t bd) {
  if (!have || chi < best) return true;
  if (chi != best) return false;
  const uint32_t gu = c.gid[u], gbu = c.gid[bu];
  if (gu != gbu) return gu < gbu;
  return c.gid[d] < c.gid[bd];
}

template <bool COUNT>
__device__ __forceinline__ void nf_row(const Ctx& c, const RowView& vu, const RowView& vd, int row, float z0,
                                       uint32_t lo, uint32_t hi, float* s_py, float* s_pz, uint32_t* s_pi) {
  const float HY = c.prm.nf_hy, HZ = c.prm.nf_hz, CHI_MAX = c.prm.nf_chi2_max, M = kGridMargin;
  const float b = c.dx_dn[row], a_ = c.dx_up[row];  // N4
  const float ratio_up = c.ratio_up[row], ratio_dn = c.ratio_dn[row];
  const float wy = c.wy, wz = c.wz;
  const int tid = threadIdx.x;
  unsigned long long n_pairs = 0ull;
  for (uint32_t i = lo + tid; i < hi; i += kNfThreads) {
    const float2 h = c.yz[i];
    const float y = h.x, z = h.y;
    const float zu = z * ratio_up, zd = z * ratio_dn;  // N1
    // down candidates (N3)
    int nd = 0;
    for_window(vd, z0, (y - HY) - M, (y + HY) + M, (zd - HZ) - M, (zd + HZ) + M, [&](uint32_t d, float2 pd) {
      if (!(fabsf(pd.x - y) <= HY && fabsf(pd.y - zd) <= HZ)) return;
      if (nd < kNfList) {
        s_py[nd * kNfThreads + tid] = (y - pd.x) * a_;
        s_pz[nd * kNfThreads + tid] = (z - pd.y) * a_;
        s_pi[nd * kNfThreads + tid] = d;
      }
      ++nd;
    });
    bool have = false;
    float best = 0.0f;
    uint32_t bu = 0u, bd = 0u;
    if (nd > 0 && nd <= kNfList) {
      for_window(vu, z0, (y - HY) - M, (y + HY) + M, (zu - HZ) - M, (zu + HZ) + M, [&](uint32_t u, float2 pu) {
        if (!(fabsf(pu.x - y) <= HY && fabsf(pu.y - zu) <= HZ)) return;  // N2
        const float ty = (pu.x - y) * b, tz = (pu.y - z) * b;
        if (COUNT) n_pairs += (unsigned)nd;
        for (int k = 0; k < nd; ++k) {
          const float dy = ty - s_py[k * kNfThreads + tid];  // N4
          const float dz = tz - s_pz[k * kNfThreads + tid];
          const float chi = ((dy * dy) * wy) + ((dz * dz) * wz);
          if (!(chi < CHI_MAX)) continue;  // N5
          const uint32_t d = s_pi[k * kNfThreads + tid];
          if (nf_better(c, have, chi, best, u, d, bu, bd)) { have = true; best = chi; bu = u; bd = d; }
        }
      });
    } else if (nd > kNfList) {  // list overflow: nested walk of both windows for this cluster
      for_window(vu, z0, (y - HY) - M, (y + HY) + M, (zu - HZ) - M, (zu + HZ) + M, [&](uint32_t u, float2 pu) {
        if (!(fabsf(pu.x - y) <= HY && fabsf(pu.y - zu) <= HZ)) return;
        const float ty = (pu.x - y) * b, tz = (pu.y - z) * b;
        for_window(vd, z0, (y - HY) - M, (y + HY) + M, (zd - HZ) - M, (zd + HZ) + M, [&](uint32_t d, float2 pd) {
          if (!(fabsf(pd.x - y) <= HY && fabsf(pd.y - zd) <= HZ)) return;
          const float dy = ty - ((y - pd.x) * a_);
          const float dz = tz - ((z - pd.y) * a_);
          const float chi = ((dy * dy) * wy) + ((dz * dz) * wz);
          if (COUNT) ++n_pairs;
          if (!(chi < CHI_MAX)) return;
          if (nf_better(c, have, chi, best, u, d, bu, bd)) { have = true; best = chi; bu = u; bd = d; }
        });
      });
    }
    c.link_up[i] = have ? (int32_t)bu : -1;
    c.link_dn[i] = have ? (int32_t)bd : -1;
  }
  if (COUNT && n_pairs) atomicAdd(&c.counters[CN_NF_PAIRS], n_pairs);
}

template <bool COUNT>
__global__ void __launch_bounds__(kNfThreads) k_neighbours(const Ctx c) {
  extern __shared__ __align__(16) unsigned char nf_smem[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(nf_smem);
  float* s_py = reinterpret_cast<float*>(nf_smem + 16);
  float* s_pz = s_py + kNfThreads * kNfList;
  uint32_t* s_pi = reinterpret_cast<uint32_t*>(s_pz + kNfThreads * kNfList);
  unsigned char* stage = nf_smem + 16 + kNfListBytes;

  const uint32_t tr = blockIdx.x;
  const int row = (int)(tr % (uint32_t)c.n_rows);
  const uint32_t task = tr / (uint32_t)c.n_rows;
  const uint32_t lo = c.row_off[tr], hi = c.row_off[tr + 1];
  if (hi == lo) return;
  if (row == 0 || row == c.n_rows - 1) {  // SPEC 3: no links in the first and last row
    for (uint32_t i = lo + threadIdx.x; i < hi; i += kNfThreads) { c.link_up[i] = -1; c.link_dn[i] = -1; }
    return;
  }
  const float z0 = side_z0(c, task);
  const RowInfo gu = load_row_info(&c.rowinfo[tr + 1]), gd = load_row_info(&c.rowinfo[tr - 1]);
  const uint32_t u_hi = c.row_off[tr + 2];
  RowView vu, vd;
  vu.ny = info_ny(gu); vu.nz = info_nz(gu); vu.inv = gu.inv; vu.y0 = -c.ymax[row + 1];
  vd.ny = info_ny(gd); vd.nz = info_nz(gd); vd.inv = gd.inv; vd.y0 = -c.ymax[row - 1];
  // 16-byte aligned source ranges: (y,z) pairs [ya0, ya1) and bin entries [ba0, ba1) of both rows
  const uint32_t uya0 = gu.row_lo & ~1u, uya1 = (u_hi + 1u) & ~1u;
  const uint32_t dya0 = gd.row_lo & ~1u, dya1 = (lo + 1u) & ~1u;
  const uint32_t unb = (uint32_t)(vu.ny * vu.nz) + 1u, dnb = (uint32_t)(vd.ny * vd.nz) + 1u;
  const uint32_t uba0 = gu.bins_off & ~3u, uba1 = (gu.bins_off + unb + 3u) & ~3u;
  const uint32_t dba0 = gd.bins_off & ~3u, dba1 = (gd.bins_off + dnb + 3u) & ~3u;
  const uint32_t b_uyz = (uya1 - uya0) * 8u, b_dyz = (dya1 - dya0) * 8u;
  const uint32_t b_ub = (uba1 - uba0) * 4u, b_db = (dba1 - dba0) * 4u;
  const bool staged = b_uyz + b_dyz + b_ub + b_db <= kNfStageBytes;
  if (staged) {
    float2* s_uyz = reinterpret_cast<float2*>(stage);
    float2* s_dyz = reinterpret_cast<float2*>(stage + b_uyz);
    uint32_t* s_ub = reinterpret_cast<uint32_t*>(stage + b_uyz + b_dyz);
    uint32_t* s_db = reinterpret_cast<uint32_t*>(stage + b_uyz + b_dyz + b_ub);
    if (threadIdx.x == 0) {
      mbar_init(bar, 1u);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      mbar_expect_tx(bar, b_uyz + b_dyz + b_ub + b_db);
      if (b_uyz) bulk_g2s(s_uyz, c.yz + uya0, b_uyz, bar);
      if (b_dyz) bulk_g2s(s_dyz, c.yz + dya0, b_dyz, bar);
      bulk_g2s(s_ub, c.bins + uba0, b_ub, bar);
      bulk_g2s(s_db, c.bins + dba0, b_db, bar);
    }
    mbar_wait(bar, 0u);
    vu.yz = s_uyz; vu.yz_base = uya0; vu.bins = s_ub + (gu.bins_off - uba0);
    vd.yz = s_dyz; vd.yz_base = dya0; vd.bins = s_db + (gd.bins_off - dba0);
    nf_row<COUNT>(c, vu, vd, row, z0, lo, hi, s_py, s_pz, s_pi);
  } else {
    vu.yz = c.yz; vu.yz_base = 0u; vu.bins = c.bins + gu.bins_off;
    vd.yz = c.yz; vd.yz_base = 0u; vd.bins = c.bins + gd.bins_off;
    nf_row<COUNT>(c, vu, vd, row, z0, lo, hi, s_py, s_pz, s_pi);
  }
}

}  // namespace tpc
