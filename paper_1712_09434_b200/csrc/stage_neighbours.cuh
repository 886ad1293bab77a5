// a2  neighbour finder (docs/ARITH_SPEC.md section 3, N1..N5; the
// Cellular-Automaton phase, one GPU thread per cluster).
//
// One block per (task,row).  The two neighbour rows r-1 and r+1 (their bin-sorted (y,z) pairs
// and their bin tables, both contiguous in memory) are staged in shared memory with two TMA 1-D
// bulk copies each (cp.async.bulk + mbarrier) when they fit; larger rows are read through L1.
// A thread owns one cluster and runs three flat loops, each entered by the whole warp together:
// the down window (clusters that pass N3 go to a short list in shared memory, stored as the
// products (y - y_d)*a_, (z - z_d)*a_ of N4), the up window (N2, list of (y_u - y)*b, (z_u - z)*b),
// and the nu*nd pairs of the two lists (N4, N5).  A window is read as ONE virtual range over its
// (at most two, else looped) bin rows, so a warp runs max-over-lanes(candidates) iterations of a
// short branch-free body instead of nested loops.  A list overflow or two pairs of equal chi2 send the
// cluster to the nested serial walk, which alone compares gids.
#pragma once
#include "device_common.cuh"

namespace tpc {

#ifndef TPC_NF_THREADS
#define TPC_NF_THREADS 128
#endif
constexpr int kNfThreads = TPC_NF_THREADS;
#ifndef TPC_NF_MINBLOCKS
#define TPC_NF_MINBLOCKS 5  // 5 blocks per SM is what the 43 KB of shared memory allow: up to 102 registers, no spill (without the bound ptxas stopped at 72 and spilled)
#endif
#ifndef TPC_NF_LIST
#define TPC_NF_LIST 8
#endif
constexpr int kNfList = TPC_NF_LIST;                    // candidates per side a cluster keeps (more -> serial search) at the
constexpr int kNfListDense = 16;              // density of a central event / in denser batches (host's choice)
constexpr uint32_t kNfDenseRow = 900;         // mean clusters per row from which the deeper lists are used
constexpr uint32_t kNfStageBytes = 18 * 1024 + 512;  // staged neighbour rows (both) must fit in this
__host__ __device__ constexpr uint32_t nf_list_bytes(int list) { return 2u * kNfThreads * (uint32_t)list * 12u; }  // 2 sides x (py, pz, idx)
__host__ __device__ constexpr uint32_t nf_smem_bytes(int list) { return 16u + nf_list_bytes(list) + kNfStageBytes; }

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
  float inv, y0, z0;
};

// Calls f(idx, (y,z)) for every cluster whose bin overlaps the window; one flat loop.
template <class F>
__device__ __forceinline__ void for_window(const RowView& v, float ylo, float yhi, float zlo, float zhi,
                                           F&& f) {
  const int iy0 = bin_coord(ylo, v.y0, v.inv, v.ny), iy1 = bin_coord(yhi, v.y0, v.inv, v.ny);
  int iz = bin_coord(zlo, v.z0, v.inv, v.nz);
  const int iz1 = bin_coord(zhi, v.z0, v.inv, v.nz);
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


// The exact serial search of one cluster (N1..N5 as written, ties by gid): nested walk of both windows.
// Used for the rare clusters the cooperative search cannot decide (chi2 ties, list overflow).
// The views are passed BY VALUE and the result comes back in a register pair: nothing of the caller has its address
// taken, so its row views and counters stay in registers (by reference they lived in local memory, and the hot loops
// of every cluster re-read them from there).
template <bool COUNT>
__device__ __noinline__ uint2 nf_serial(const Ctx& c, const RowView vu, const RowView vd, int row, float y, float z,
                                        unsigned long long* pairs_out) {
  const float HY = c.prm.nf_hy, HZ = c.prm.nf_hz, CHI_MAX = c.prm.nf_chi2_max, M = kGridMargin;
  const float b = c.dx_dn[row], a_ = c.dx_up[row];  // N4
  const float zu = z * c.ratio_up[row], zd = z * c.ratio_dn[row];  // N1
  const float wy = c.wy, wz = c.wz;
  bool have = false;
  float best = 0.0f;
  uint32_t bu = 0u, bd = 0u;
  unsigned long long n_pairs = 0ull;
  for_window(vu, (y - HY) - M, (y + HY) + M, (zu - HZ) - M, (zu + HZ) + M, [&](uint32_t u, float2 pu) {
    if (!(fabsf(pu.x - y) <= HY && fabsf(pu.y - zu) <= HZ)) return;  // N2
    const float ty = (pu.x - y) * b, tz = (pu.y - z) * b;
    for_window(vd, (y - HY) - M, (y + HY) + M, (zd - HZ) - M, (zd + HZ) + M, [&](uint32_t d, float2 pd) {
      if (!(fabsf(pd.x - y) <= HY && fabsf(pd.y - zd) <= HZ)) return;  // N3
      const float dy = ty - ((y - pd.x) * a_);  // N4
      const float dz = tz - ((z - pd.y) * a_);
      const float chi = ((dy * dy) * wy) + ((dz * dz) * wz);
      if (COUNT) ++n_pairs;
      if (!(chi < CHI_MAX)) return;  // N5: lexicographic (chi, gid_u, gid_d)
      bool take = !have || chi < best;
      if (have && chi == best) {
        const uint32_t gu = c.gid[u], gbu = c.gid[bu];
        take = gu != gbu ? gu < gbu : c.gid[d] < c.gid[bd];
      }
      if (take) { have = true; best = chi; bu = u; bd = d; }
    });
  });
  if (COUNT) *pairs_out += n_pairs;
  return have ? make_uint2(bu, bd) : make_uint2(0xFFFFFFFFu, 0xFFFFFFFFu);
}

// Window walk of one thread around (y, zc) (zc = the projected z of N1) in row view v: the clusters that
// pass the window test are appended to the thread's list as ((p.x - y)*sgn*fac, (p.y - z)*sgn*fac, idx).
// Returns the number that passed (entries beyond LIST are not stored).
template <int LIST>
__device__ __forceinline__ uint32_t nf_collect(const RowView& v, bool act, float y, float z, float zc,
                                               float HY, float HZ, float sgn, float fac, float2* l_p,
                                               uint32_t* l_i) {
  const float M = kGridMargin;
  const int iy0 = bin_coord((y - HY) - M, v.y0, v.inv, v.ny), iy1 = bin_coord((y + HY) + M, v.y0, v.inv, v.ny) + 1;
  const int iz0 = bin_coord((zc - HZ) - M, v.z0, v.inv, v.nz);
  const int nzr = act ? bin_coord((zc + HZ) + M, v.z0, v.inv, v.nz) - iz0 + 1 : 0;
  uint32_t n = 0u;
  for (int r = 0; r < nzr; r += 2) {
    const uint32_t* bp = v.bins + (iz0 + r) * v.ny;
    const uint32_t i1 = bp[iy0], n1 = bp[iy1] - i1;
    uint32_t i2 = 0u, n2 = 0u;
    if (r + 1 < nzr) { i2 = bp[v.ny + iy0]; n2 = bp[v.ny + iy1] - i2; }
    const uint32_t n_tot = n1 + n2;
    const uint32_t skip = i2 - (i1 + n1);  // idx of candidate k >= n1 is i1 + k + skip
    for (uint32_t k = 0u; k < n_tot; ++k) {
      const uint32_t idx = i1 + k + (k < n1 ? 0u : skip);
      const float2 p = v.yz[idx - v.yz_base];
      const float ry = p.x - y;
      const bool pass = (fabsf(ry) <= HY) & (fabsf(p.y - zc) <= HZ);  // N2 / N3
      // stored whether it passes or not: a cluster that fails is overwritten by the next one (n stays)
      if (n < (uint32_t)LIST) {
        const uint32_t slot = n * kNfThreads;
        // up: (y_u - y)*b, (z_u - z)*b.  down: (y - y_d)*a_, (z - z_d)*a_ (exact negation of the difference)
        l_p[slot] = make_float2((sgn * ry) * fac, (sgn * (p.y - z)) * fac);
        l_i[slot] = idx;
      }
      n += pass ? 1u : 0u;
    }
  }
  return n;
}

template <bool COUNT, int LIST>
__device__ __forceinline__ void nf_row(const Ctx& c, const RowView& vu, const RowView& vd, int row,
                                       uint32_t lo, uint32_t hi, unsigned char* list_smem) {
  const float HY = c.prm.nf_hy, HZ = c.prm.nf_hz, CHI_MAX = c.prm.nf_chi2_max;
  const float b = c.dx_dn[row], a_ = c.dx_up[row];  // N4
  const float ratio_up = c.ratio_up[row], ratio_dn = c.ratio_dn[row];
  const float wy = c.wy, wz = c.wz;
  const int tid = threadIdx.x;
  float2* d_p = reinterpret_cast<float2*>(list_smem) + tid;  // [LIST][kNfThreads] each, this thread's column
  float2* u_p = d_p + LIST * kNfThreads;
  uint32_t* d_i = reinterpret_cast<uint32_t*>(reinterpret_cast<float2*>(list_smem) + 2 * LIST * kNfThreads) + tid;
  uint32_t* u_i = d_i + LIST * kNfThreads;
  unsigned long long n_pairs = 0ull;
  for (uint32_t i0 = lo + (uint32_t)(tid & ~31); i0 < hi; i0 += kNfThreads) {  // warp-uniform trip count
    const uint32_t i = i0 + (uint32_t)(tid & 31);
    const bool act = i < hi;
    float y = 0.0f, z = 0.0f;
    if (act) { const float2 h = c.yz[i]; y = h.x; z = h.y; }
    const float zu = z * ratio_up, zd = z * ratio_dn;  // N1
    const uint32_t nd = nf_collect<LIST>(vd, act, y, z, zd, HY, HZ, -1.0f, a_, d_p, d_i);  // N3
    __syncwarp();
    const uint32_t nu = nd ? nf_collect<LIST>(vu, act, y, z, zu, HY, HZ, 1.0f, b, u_p, u_i) : 0u;  // N2
    __syncwarp();
    const bool overflow = nd > (uint32_t)LIST || nu > (uint32_t)LIST;
    const uint32_t n_pr = overflow ? 0u : nu * nd;
    if (COUNT) n_pairs += n_pr;
    float best = CHI_MAX;  // N5: only chi < CHI_MAX is eligible
    uint32_t bu = 0u, bd = 0u;
    bool tie = false;
    for (uint32_t k = 0u, u = 0u, d = 0u; k < n_pr; ++k) {  // pair k = (u, d) = (k / nd, k % nd), counted along
      const float2 pu = u_p[u * kNfThreads], pd = d_p[d * kNfThreads];
      const float dy = pu.x - pd.x, dz = pu.y - pd.y;  // N4
      const float chi = ((dy * dy) * wy) + ((dz * dz) * wz);
      const bool lt = chi < best;
      tie |= chi == best;  // equal chi2 (or chi2 == CHI_MAX exactly): the gids decide (N5), left to the serial search
      best = lt ? chi : best;
      bu = lt ? u : bu;
      bd = lt ? d : bd;
      const bool wrap = d + 1u == nd;
      d = wrap ? 0u : d + 1u;
      u += wrap ? 1u : 0u;
    }
    const bool have = best < CHI_MAX;
    __syncwarp();
    if (act) {
      int32_t up = -1, dn = -1;
      if (overflow || tie) {
        unsigned long long extra = 0ull;
        const uint2 l = nf_serial<COUNT>(c, vu, vd, row, y, z, &extra);
        up = (int32_t)l.x; dn = (int32_t)l.y;
        if (COUNT) n_pairs += extra;
      } else if (have) {
        up = (int32_t)u_i[bu * kNfThreads];
        dn = (int32_t)d_i[bd * kNfThreads];
      }
      c.link_up[i] = up;
      c.link_dn[i] = dn;
    }
  }
  if (COUNT && n_pairs) atomicAdd(&c.counters[CN_NF_PAIRS], n_pairs);
}

template <bool COUNT, int LIST>
__global__ void __launch_bounds__(kNfThreads, TPC_NF_MINBLOCKS) k_neighbours(const __grid_constant__ Ctx c) {
  extern __shared__ __align__(16) unsigned char nf_smem[];
  uint64_t* bar = reinterpret_cast<uint64_t*>(nf_smem);
  unsigned char* list_smem = nf_smem + 16;
  unsigned char* stage = nf_smem + 16 + nf_list_bytes(LIST);

  const uint32_t tr = blockIdx.x;
  const int row = (int)(tr % (uint32_t)c.n_rows);
  const uint32_t lo = c.row_off[tr], hi = c.row_off[tr + 1];
  if (hi == lo) return;
  if (row == 0 || row == c.n_rows - 1) {  // SPEC 3: no links in the first and last row
    for (uint32_t i = lo + threadIdx.x; i < hi; i += kNfThreads) { c.link_up[i] = -1; c.link_dn[i] = -1; }
    return;
  }
  const RowInfo gu = load_row_info(&c.rowinfo[tr + 1]), gd = load_row_info(&c.rowinfo[tr - 1]);
  const uint32_t u_hi = c.row_off[tr + 2];
  RowView vu, vd;
  vu.ny = info_ny(gu); vu.nz = info_nz(gu); vu.inv = gu.inv; vu.y0 = gu.y0; vu.z0 = gu.z0;
  vd.ny = info_ny(gd); vd.nz = info_nz(gd); vd.inv = gd.inv; vd.y0 = gd.y0; vd.z0 = gd.z0;
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
    nf_row<COUNT, LIST>(c, vu, vd, row, lo, hi, list_smem);
  } else {
    vu.yz = c.yz; vu.yz_base = 0u; vu.bins = c.bins + gu.bins_off;
    vd.yz = c.yz; vd.yz_base = 0u; vd.bins = c.bins + gd.bins_off;
    nf_row<COUNT, LIST>(c, vu, vd, row, lo, hi, list_smem);
  }
}

}  // namespace tpc
