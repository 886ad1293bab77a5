// Sector-segment merger and final refit (the tracker "merges the
// tracks segments afterward"; L140: the Kalman refit the paper wants on the GPU next to the tracker, so that
// track segments never cross PCIe between the two).  docs/ARITH_SPEC.md section 9: ROTATE (R1..R7), matching
// (G1..G7), refit (F1..F3).  Runs behind a7 on the arrays the tracker left in its workspace: the bin-sorted
// (y,z), the row maps with their kept hits flagged by k_resolve, and what k_select_output noted per track.
//   k_merge_ends    G1   one thread per sector track: the fitted helix at the row of its outermost kept hit
//   k_merge_match   G2..G5  one thread per track: its best continuation in the two neighbouring sectors and
//                        the best segment it continues, both by the full test (rotate, transport, chi2) on
//                        every candidate that passes the row test; no atomics, ties by first-hit gid
//   k_merge_link    G6, G7  mutual choices become links; chain heads are numbered in track order
//   k_merge_refit   F1..F3  one thread per chain: the filter pass from the outermost hit inwards, rotating the
//                        state where the chain changes sector
#pragma once
#include "device_common.cuh"
#include "stage_tracklet.cuh"

namespace tpc {

constexpr int kMergeThreads = 128;
constexpr int kEndFloats = 24;  // outer end of a track: p[5], C[15], 1.0f if it exists, 3 pad  (6 float4)

// SPEC 9.1 ROTATE.  sa carries the sign of the direction.  Fails (state untouched) beyond the angle limit.
__device__ __forceinline__ bool rotate_state(TrackState& S, float& x, float ca, float sa, float a, float max_sinphi) {
  const float y = S.y, s = S.s, t = S.t, q = S.q;
  const float c = sqrtf(1.0f - s * s);                     // R1
  const float s1 = s * ca - c * sa;                        // R2
  const float c1 = c * ca + s * sa;
  if (!(c1 > 0.0f && fabsf(s1) <= max_sinphi)) return false;  // R3
  const float j00 = ca - (s1 / c1) * sa;                   // R5
  const float j10 = -((t / c1) * sa);
  const float j20 = -((a * q) * sa);
  const float j22 = ca + (s / c) * sa;
  const float c00 = S.c00, c10 = S.c10, c11 = S.c11, c20 = S.c20, c21 = S.c21, c22 = S.c22, c30 = S.c30, c31 = S.c31,
              c32 = S.c32, c40 = S.c40, c41 = S.c41, c42 = S.c42;
  const float m00 = j00 * c00;                             // R6
  const float m10 = j10 * c00 + c10, m11 = j10 * c10 + c11;
  const float m20 = j20 * c00 + j22 * c20, m21 = j20 * c10 + j22 * c21, m22 = j20 * c20 + j22 * c22;
  S.c00 = m00 * j00;                                       // R7
  S.c10 = m10 * j00; S.c11 = m10 * j10 + m11;
  S.c20 = m20 * j00; S.c21 = m20 * j10 + m21; S.c22 = m20 * j20 + m22 * j22;
  S.c30 = c30 * j00; S.c31 = c30 * j10 + c31; S.c32 = c30 * j20 + c32 * j22;
  S.c40 = c40 * j00; S.c41 = c40 * j10 + c41; S.c42 = c40 * j20 + c42 * j22;
  const float xn = x * ca + y * sa;                        // R4
  S.y = y * ca - x * sa;
  S.s = s1;
  x = xn;
  return true;
}

// output state of sector track i (L3) from the SoA columns of tpc_tracks
__device__ __forceinline__ void load_track_state(const tpc_tracks& o, uint32_t i, TrackState& S, float& x) {
  const size_t cap = o.track_capacity;
  x = o.track_x[i];
  S.y = o.track_par[i]; S.z = o.track_par[cap + i]; S.s = o.track_par[2 * cap + i];
  S.t = o.track_par[3 * cap + i]; S.q = o.track_par[4 * cap + i];
  const float* cv = o.track_cov + i;
  S.c00 = cv[0]; S.c10 = cv[cap]; S.c11 = cv[2 * cap]; S.c20 = cv[3 * cap]; S.c21 = cv[4 * cap]; S.c22 = cv[5 * cap];
  S.c30 = cv[6 * cap]; S.c31 = cv[7 * cap]; S.c32 = cv[8 * cap]; S.c33 = cv[9 * cap];
  S.c40 = cv[10 * cap]; S.c41 = cv[11 * cap]; S.c42 = cv[12 * cap]; S.c43 = cv[13 * cap]; S.c44 = cv[14 * cap];
  S.chi2 = 0.0f; S.ndf = 0;
}
__device__ __forceinline__ void store_end(float4* e, const TrackState& S, bool ok) {
  e[0] = make_float4(S.y, S.z, S.s, S.t);
  e[1] = make_float4(S.q, S.c00, S.c10, S.c11);
  e[2] = make_float4(S.c20, S.c21, S.c22, S.c30);
  e[3] = make_float4(S.c31, S.c32, S.c33, S.c40);
  e[4] = make_float4(S.c41, S.c42, S.c43, S.c44);
  e[5] = make_float4(ok ? 1.0f : 0.0f, 0.0f, 0.0f, 0.0f);
}
__device__ __forceinline__ bool load_end(const float4* e, TrackState& S) {
  const float4 a0 = e[0], a1 = e[1], a2 = e[2], a3 = e[3], a4 = e[4], a5 = e[5];
  S.y = a0.x; S.z = a0.y; S.s = a0.z; S.t = a0.w;
  S.q = a1.x; S.c00 = a1.y; S.c10 = a1.z; S.c11 = a1.w;
  S.c20 = a2.x; S.c21 = a2.y; S.c22 = a2.z; S.c30 = a2.w;
  S.c31 = a3.x; S.c32 = a3.y; S.c33 = a3.z; S.c40 = a3.w;
  S.c41 = a4.x; S.c42 = a4.y; S.c43 = a4.z; S.c44 = a4.w;
  S.chi2 = 0.0f; S.ndf = 0;
  return a5.x != 0.0f;
}

// Everything the merger kernels need beside the tracker's Ctx.
struct MergeCtx {
  tpc_merged out;
  float chi2_max;
  int32_t max_row_gap;
  int32_t n_half;             // sectors per side
  float ca, sa;               // cos, sin of the sector pitch (SPEC 9 tables)
  uint32_t n_tracks_cap;      // = tpc_tracks::track_capacity
  // merge workspace (device)
  float4* ends;               // [cap][6]   G1
  uint32_t* track_off;        // [n_tasks + 1] first track of every task (tracks are in task order)
  int32_t *best_out, *best_in;  // [cap]
  unsigned long long* scan;   // look-back state of the chain-head numbering, [tiles]
  uint32_t* ticket;           // [1]
};

// sector tracks the merger works on: none if the tracker reported an overflow (their arrays may be incomplete)
__device__ __forceinline__ uint32_t merge_n_tracks(const Ctx& c, const MergeCtx& m) {
  if (c.out.header[2] != 0u) return 0u;
  return min(min(c.out.header[0], c.out.track_capacity), m.out.capacity);
}

// first track of every task
__global__ void k_merge_task_offsets(const Ctx c, const MergeCtx m) {
  const uint32_t n_trk = merge_n_tracks(c, m);
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < n_trk; t += gridDim.x * blockDim.x) {
    const uint32_t task = c.out.track_task[t];
    const uint32_t from = t ? c.out.track_task[t - 1u] + 1u : 0u;
    for (uint32_t k = from; k <= task; ++k) m.track_off[k] = t;
    if (t == n_trk - 1u)
      for (uint32_t k = task + 1u; k <= c.n_tasks; ++k) m.track_off[k] = n_trk;
  }
}

// G1: the fitted helix at the row of the outermost kept hit
__global__ void __launch_bounds__(kMergeThreads) k_merge_ends(const Ctx c, const MergeCtx m) {
  const uint32_t n_trk = merge_n_tracks(c, m);
  const uint32_t i = blockIdx.x * kMergeThreads + threadIdx.x;
  if (i >= n_trk) return;
  TrackState S;
  float x;
  load_track_state(c.out, i, S, x);
  const uint32_t rows = c.out_rows[i];
  const float x_end = c.X[rows >> 16];
  bool ok = true;
  if (x_end != x) ok = transport(S, x_end - x, c.a, c.prm.max_sinphi);
  store_end(m.ends + (size_t)i * 6, S, ok);
}

// G3, G4 for the pair (inner i -> outer j) in direction d; Q = outer end of i at X[rl_i].  Returns chi or +inf.
__device__ __forceinline__ float merge_chi(const Ctx& c, const MergeCtx& m, TrackState Q, float xq, int d, uint32_t j) {
  const float kInf = __int_as_float(0x7f800000);
  if (!rotate_state(Q, xq, m.ca, d > 0 ? m.sa : -m.sa, c.a, c.prm.max_sinphi)) return kInf;
  TrackState B;
  float xb;
  load_track_state(c.out, j, B, xb);
  if (xb != xq && !transport(Q, xb - xq, c.a, c.prm.max_sinphi)) return kInf;
  const float d0 = Q.y - B.y, d1 = Q.z - B.z, d2 = Q.s - B.s, d3 = Q.t - B.t, d4 = Q.q - B.q;
  float chi = (d0 * d0) / (Q.c00 + B.c00);                 // G4, left to right
  chi = chi + (d1 * d1) / (Q.c11 + B.c11);
  chi = chi + (d2 * d2) / (Q.c22 + B.c22);
  chi = chi + (d3 * d3) / (Q.c33 + B.c33);
  chi = chi + (d4 * d4) / (Q.c44 + B.c44);
  return chi;
}

// G2..G5.  Thread t: best_out[t] over the tracks t may continue into, best_in[t] over the tracks that may
// continue into t.  Both loops apply the same test to the same ordered pair, so the two sides agree bit for bit.
__global__ void __launch_bounds__(kMergeThreads) k_merge_match(const Ctx c, const MergeCtx m) {
  const uint32_t n_trk = merge_n_tracks(c, m);
  const uint32_t t = blockIdx.x * kMergeThreads + threadIdx.x;
  if (t >= n_trk) return;
  const int ns = c.n_sectors, nh = m.n_half;
  const uint32_t task = c.out.track_task[t];
  const int sec = (int)(task % (uint32_t)ns), side = nh > 0 ? sec / nh : 0, f = sec - side * nh;
  const uint32_t ev_base = task - (uint32_t)sec;
  const uint32_t rows_t = c.out_rows[t];
  const int rf_t = (int)(rows_t & 0xFFFFu), rl_t = (int)(rows_t >> 16);
  const int gap = m.max_row_gap;
  int32_t best_out = -1, best_in = -1;
  float chi_out = 0.0f, chi_in = 0.0f;
  uint32_t gid_out = 0u, gid_in = 0u;
  const int n_dir = nh >= 3 ? 2 : (nh == 2 ? 1 : 0);
  TrackState E;
  const bool has_end = load_end(m.ends + (size_t)t * 6, E);
  for (int k = 0; k < n_dir; ++k) {
    const int d = k == 0 ? +1 : -1;
    // t as the inner segment: candidates j in the neighbour in direction d
    if (has_end) {
      const uint32_t tj = ev_base + (uint32_t)(side * nh + (f + d + nh) % nh);
      for (uint32_t j = m.track_off[tj], je = m.track_off[tj + 1u]; j < je; ++j) {
        const int rf_j = (int)(c.out_rows[j] & 0xFFFFu);
        if (!(rl_t < rf_j && rf_j <= rl_t + gap)) continue;                        // G2
        const float chi = merge_chi(c, m, E, c.X[rl_t], d, j);                      // G3, G4
        if (!(chi < m.chi2_max)) continue;
        const uint32_t g = c.out.hit_cluster[c.out.track_hit_begin[j]];
        if (best_out < 0 || chi < chi_out || (chi == chi_out && g < gid_out)) { best_out = (int32_t)j; chi_out = chi; gid_out = g; }  // G5
      }
    }
    // t as the outer segment: candidates i whose neighbour in direction d is this sector
    {
      const uint32_t ti = ev_base + (uint32_t)(side * nh + (f - d + nh) % nh);
      for (uint32_t i = m.track_off[ti], ie = m.track_off[ti + 1u]; i < ie; ++i) {
        const int rl_i = (int)(c.out_rows[i] >> 16);
        if (!(rl_i < rf_t && rf_t <= rl_i + gap)) continue;
        TrackState Ei;
        if (!load_end(m.ends + (size_t)i * 6, Ei)) continue;
        const float chi = merge_chi(c, m, Ei, c.X[rl_i], d, t);
        if (!(chi < m.chi2_max)) continue;
        const uint32_t g = c.out.hit_cluster[c.out.track_hit_begin[i]];
        if (best_in < 0 || chi < chi_in || (chi == chi_in && g < gid_in)) { best_in = (int32_t)i; chi_in = chi; gid_in = g; }
      }
    }
  }
  m.best_out[t] = best_out;
  m.best_in[t] = best_in;
}

// G6: mutual choices become links.
__global__ void __launch_bounds__(kMergeThreads) k_merge_link(const Ctx c, const MergeCtx m) {
  const uint32_t n_trk = merge_n_tracks(c, m);
  const uint32_t t = blockIdx.x * kMergeThreads + threadIdx.x;
  if (t >= n_trk) return;
  const int32_t j = m.best_out[t], i = m.best_in[t];
  const bool fwd = j >= 0 && m.best_in[j] == (int32_t)t, bwd = i >= 0 && m.best_out[i] == (int32_t)t;
  m.out.seg_next[t] = fwd ? j : -1;
  m.out.seg_prev[t] = bwd ? i : -1;
  if (fwd) atomicAdd(&m.out.header[1], 1u);
}

// G7 + F1..F3.  One thread per sector track; the heads of chains (no previous segment) are numbered in track
// order (block scan + chained scan with decoupled look-back) and refit their chain.
__global__ void __launch_bounds__(kMergeThreads) k_merge_refit(const Ctx c, const MergeCtx m) {
  __shared__ uint32_t s_warp[33];
  __shared__ uint32_t s_tile;
  __shared__ unsigned long long s_prefix;
  if (threadIdx.x == 0) s_tile = atomicAdd(m.ticket, 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t n_trk = merge_n_tracks(c, m);
  const uint32_t i1 = tile * kMergeThreads + threadIdx.x;
  const bool head = i1 < n_trk && m.out.seg_prev[i1] < 0;
  uint32_t total;
  const uint32_t excl = block_exclusive_scan(head ? 1u : 0u, s_warp, &total);
  if (threadIdx.x < 32) {
    const unsigned long long p = lookback_exclusive(m.scan, tile, (unsigned long long)total);
    if (threadIdx.x == 0) s_prefix = p;
  }
  __syncthreads();
  const uint32_t slot = (uint32_t)s_prefix + excl;
  if (threadIdx.x == 0 && tile == gridDim.x - 1) m.out.header[0] = (uint32_t)s_prefix + total;
  if (!head) return;
  const int n_rows = c.n_rows, ns = c.n_sectors, nh = m.n_half;
  // the chain: its outermost segment, number of segments and of kept hits
  uint32_t im = i1, n_seg = 1u, n_hits = c.out.track_nhits[i1];
  for (int32_t k = m.out.seg_next[i1]; k >= 0; k = m.out.seg_next[k]) { im = (uint32_t)k; ++n_seg; n_hits += c.out.track_nhits[k]; }
  TrackState S;
  float x = c.X[c.out_rows[im] >> 16];
  int sector = (int)(c.out.track_task[im] % (uint32_t)ns);
  uint32_t n_fit = 0u;
  if (load_end(m.ends + (size_t)im * 6, S)) {
    const float f = c.prm.turn_cov_scale;                                          // F1
    S.c00 *= f; S.c10 *= f; S.c11 *= f; S.c20 *= f; S.c21 *= f; S.c22 *= f; S.c30 *= f; S.c31 *= f;
    S.c32 *= f; S.c33 *= f; S.c40 *= f; S.c41 *= f; S.c42 *= f; S.c43 *= f; S.c44 *= f;
    S.chi2 = 0.0f; S.ndf = -5;
    bool go = true;
    for (int32_t k = (int32_t)im; k >= 0 && go; k = m.out.seg_prev[k]) {           // F2: segments outermost first
      const int sec_k = (int)(c.out.track_task[k] % (uint32_t)ns);
      const uint32_t rows = c.out_rows[k];
      const uint32_t* map = c.trk_hits + (size_t)c.out_trk[k] * map_stride(n_rows);
      const int r_lo = (int)(rows & 0xFFFFu);
      uint32_t e_next = map[rows >> 16];
      for (int r = (int)(rows >> 16); r >= r_lo; --r) {
        const uint32_t e = e_next;
        if (r > r_lo) e_next = map[r - 1];
        if (e == kNoHit || !(e & kOwnedBit)) continue;                             // kept hits only (L1)
        const float2 h = c.yz[e & ~kOwnedBit];
        if (sec_k != sector) {
          const int fs = sector % nh, fk = sec_k % nh;
          const int d = (fs + 1) % nh == fk ? +1 : -1;
          if (!rotate_state(S, x, m.ca, d > 0 ? m.sa : -m.sa, c.a, c.prm.max_sinphi)) { go = false; break; }
          sector = sec_k;
        }
        const float xr = c.X[r];
        if (x != xr) {
          if (!transport(S, xr - x, c.a, c.prm.max_sinphi)) { go = false; break; }
          x = xr;
        }
        update_hit(S, h.x, h.y, c.sy2, c.sz2);
        ++n_fit;
      }
    }
  } else {  // F1: no outer end, no refit: the segment's own fit
    load_track_state(c.out, im, S, x);
    S.chi2 = c.out.track_chi2[im];
    S.ndf = c.out.track_ndf[im];
  }
  const tpc_merged& o = m.out;
  const size_t cap = o.capacity;
  o.merged_first[slot] = i1; o.merged_nseg[slot] = n_seg; o.merged_nhits[slot] = n_hits; o.merged_nfit[slot] = n_fit;
  o.merged_sector[slot] = (uint32_t)sector; o.merged_ndf[slot] = S.ndf;
  o.merged_x[slot] = x; o.merged_chi2[slot] = S.chi2;
  float* par = o.merged_par + slot;
  par[0] = S.y; par[cap] = S.z; par[2 * cap] = S.s; par[3 * cap] = S.t; par[4 * cap] = S.q;
  float* cv = o.merged_cov + slot;
  cv[0] = S.c00; cv[cap] = S.c10; cv[2 * cap] = S.c11; cv[3 * cap] = S.c20; cv[4 * cap] = S.c21; cv[5 * cap] = S.c22;
  cv[6 * cap] = S.c30; cv[7 * cap] = S.c31; cv[8 * cap] = S.c32; cv[9 * cap] = S.c33;
  cv[10 * cap] = S.c40; cv[11 * cap] = S.c41; cv[12 * cap] = S.c42; cv[13 * cap] = S.c43; cv[14 * cap] = S.c44;
}

}  // namespace tpc
