// Sector-segment merger and final refit (the tracker "merges the
// tracks segments afterward"; L140: the Kalman refit the paper wants on the GPU next to the tracker, so that
// track segments never cross PCIe between the two).  docs/ARITH_SPEC.md section 9: ROTATE (R1..R7), matching
// (G1..G7), refit (F1..F3).  Runs behind a7 on the arrays the tracker left in its workspace: the bin-sorted
// (y,z), the row maps with their kept hits flagged by k_resolve, and what k_select_output noted per track.
//   k_merge_ends    G1   one thread per sector track: the fitted helix at the row of its outermost kept hit
//   k_merge_row_scan / k_merge_row_fill   the tracks of every task listed by the row of their first kept hit, so
//                        that the candidates of G2 are one contiguous run of that list
//   k_merge_match   G2..G5  one thread per track: the full test (rotate, transport, chi2) on every candidate, once
//                        per pair; its best continuation is kept, the best segment a track continues is an
//                        atomicMin over (chi2, first-hit gid) - order-free
//   k_merge_link    G6   mutual choices become links
//   k_merge_heads   G7   chain heads are numbered in track order (ordered compaction)
//   k_merge_refit   F1..F3  persistent, one lane per chain: the filter pass from the outermost hit inwards,
//                        rotating the state where the chain changes sector
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
  int32_t n_slices;           // SPEC 11: slices per frame (1: events)
  float ca, sa;               // cos, sin of the sector pitch (SPEC 9 tables)
  // merge workspace (device)
  float4* ends;               // [cap][6]   G1
  uint32_t* row_cnt;          // [n_tr + 1] tracks whose first kept hit is in (task,row); zeroed per call
  uint32_t* row_start;        // [n_tr + 1] exclusive scan of row_cnt
  uint32_t* row_fill;         // [n_tr + 1] running fill position; zeroed per call
  uint32_t* row_list;         // [cap] track indices ordered by (task, first row)
  int32_t* best_out;          // [cap] G5: the j track i would continue into
  float* best_chi;            // [cap] its chi2
  unsigned long long* key_in; // [cap] G5, seen from j: min over i of chi2 bits << 32 | gid of i's first hit; all ones = none
  unsigned long long* scan;   // look-back state of the chain-head numbering, [tiles]
  uint32_t* ticket;           // [2] tile ticket of k_merge_heads, queue head of k_merge_refit
};

// sector tracks the merger works on: none if the tracker reported an overflow (their arrays may be incomplete)
__device__ __forceinline__ uint32_t merge_n_tracks(const Ctx& c, const MergeCtx& m) {
  if (c.out.header[2] != 0u) return 0u;
  return min(min(c.out.header[0], c.out.track_capacity), m.out.capacity);
}

// G1: the fitted helix at the row of the outermost kept hit; the track is counted in the bucket of its first row
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
  m.out.seg_next[i] = -1;
  m.out.seg_prev[i] = -1;
  m.best_out[i] = -1;
  atomicAdd(&m.row_cnt[c.out.track_task[i] * (uint32_t)c.n_rows + (rows & 0xFFFFu)], 1u);
}

// exclusive scan of row_cnt (one block: n_tasks * n_rows entries, 92 k for 16 events)
__global__ void __launch_bounds__(1024) k_merge_row_scan(const Ctx c, const MergeCtx m) {
  __shared__ uint32_t s_warp[33];
  const uint32_t n = c.n_tr + 1u, per = (n + 1023u) / 1024u;
  const uint32_t b0 = min(threadIdx.x * per, n), b1 = min(b0 + per, n);
  uint32_t sum = 0u;
  for (uint32_t k = b0; k < b1; ++k) sum += m.row_cnt[k];
  uint32_t total;
  uint32_t run = block_exclusive_scan(sum, s_warp, &total);
  for (uint32_t k = b0; k < b1; ++k) { const uint32_t v = m.row_cnt[k]; m.row_start[k] = run; run += v; }
}

// tracks into their (task, first row) bucket; the order inside a bucket is whatever the atomics give - every use
// of the list takes an order-free minimum
__global__ void __launch_bounds__(kMergeThreads) k_merge_row_fill(const Ctx c, const MergeCtx m) {
  const uint32_t n_trk = merge_n_tracks(c, m);
  const uint32_t i = blockIdx.x * kMergeThreads + threadIdx.x;
  if (i >= n_trk) return;
  const uint32_t b = c.out.track_task[i] * (uint32_t)c.n_rows + (c.out_rows[i] & 0xFFFFu);
  m.row_list[m.row_start[b] + atomicAdd(&m.row_fill[b], 1u)] = i;
}

// G3, G4 for the pair (inner i -> outer j) in direction d (0: same sector, neighbouring slice - no ROTATE);
// Q = outer end of i at X[rl_i].  Returns chi or +inf.
__device__ __forceinline__ float merge_chi(const Ctx& c, const MergeCtx& m, TrackState Q, float xq, int d, uint32_t j) {
  const float kInf = __int_as_float(0x7f800000);
  if (d != 0 && !rotate_state(Q, xq, m.ca, d > 0 ? m.sa : -m.sa, c.a, c.prm.max_sinphi)) return kInf;
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

// G2..G5.  One thread per track i: in both directions the candidates - tracks of the neighbouring sector whose
// first row lies in (rl_i, rl_i + gap] - are one contiguous run of row_list.  Every pair is tested once: i keeps
// its best j, and j's best i is the minimum of chi2 bits << 32 | first-hit gid taken with atomicMin (chi2 >= 0,
// so its bits order like its value; the minimum does not depend on the order of the atomics).
__global__ void __launch_bounds__(kMergeThreads) k_merge_match(const Ctx c, const MergeCtx m) {
  const uint32_t n_trk = merge_n_tracks(c, m);
  const int nh = m.n_half, n_sl = m.n_slices;
  const int n_dir = nh >= 3 ? 2 : (nh == 2 ? 1 : 0);
  const uint32_t t = blockIdx.x * kMergeThreads + threadIdx.x;
  if ((n_dir == 0 && n_sl < 2) || t >= n_trk) return;
  const int ns = c.n_sectors, n_rows = c.n_rows;
  const int rl_t = (int)(c.out_rows[t] >> 16);
  if (rl_t + 1 >= n_rows) return;                                                   // nothing starts above the last row
  TrackState E;
  if (!load_end(m.ends + (size_t)t * 6, E)) return;
  const uint32_t task = c.out.track_task[t];
  const int sec = (int)(task % (uint32_t)ns), side = sec / nh, f = sec - side * nh;
  const uint32_t slice = (task / (uint32_t)ns) % (uint32_t)n_sl;                    // SPEC 11
  const uint32_t g_t = c.out.hit_cluster[c.out.track_hit_begin[t]];
  const float x_end = c.X[rl_t];
  int32_t best = -1;
  float chi_best = 0.0f;
  uint32_t gid_best = 0u;
  // candidate tasks: the neighbouring sectors of the same slice (d = +1, -1), the same sector of the neighbouring
  // slices (d = 0)
  for (int k = 0; k < 4; ++k) {
    int d;
    uint32_t tj;
    if (k < 2) {
      if (k >= n_dir) continue;
      d = k == 0 ? +1 : -1;
      tj = task - (uint32_t)sec + (uint32_t)(side * nh + (f + d + nh) % nh);
    } else {
      d = 0;
      if (k == 2) { if (slice + 1u >= (uint32_t)n_sl) continue; tj = task + (uint32_t)ns; }
      else { if (slice == 0u) continue; tj = task - (uint32_t)ns; }
    }
    const uint32_t b0 = tj * (uint32_t)n_rows + (uint32_t)(rl_t + 1);               // G2: rl_i < rf_j <= rl_i + gap
    const uint32_t b1 = tj * (uint32_t)n_rows + (uint32_t)min(rl_t + m.max_row_gap, n_rows - 1) + 1u;
    for (uint32_t q = m.row_start[b0], qe = m.row_start[b1]; q < qe; ++q) {
      const uint32_t j = m.row_list[q];
      const float chi = merge_chi(c, m, E, x_end, d, j);                            // G3, G4
      if (!(chi < m.chi2_max)) continue;
      const uint32_t g = c.out.hit_cluster[c.out.track_hit_begin[j]];
      if (best < 0 || chi < chi_best || (chi == chi_best && g < gid_best)) { best = (int32_t)j; chi_best = chi; gid_best = g; }  // G5
      atomicMin(&m.key_in[j], ((unsigned long long)__float_as_uint(chi) << 32) | (unsigned long long)g_t);
    }
  }
  m.best_out[t] = best;
  m.best_chi[t] = chi_best;
}

// G6: i -> j is a link iff j is i's best and i is j's best (its key is the minimum j has seen).
__global__ void __launch_bounds__(kMergeThreads) k_merge_link(const Ctx c, const MergeCtx m) {
  const uint32_t n_trk = merge_n_tracks(c, m);
  const uint32_t t = blockIdx.x * kMergeThreads + threadIdx.x;
  if (t >= n_trk) return;
  const int32_t j = m.best_out[t];
  if (j < 0) return;
  const uint32_t g_t = c.out.hit_cluster[c.out.track_hit_begin[t]];
  const unsigned long long mine = ((unsigned long long)__float_as_uint(m.best_chi[t]) << 32) | (unsigned long long)g_t;
  if (m.key_in[j] != mine) return;
  m.out.seg_next[t] = j;
  m.out.seg_prev[j] = (int32_t)t;
  atomicAdd(&m.out.header[1], 1u);
}

// G7: the heads of chains (no previous segment) are numbered in track order (block scan + chained scan with
// decoupled look-back): merged track `slot` starts with sector track merged_first[slot].
__global__ void __launch_bounds__(kMergeThreads) k_merge_heads(const Ctx c, const MergeCtx m) {
  __shared__ uint32_t s_warp[33];
  __shared__ uint32_t s_tile;
  __shared__ unsigned long long s_prefix;
  if (threadIdx.x == 0) s_tile = atomicAdd(&m.ticket[0], 1u);
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
  if (head) m.out.merged_first[(uint32_t)s_prefix + excl] = i1;
  if (threadIdx.x == 0 && tile == gridDim.x - 1) m.out.header[0] = (uint32_t)s_prefix + total;
}

// F1..F3.  Persistent, one LANE per chain, a lane that has finished takes the next chain from the queue (chains
// hold 10..500 hits).  Every loop iteration is one pad row of the lane's current segment: map entry two rows ahead
// and (y,z) one row ahead are requested before the arithmetic (as in k_trk_refit); a row without a kept hit costs
// the lane an idle iteration.  The state is turned (ROTATE) where the chain changes sector.
constexpr int kMergeRefitBlocksPerSm = 6;

__global__ void __launch_bounds__(kMergeThreads, kMergeRefitBlocksPerSm) k_merge_refit(const Ctx c, const MergeCtx m) {
  extern __shared__ __align__(16) float sX[];  // [n_rows]
  constexpr unsigned FULL = 0xffffffffu;
  const int n_rows = c.n_rows, ns = c.n_sectors, nh = m.n_half, lane = (int)threadIdx.x & 31;
  for (int r = (int)threadIdx.x; r < n_rows; r += (int)blockDim.x) sX[r] = c.X[r];
  __syncthreads();
  const uint32_t n_merged = min(m.out.header[0], m.out.capacity);
  const float a = c.a, max_sin = c.prm.max_sinphi, sy2 = c.sy2, sz2 = c.sz2;
  const size_t stride = map_stride(n_rows);
  TrackState S;
  zero_state(S);
  float x = 0.0f;
  uint32_t slot = 0u, i1 = 0u, n_seg = 0u, n_hits = 0u, n_fit = 0u;
  int32_t k = -1;                       // current segment (sector track)
  const uint32_t* map = c.trk_hits;
  int r = 0, r_lo = 0, sec_k = 0, sector = 0;
  uint32_t e_cur = kNoHit, e_next = kNoHit;
  float2 p_cur = make_float2(0.0f, 0.0f);
  bool fit = false;                     // the refit is still running (F2 has not stopped)
  int st = LN_IDLE;
  TicketPool pool{0u, 0u};
  auto kept = [](uint32_t e) { return e != kNoHit && (e & kOwnedBit) != 0u; };
  auto open_segment = [&](int32_t seg) {  // rows and map of sector track `seg`, its outermost row first
    const uint32_t rows = c.out_rows[seg];
    map = c.trk_hits + (size_t)c.out_trk[seg] * stride;
    r = (int)(rows >> 16); r_lo = (int)(rows & 0xFFFFu);
    sec_k = (int)(c.out.track_task[seg] % (uint32_t)ns);
    e_cur = map[r];
    e_next = r - 1 >= r_lo ? map[r - 1] : kNoHit;
    if (kept(e_cur)) p_cur = c.yz[e_cur & ~kOwnedBit];
  };
  while (true) {
    const unsigned need = __ballot_sync(FULL, st == LN_IDLE);
    if (need) {
      const uint32_t tk = pool_take_seq(pool, &m.ticket[1], need, lane);
      if (st == LN_IDLE) {
        if (tk >= n_merged) {
          st = LN_EXIT;
        } else {
          slot = tk;
          i1 = m.out.merged_first[slot];
          uint32_t im = i1;
          n_seg = 1u; n_hits = c.out.track_nhits[i1];
          for (int32_t q = m.out.seg_next[i1]; q >= 0; q = m.out.seg_next[q]) { im = (uint32_t)q; ++n_seg; n_hits += c.out.track_nhits[q]; }
          n_fit = 0u;
          k = (int32_t)im;
          open_segment(k);
          sector = sec_k;
          x = sX[r];
          fit = load_end(m.ends + (size_t)im * 6, S);
          if (fit) {                                                                   // F1
            const float f = c.prm.turn_cov_scale;
            S.c00 *= f; S.c10 *= f; S.c11 *= f; S.c20 *= f; S.c21 *= f; S.c22 *= f; S.c30 *= f; S.c31 *= f;
            S.c32 *= f; S.c33 *= f; S.c40 *= f; S.c41 *= f; S.c42 *= f; S.c43 *= f; S.c44 *= f;
            S.chi2 = 0.0f; S.ndf = -5;
          } else {  // no outer end, no refit: the segment's own fit
            load_track_state(c.out, im, S, x);
            S.chi2 = c.out.track_chi2[im];
            S.ndf = c.out.track_ndf[im];
          }
          st = LN_RUN;
        }
      }
    }
    if (__ballot_sync(FULL, st != LN_EXIT) == 0u) break;
    const bool run = st == LN_RUN && fit;
    if (run && r < r_lo) {              // the segment is exhausted: the next one inwards, or the end of the chain
      k = m.out.seg_prev[k];
      if (k >= 0) open_segment(k);
    }
    const bool step = run && k >= 0;
    const bool use = step && kept(e_cur);
    uint32_t e_n2 = kNoHit;
    float2 p_next = make_float2(0.0f, 0.0f);
    bool ok = true;
    if (step) {
      if (kept(e_next)) p_next = c.yz[e_next & ~kOwnedBit];
      if (r - 2 >= r_lo) e_n2 = map[r - 2];
    }
    if (use) {                                                                         // F2
      if (sec_k != sector) {
        const int d = (sector % nh + 1) % nh == sec_k % nh ? +1 : -1;
        ok = rotate_state(S, x, m.ca, d > 0 ? m.sa : -m.sa, a, max_sin);
        if (ok) sector = sec_k;
      }
      const float xr = sX[r];
      if (ok && x != xr) {
        ok = transport(S, xr - x, a, max_sin);
        if (ok) x = xr;
      }
    }
    __syncwarp();
    if (use && ok) {
      update_hit(S, p_cur.x, p_cur.y, sy2, sz2);
      ++n_fit;
    }
    if (step) { e_cur = e_next; p_cur = p_next; e_next = e_n2; --r; }
    if (use && !ok) fit = false;                                                       // F2: the refit stops here
    if (st == LN_RUN && (!fit || k < 0)) {                                             // F3
      const tpc_merged& o = m.out;
      const size_t cap = o.capacity;
      o.merged_nseg[slot] = n_seg; o.merged_nhits[slot] = n_hits; o.merged_nfit[slot] = n_fit;
      o.merged_sector[slot] = (uint32_t)sector; o.merged_ndf[slot] = S.ndf;
      o.merged_x[slot] = x; o.merged_chi2[slot] = S.chi2;
      float* par = o.merged_par + slot;
      par[0] = S.y; par[cap] = S.z; par[2 * cap] = S.s; par[3 * cap] = S.t; par[4 * cap] = S.q;
      float* cv = o.merged_cov + slot;
      cv[0] = S.c00; cv[cap] = S.c10; cv[2 * cap] = S.c11; cv[3 * cap] = S.c20; cv[4 * cap] = S.c21; cv[5 * cap] = S.c22;
      cv[6 * cap] = S.c30; cv[7 * cap] = S.c31; cv[8 * cap] = S.c32; cv[9 * cap] = S.c33;
      cv[10 * cap] = S.c40; cv[11 * cap] = S.c41; cv[12 * cap] = S.c42; cv[13 * cap] = S.c43; cv[14 * cap] = S.c44;
      st = LN_IDLE;
    }
  }
}

}  // namespace tpc
