// a5  tracklet constructor ("Kalman filter for track fitting and
// track following"; L123: "in the track following phase, 1 GPU thread handles 1
// track").  docs/ARITH_SPEC.md sections 5 (track model) and 6 (K1..K7).
//
// One LANE per tracklet, the whole filter state (5 parameters, 15 covariance
// entries, chi2) in registers.  The life of a tracklet is cut where the KIND of
// its row steps changes, and every part is its own persistent kernel, so that
// the 32 lanes of a warp always execute the same kind of step:
//   k_trk_chain   K1 + K2   seed, then the fit along the link chain   (hit known, no search)
//   k_trk_up      K3 + K4   up pass and turn-around                   (every step searches)
//   k_trk_refit   K5 (a)    down pass over the rows that have a hit   (hit known, no search)
//   k_trk_finish  K5 (b), K6       rest of the down pass (searches below firstRow or in a hole of
//                                  the map), finish
// Between two kernels the tracklet rests in its record (Ctx::trk_rec, 128 bytes).  In every kernel
// a lane whose tracklet has ended takes the next one from a queue (tickets drawn 32 at a time per
// warp), so the lanes stay busy although tracklets live for very different numbers of row steps;
// the record of the next tracklet is copied to the lane's shared-memory slot with cp.async while
// the lane runs the last step of the current one, so no warp ever waits for a fetch.  A row step is
//     transport -> choose the hit (chain link / row map / search) -> update
// with the loads that do not depend on the transported state issued before the transport.  The
// row -> hit map of a tracklet is its row of Ctx::trk_hits in global memory (idx per pad row or
// kNoHit).  Registers alone bound the tracklets in flight.
#pragma once
#include "device_common.cuh"

namespace tpc {

constexpr int kTrackletThreads = 128;
#ifndef TPC_FIT_BLOCKS
#define TPC_FIT_BLOCKS 7
#endif
#ifndef TPC_SEARCH_BLOCKS
#define TPC_SEARCH_BLOCKS 6
#endif
constexpr int kFitBlocksPerSm = TPC_FIT_BLOCKS;     // k_trk_chain, k_trk_refit: registers per thread <= 65536 / (128 * 8) = 64
constexpr int kSearchBlocksPerSm = TPC_SEARCH_BLOCKS;  // k_trk_up, k_trk_finish:  <= 85

struct TrackState {
  float y, z, s, t, q;  // SPEC 5: y, z, sinphi, dz/dl, q/pT
  float c00, c10, c11, c20, c21, c22, c30, c31, c32, c33, c40, c41, c42, c43, c44;
  float chi2;
  int32_t ndf;
};

// SPEC 5.1 P1..P24.  dx = X[target] - X[current].  Fails (state untouched) beyond max_sinphi.
__device__ __forceinline__ bool transport(TrackState& S, float dx, float a, float max_sinphi) {
  const float y = S.y, z = S.z, s = S.s, t = S.t, q = S.q;
  const float k = a * q;                                   // P2
  const float s1 = s + k * dx;                             // P3
  if (!(fabsf(s) <= max_sinphi && fabsf(s1) <= max_sinphi)) return false;  // P4
  const float c = sqrtf(1.0f - s * s);                     // P5
  const float c1 = sqrtf(1.0f - s1 * s1);
  const float cs = c + c1;                                 // P6
  const float tt = (s + s1) / cs;                          // P7
  const float dy = dx * tt;                                // P8
  const float dl = dx * sqrtf(1.0f + tt * tt);             // P9
  const float u = (0.5f * k) * dl;                         // P10
  const float u2 = u * u;
  const float A1 = 0.16666667f, A2 = 0.075f, A3 = 0.044642857f;
  const float dS = dl * (1.0f + u2 * (A1 + u2 * (A2 + u2 * A3)));  // P11
  const float g = s * dy + c * dx;                         // P13
  const float cc = c * c1;                                 // P14
  const float f02 = g / cc;                                // P15
  const float f04 = ((a * dx) * g) / (c1 * cs);            // P16
  const float f12 = (t * dy) / cc;                         // P17
  const float f13 = dS;                                    // P18
  const float f14 = ((t * a) * ((0.5f * dx) * dy)) / cc;   // P19
  const float f24 = a * dx;                                // P20
  const float c00 = S.c00, c10 = S.c10, c11 = S.c11, c20 = S.c20, c21 = S.c21, c22 = S.c22, c30 = S.c30,
              c31 = S.c31, c32 = S.c32, c33 = S.c33, c40 = S.c40, c41 = S.c41, c42 = S.c42, c43 = S.c43,
              c44 = S.c44;
  // P21 row 0 of M = F*C
  const float m00 = c00 + f02 * c20 + f04 * c40;
  const float m02 = c20 + f02 * c22 + f04 * c42;
  const float m04 = c40 + f02 * c42 + f04 * c44;
  // P22 row 1
  const float m10 = c10 + f12 * c20 + f13 * c30 + f14 * c40;
  const float m11 = c11 + f12 * c21 + f13 * c31 + f14 * c41;
  const float m12 = c21 + f12 * c22 + f13 * c32 + f14 * c42;
  const float m13 = c31 + f12 * c32 + f13 * c33 + f14 * c43;
  const float m14 = c41 + f12 * c42 + f13 * c43 + f14 * c44;
  // P23 row 2
  const float m20 = c20 + f24 * c40;
  const float m21 = c21 + f24 * c41;
  const float m22 = c22 + f24 * c42;
  const float m23 = c32 + f24 * c43;
  const float m24 = c42 + f24 * c44;
  // P24 C' = M*F^T
  S.c00 = m00 + f02 * m02 + f04 * m04;
  S.c10 = m10 + f02 * m12 + f04 * m14;
  S.c11 = m11 + f12 * m12 + f13 * m13 + f14 * m14;
  S.c20 = m20 + f02 * m22 + f04 * m24;
  S.c21 = m21 + f12 * m22 + f13 * m23 + f14 * m24;
  S.c22 = m22 + f24 * m24;
  S.c30 = c30 + f02 * c32 + f04 * c43;
  S.c31 = c31 + f12 * c32 + f13 * c33 + f14 * c43;
  S.c32 = c32 + f24 * c43;
  S.c40 = c40 + f02 * c42 + f04 * c44;
  S.c41 = c41 + f12 * c42 + f13 * c43 + f14 * c44;
  S.c42 = c42 + f24 * c44;
  S.y = y + dy;                                            // P12
  S.z = z + dS * t;
  S.s = s1;
  return true;
}

// SPEC 5.2 UPDATE(0, m, sy2) then UPDATE(1, m, sz2)
__device__ __forceinline__ void update_hit(TrackState& S, float ym, float zm, float sy2, float sz2) {
  {
    const float w = 1.0f / (S.c00 + sy2);                  // U1
    const float res = ym - S.y;                            // U2
    const float o0 = S.c00, o1 = S.c10, o2 = S.c20, o3 = S.c30, o4 = S.c40;  // U3
    const float k0 = o0 * w, k1 = o1 * w, k2 = o2 * w, k3 = o3 * w, k4 = o4 * w;  // U4
    S.y = S.y + k0 * res; S.z = S.z + k1 * res; S.s = S.s + k2 * res;        // U5
    S.t = S.t + k3 * res; S.q = S.q + k4 * res;
    S.c00 = S.c00 - k0 * o0;                               // U6
    S.c10 = S.c10 - k1 * o0; S.c11 = S.c11 - k1 * o1;
    S.c20 = S.c20 - k2 * o0; S.c21 = S.c21 - k2 * o1; S.c22 = S.c22 - k2 * o2;
    S.c30 = S.c30 - k3 * o0; S.c31 = S.c31 - k3 * o1; S.c32 = S.c32 - k3 * o2; S.c33 = S.c33 - k3 * o3;
    S.c40 = S.c40 - k4 * o0; S.c41 = S.c41 - k4 * o1; S.c42 = S.c42 - k4 * o2; S.c43 = S.c43 - k4 * o3;
    S.c44 = S.c44 - k4 * o4;
    S.chi2 = S.chi2 + (res * res) * w;                     // U7
  }
  {
    const float w = 1.0f / (S.c11 + sz2);
    const float res = zm - S.z;
    const float o0 = S.c10, o1 = S.c11, o2 = S.c21, o3 = S.c31, o4 = S.c41;
    const float k0 = o0 * w, k1 = o1 * w, k2 = o2 * w, k3 = o3 * w, k4 = o4 * w;
    S.y = S.y + k0 * res; S.z = S.z + k1 * res; S.s = S.s + k2 * res;
    S.t = S.t + k3 * res; S.q = S.q + k4 * res;
    S.c00 = S.c00 - k0 * o0;
    S.c10 = S.c10 - k1 * o0; S.c11 = S.c11 - k1 * o1;
    S.c20 = S.c20 - k2 * o0; S.c21 = S.c21 - k2 * o1; S.c22 = S.c22 - k2 * o2;
    S.c30 = S.c30 - k3 * o0; S.c31 = S.c31 - k3 * o1; S.c32 = S.c32 - k3 * o2; S.c33 = S.c33 - k3 * o3;
    S.c40 = S.c40 - k4 * o0; S.c41 = S.c41 - k4 * o1; S.c42 = S.c42 - k4 * o2; S.c43 = S.c43 - k4 * o3;
    S.c44 = S.c44 - k4 * o4;
    S.chi2 = S.chi2 + (res * res) * w;
  }
  S.ndf += 2;
}


__device__ __forceinline__ float sqrt_approx(float v) {
  float r;
  asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}

// SPEC 5.3 SEARCH (H1..H6), exact and serial: one flat loop over the window, ties decided by gid.  The fast
// search below hands over to this one when it meets two valid clusters with the same distance.
__device__ __noinline__ int32_t search_row_serial(const float2* __restrict__ yz, const uint32_t* __restrict__ gid,
                                                  const uint32_t* bp, int ny, int iy0, int iy1, int n_zrows, float y,
                                                  float z, float hy2, float hz2, float ey, float ez) {
  bool have = false;
  float best = 0.0f;
  uint32_t bi = 0u;
  for (int r = 0; r < n_zrows; ++r, bp += ny) {
    for (uint32_t i = bp[iy0], e = bp[iy1]; i < e; ++i) {
      const float2 p = yz[i];
      const float dy = p.x - y, dz = p.y - z;                          // H3
      const float dy2 = dy * dy, dz2 = dz * dz;
      if (dy2 <= hy2 && dz2 <= hz2) {                                  // H4
        const float d = (dy2 * ez) + (dz2 * ey);                       // H5
        bool take = !have || d < best;                                 // H6
        if (have && d == best) take = gid[i] < gid[bi];
        if (take) { have = true; best = d; bi = i; }
      }
    }
  }
  return have ? (int32_t)bi : -1;
}

// SPEC 5.3 SEARCH in the row described by g; returns the idx of the best cluster or -1 and its (y,z) in
// best_p.  The window covers 1..4 bin rows in z, almost always 1 or 2: the four bin bounds of two rows
// are loaded together, then their candidates are read as ONE virtual range, kSearchUnroll at a time, all
// loads of a group in flight before the first is tested (the walk is latency bound) and the tests written
// without branches (lanes of a warp are at different candidates of different windows).
#ifndef TPC_SEARCH_UNROLL
#define TPC_SEARCH_UNROLL 2
#endif
constexpr int kSearchUnroll = TPC_SEARCH_UNROLL;

template <bool COUNT>
__device__ __forceinline__ int32_t search_row(const Ctx& c, const TrackState& S, const RowInfo g,
                                              float2& best_p, uint32_t& n_cand) {
  const float y = S.y, z = S.z;
  const float ey = S.c00 + c.sy2, ez = S.c11 + c.sz2;                 // H1
  const float hy2 = fminf(c.prm.accept_k2 * ey, c.smax2);              // H2
  const float hz2 = fminf(c.prm.accept_k2 * ez, c.smax2);
  // half widths of the grid window: acceleration only (SPEC 2), so the approximate square root (about 1 ulp) will
  // do - kGridMargin is four orders of magnitude larger than its error
  const float wy = sqrt_approx(fmaxf(hy2, 0.0f)) + kGridMargin, wz = sqrt_approx(fmaxf(hz2, 0.0f)) + kGridMargin;
  const int ny = info_ny(g), nz = info_nz(g);
  const int iy0 = bin_coord(y - wy, g.y0, g.inv, ny), iy1 = bin_coord(y + wy, g.y0, g.inv, ny) + 1;
  const int iz0 = bin_coord(z - wz, g.z0, g.inv, nz), iz1 = bin_coord(z + wz, g.z0, g.inv, nz);
  const uint32_t* bp = c.bins + g.bins_off + iz0 * ny;
  float best = __int_as_float(0x7f800000);  // +inf: a valid cluster at distance +inf counts as a tie
  float bx = 0.0f, bz = 0.0f;
  int32_t bi = -1;
  const int n_zrows = iz1 - iz0 + 1;
  bool tie = n_zrows > 2;  // a window over 3 or 4 bin rows (6 in a million) is left to the serial search as well
  {
    const bool two = n_zrows > 1;
    const uint32_t i1 = __ldg(bp + iy0), e1 = __ldg(bp + iy1);
    const uint32_t i2 = two ? __ldg(bp + ny + iy0) : 0u, e2 = two ? __ldg(bp + ny + iy1) : 0u;
    const uint32_t n1 = e1 - i1, n_tot = n1 + (e2 - i2);
    const uint32_t skip = i2 - e1;  // idx of candidate k >= n1 is i1 + k + skip
    if (COUNT) n_cand += n_tot;
    for (uint32_t k0 = 0u; k0 < n_tot; k0 += kSearchUnroll) {
      uint32_t idx[kSearchUnroll];
      float2 p[kSearchUnroll];
#pragma unroll
      for (int j = 0; j < kSearchUnroll; ++j) {
        const uint32_t k = k0 + j;
        idx[j] = i1 + k + (k < n1 ? 0u : skip);
        p[j] = k < n_tot ? c.yz[idx[j]] : make_float2(0.0f, 0.0f);
      }
#pragma unroll
      for (int j = 0; j < kSearchUnroll; ++j) {
        const float dy = p[j].x - y, dz = p[j].y - z;                  // H3
        const float dy2 = dy * dy, dz2 = dz * dz;
        const bool ok = (k0 + j < n_tot) & (dy2 <= hy2) & (dz2 <= hz2);  // H4
        const float d = (dy2 * ez) + (dz2 * ey);                       // H5
        const bool lt = ok & (d < best);                               // H6
        tie |= ok & (d == best);
        best = lt ? d : best;
        bi = lt ? (int32_t)idx[j] : bi;
        bx = lt ? p[j].x : bx;
        bz = lt ? p[j].y : bz;
      }
    }
  }
  if (tie) {  // the (y,z) is re-read here so that best_p never has its address taken (it stays in registers)
    bi = search_row_serial(c.yz, c.gid, bp, ny, iy0, iy1, n_zrows, y, z, hy2, hz2, ey, ez);
    if (bi >= 0) { const float2 p = c.yz[bi]; bx = p.x; bz = p.y; }
  }
  best_p = make_float2(bx, bz);
  return bi;
}


constexpr uint32_t kNoHit = 0xFFFFFFFFu;  // row map entry of a row without a hit

// Tracklet record (Ctx::trk_rec), 32 words: [0] x, [1..5] p, [6..20] C, [21] chi2, [22] ndf, [23] nHits,
// [24] firstRow, [25] lastRow, [26] rows packed (below), [27] task*n_rows, [28] ia, [29] ib, [30..31] unused.
// Words 0..25 are what the selector and the output read once k_trk_finish has stored them; between the
// kernels the record carries the tracklet.
//   pack = row_cur | (r_down + 1) << 10 | r0 << 20 | skip_up << 30       (n_rows <= 1024)
// row_cur = row the state is at, r_down = next row of the down pass (-1: none left), r0 = row of the start
// hit, skip_up = the chain fit ended with a failed transport (K2 -> K4).
//   ia, ib: what the next kernel would otherwise have to load after the record (a second round trip):
//   chain -> up: ia = hit of lastRow;  up -> refit: ia = map[r_down], ib = map[r_down - 1];
//   refit -> finish: ia = map[r_down]   (kNoHit where the row is below r0)
__device__ __forceinline__ uint32_t pack_rows(int row_cur, int r_down, int r0, bool skip_up) {
  return (uint32_t)row_cur | ((uint32_t)(r_down + 1) << 10) | ((uint32_t)r0 << 20) | (skip_up ? 1u << 30 : 0u);
}
#ifdef TPC_STREAM_STORES
#define TPC_ST4(p, v) __stcs((p), (v))
#define TPC_ST1(p, v) __stcs((p), (v))
#else
#define TPC_ST4(p, v) (*(p) = (v))
#define TPC_ST1(p, v) (*(p) = (v))
#endif
__device__ __forceinline__ void store_rec(float4* rec, const TrackState& S, float x, int n_hits, int first_row,
                                          int last_row, uint32_t pack, uint32_t tr_base, uint32_t ia, uint32_t ib) {
  TPC_ST4(rec + 0, make_float4(x, S.y, S.z, S.s));
  TPC_ST4(rec + 1, make_float4(S.t, S.q, S.c00, S.c10));
  TPC_ST4(rec + 2, make_float4(S.c11, S.c20, S.c21, S.c22));
  TPC_ST4(rec + 3, make_float4(S.c30, S.c31, S.c32, S.c33));
  TPC_ST4(rec + 4, make_float4(S.c40, S.c41, S.c42, S.c43));
  TPC_ST4(rec + 5, make_float4(S.c44, S.chi2, __int_as_float(S.ndf), __int_as_float(n_hits)));
  TPC_ST4(rec + 6, make_float4(__int_as_float(first_row), __int_as_float(last_row), __uint_as_float(pack),
                               __uint_as_float(tr_base)));
  TPC_ST4(rec + 7, make_float4(__uint_as_float(ia), __uint_as_float(ib), 0.0f, 0.0f));
}
// rec: the lane's shared-memory copy of the record
__device__ __forceinline__ void load_rec(const float4* rec, TrackState& S, int& n_hits, int& first_row,
                                         int& last_row, uint32_t& pack, uint32_t& tr_base, uint32_t& ia,
                                         uint32_t& ib) {
  const float4 a0 = rec[0], a1 = rec[1], a2 = rec[2], a3 = rec[3], a4 = rec[4], a5 = rec[5], a6 = rec[6], a7 = rec[7];
  S.y = a0.y; S.z = a0.z; S.s = a0.w;
  S.t = a1.x; S.q = a1.y; S.c00 = a1.z; S.c10 = a1.w;
  S.c11 = a2.x; S.c20 = a2.y; S.c21 = a2.z; S.c22 = a2.w;
  S.c30 = a3.x; S.c31 = a3.y; S.c32 = a3.z; S.c33 = a3.w;
  S.c40 = a4.x; S.c41 = a4.y; S.c42 = a4.z; S.c43 = a4.w;
  S.c44 = a5.x; S.chi2 = a5.y; S.ndf = __float_as_int(a5.z); n_hits = __float_as_int(a5.w);
  first_row = __float_as_int(a6.x); last_row = __float_as_int(a6.y);
  pack = __float_as_uint(a6.z); tr_base = __float_as_uint(a6.w);
  ia = __float_as_uint(a7.x); ib = __float_as_uint(a7.y);
}

// ---- the queue of a tracklet kernel -------------------------------------------------------------------
// Ticket k stands for tracklet perm[k] (Ctx::trk_perm, the queue order built in front of every kernel, below).
// The order only does its work if a ticket is STARTED soon after it is drawn: a warp that drew 32 tickets at a
// time would sit on them for about 50 row steps (its lanes end 0.6 tracklets per step) and start them up to 50
// rows behind the wavefront they belong to.  So a warp keeps a small reserve, half a batch to one and a half batches of
// tickets in the registers of its lanes (lane j holds entry j of a ring of 32), and refills it in two steps that
// nobody waits for: iteration i asks for the next batch of tickets (one atomic, lane 0); iteration i + 1
// loads their perm[] entries into the ring; from iteration i + 2 on they are handed out by shuffle.  A lane that
// finds the reserve empty stays idle for an iteration.  A ticket >= the number of tracklets becomes kQueueEnd.
// Batch per kernel (0 chain fit ... 3 rest of the down pass), from a sweep on 16 central events: the searching kernels
// want the tightest wavefront (4; 2 starves the lanes, 8 and 16 are 3 % and 7 % slower), the chain fit, whose
// tracklets live for 26 steps only, starves below 16.  The reserve is refilled below half a batch.
#ifndef TPC_QUEUE_BATCH0
#define TPC_QUEUE_BATCH0 16
#endif
#ifndef TPC_QUEUE_BATCH1
#define TPC_QUEUE_BATCH1 4
#endif
#ifndef TPC_QUEUE_BATCH2
#define TPC_QUEUE_BATCH2 8
#endif
#ifndef TPC_QUEUE_BATCH3
#define TPC_QUEUE_BATCH3 4
#endif
__host__ __device__ constexpr uint32_t queue_batch_of(int kind) {
  return kind == 0 ? TPC_QUEUE_BATCH0 : kind == 1 ? TPC_QUEUE_BATCH1 : kind == 2 ? TPC_QUEUE_BATCH2 : TPC_QUEUE_BATCH3;
}
constexpr uint32_t kQueueEnd = 0xFFFFFFFFu;
struct TrackletQueue {
  uint32_t perm;       // lane j: tracklet of ring entry j, or kQueueEnd
  uint32_t head, cnt;  // entries head .. head + cnt - 1 (mod 32) are waiting        (the same in all lanes)
  uint32_t base;       // lane 0: first ticket of the batch asked for in the last iteration
  bool asked;          // such a batch exists                                        (the same in all lanes)
};
// Start of a kernel: the first 32 tickets of the warp at once.
__device__ __forceinline__ void queue_open(TrackletQueue& q, uint32_t* head, const uint32_t* __restrict__ perm,
                                           uint32_t n_trk, int lane) {
  uint32_t base = 0u;
  if (lane == 0) base = atomicAdd(head, 32u);
  base = __shfl_sync(0xffffffffu, base, 0);
  const uint32_t k = base + (uint32_t)lane;
  q.perm = k < n_trk ? __ldg(perm + k) : kQueueEnd;
  q.head = 0u; q.cnt = 32u; q.base = 0u; q.asked = false;
}
// One call per loop iteration by the whole warp; `need`: the lanes that want a tracklet.  Returns true in a lane
// that got one (t_out; kQueueEnd: the queue is empty).
template <int KIND>
__device__ __forceinline__ bool queue_step(TrackletQueue& q, uint32_t* head, const uint32_t* __restrict__ perm,
                                           uint32_t n_trk, unsigned need, int lane, uint32_t& t_out) {
  constexpr uint32_t kQueueBatch = queue_batch_of(KIND), kQueueLow = kQueueBatch / 2u;
  static_assert(kQueueBatch + kQueueLow <= 32u && kQueueBatch >= 1u, "the ring has 32 entries");
  const uint32_t n_need = (uint32_t)__popc(need), rank = (uint32_t)__popc(need & ((1u << lane) - 1u));
  const uint32_t n_give = min(n_need, q.cnt);
  bool got = false;
  if (n_give) {  // hand out (entries loaded in earlier iterations only: nothing waits for a load here)
    t_out = __shfl_sync(0xffffffffu, q.perm, (int)((q.head + rank) & 31u));
    got = ((need >> lane) & 1u) != 0u && rank < n_give;
    q.head = (q.head + n_give) & 31u;
    q.cnt -= n_give;
  }
  if (q.asked) {  // the batch asked for in the last iteration: its perm[] entries go behind the waiting ones
    const uint32_t base = __shfl_sync(0xffffffffu, q.base, 0);
    const uint32_t j = ((uint32_t)lane - (q.head + q.cnt)) & 31u;
    if (j < kQueueBatch) {
      const uint32_t k = base + j;
      q.perm = k < n_trk ? __ldg(perm + k) : kQueueEnd;
    }
    q.cnt += kQueueBatch;
    q.asked = false;
  }
  if (q.cnt <= kQueueLow) {  // ask for the next batch
    if (lane == 0) q.base = atomicAdd(head, kQueueBatch);
    q.asked = true;
  }
  return got;
}
// The same queue without a permutation (ticket k is item k): the merger's refit.
constexpr uint32_t kPoolBatch = 32;
struct TicketPool { uint32_t next, end; };
__device__ __forceinline__ uint32_t pool_take_seq(TicketPool& p, uint32_t* head, unsigned need, int lane) {
  const uint32_t cnt = (uint32_t)__popc(need), have = p.end - p.next;
  const uint32_t rank = (uint32_t)__popc(need & ((1u << lane) - 1u));
  if (cnt <= have) {
    const uint32_t tk = p.next + rank;
    p.next += cnt;
    return tk;
  }
  uint32_t base = 0u;
  if (lane == 0) base = atomicAdd(head, kPoolBatch);
  base = __shfl_sync(0xffffffffu, base, 0);
  const uint32_t tk = rank < have ? p.next + rank : base + (rank - have);
  p.next = base + (cnt - have);
  p.end = base + kPoolBatch;
  return tk;
}
// Asynchronous copy of n16 x 16 bytes, global -> this lane's slot in shared memory (no register is the
// target, so the warp goes on; the lane reads the slot one loop iteration later).
__device__ __forceinline__ void prefetch_slot(void* slot, const void* src, int n16) {
  const uint32_t d = smem_u32(slot);
  for (int k = 0; k < n16; ++k)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d + 16u * (uint32_t)k),
                 "l"(reinterpret_cast<const char*>(src) + 16 * k)
                 : "memory");
  asm volatile("cp.async.commit_group;" ::: "memory");
}
__device__ __forceinline__ void prefetch_wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }

enum LaneState { LN_IDLE = 0, LN_RUN = 1, LN_EXIT = 2 };
enum PrefetchState { PF_NONE = 0, PF_ISSUED = 1, PF_READY = 2, PF_DRAINED = 3 };  // ISSUED this iteration, READY from the next on

// The fetch protocol of a lane, the same in all four kernels (macro-free: three calls per loop iteration):
//   fetch_request: lanes that are idle, or run the last step of their tracklet (`ending`), and have nothing
//                  requested draw a ticket and start the copy of that tracklet's record to their slot;
//   (the kernel's own "consume" block turns an idle lane with a READY slot into a running one);
//   fetch_advance: ISSUED -> READY at the end of the iteration.
template <int KIND>
__device__ __forceinline__ void fetch_request(TrackletQueue& q, uint32_t* head, const uint32_t* perm, bool want, int lane,
                                              uint32_t n_trk, int& pf, uint32_t& t_next, void* slot, const void* src_base,
                                              size_t src_stride, int n16) {
  const unsigned need = __ballot_sync(0xffffffffu, want);
  if (need || q.asked) {
    uint32_t t = 0u;
    if (queue_step<KIND>(q, head, perm, n_trk, need, lane, t)) {
      if (t == kQueueEnd) {
        pf = PF_DRAINED;
      } else {
        t_next = t;
        prefetch_slot(slot, reinterpret_cast<const char*>(src_base) + (size_t)t * src_stride, n16);
        pf = PF_ISSUED;
      }
    }
  }
}

__device__ __forceinline__ void zero_state(TrackState& S) {
  S.y = S.z = S.s = S.t = S.q = 0.0f;
  S.c00 = S.c10 = S.c11 = S.c20 = S.c21 = S.c22 = S.c30 = S.c31 = S.c32 = S.c33 = 0.0f;
  S.c40 = S.c41 = S.c42 = S.c43 = S.c44 = 0.0f;
  S.chi2 = 0.0f; S.ndf = -5;
}

// shared memory of a tracklet kernel: [n_rows floats, padded to 16 bytes][blockDim.x slots of SLOT16 x 16 bytes]
__host__ __device__ inline size_t trk_smem_bytes(int n_rows, int slot16) {
  return (size_t)((n_rows + 3) & ~3) * sizeof(float) + (size_t)kTrackletThreads * slot16 * 16;
}

// ---------------------------------------------------------------------------
// Queue order of a5 (Ctx::trk_perm), built anew in front of each of the four kernels.
// A lane moves its tracklet one pad row per step, and a search reads the bins and clusters of that one
// row of its sector task.  Tracklets are numbered in (task, row of the start hit, bin) order; drawn in
// that order, the 2 200 tracklets of a task start together but at rows spread over the whole sector, so
// a grid row is read again only after its lines have left the L2 (44 % hits, 10 x the grid in DRAM reads),
// and the queue ends with tracklets that still have up to n_rows steps to go while the device idles.
// Instead the queue is sorted by the DIAGONAL
//     d = (rows the tracklet's first step is away from the row where the pass begins) + stagger * task
// (chain fit, up pass: counted from row 0 upwards; refit, rest of the down pass: from the last row
// downwards).  Lanes draw about one diagonal per step, so that the tracklets of a task still start when
// the others of that task reach their row: every task is swept by a wavefront a few rows wide, the tasks
// one after the other `stagger` rows apart, and a grid row is read by all its tracklets while it is in
// the L2.  The last diagonals hold the last rows of the last tasks only: short tracklets, no tail.
// The stagger follows from the tracklets per task and the lanes of the kernel (order_stagger, device_common.cuh).
// A counting sort by d: the kernel that finishes a tracklet in front of this one notes the task and the row
// where its next pass begins (order_note), k_order_count counts the tracklets of every diagonal, k_order_scan
// turns the counts into the first slot of every diagonal (one block), k_order_fill hands the slots out.  The
// order inside a diagonal is what the atomics give; it only decides which lane follows which tracklet - the
// result does not depend on it.  With no more tracklets than lanes the order is the identity.
// ---------------------------------------------------------------------------
constexpr int kOrderThreads = 256;
// One block per chunk of kOrderChunk consecutive tracklets (one or two tasks: a few hundred diagonals next to
// each other): the diagonals within kOrderWindow of the chunk's smallest are counted in shared memory first, so
// that global memory sees one atomic per block and diagonal; a tracklet beyond the window (a chunk over many
// small tasks) goes to global memory directly.
constexpr int kOrderItems = 8;
constexpr uint32_t kOrderChunk = kOrderThreads * kOrderItems;
constexpr uint32_t kOrderWindow = 2048;
__global__ void __launch_bounds__(kOrderThreads) k_order_count(const Ctx c, int kind, uint32_t lanes) {
  __shared__ uint32_t s_cnt[kOrderWindow];
  __shared__ uint32_t s_min;
  constexpr uint32_t kNone = 0xFFFFFFFFu;
  const uint32_t n_trk = *c.n_tracklets, n_keys = order_keys((uint32_t)c.n_rows, c.n_tasks);
  uint32_t* cnt = c.order_cnt + (size_t)(2 * kind) * n_keys;
  const uint32_t stagger = order_stagger(c, kind, lanes, n_trk);
  for (uint32_t k = threadIdx.x; k < kOrderWindow; k += kOrderThreads) s_cnt[k] = 0u;
  for (uint32_t t0 = blockIdx.x * kOrderChunk; t0 < n_trk; t0 += gridDim.x * kOrderChunk) {
    if (threadIdx.x == 0) s_min = kNone;
    __syncthreads();
    uint32_t key[kOrderItems];
    uint32_t kmin = kNone;
#pragma unroll
    for (int i = 0; i < kOrderItems; ++i) {
      const uint32_t t = t0 + (uint32_t)i * kOrderThreads + threadIdx.x;
      key[i] = t < n_trk ? order_diagonal(c, c.trk_key[t], stagger) : kNone;
      kmin = min(kmin, key[i]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
    if ((threadIdx.x & 31) == 0) atomicMin(&s_min, kmin);
    __syncthreads();
    kmin = s_min;
#pragma unroll
    for (int i = 0; i < kOrderItems; ++i) {
      if (key[i] == kNone) continue;
      if (key[i] - kmin < kOrderWindow) atomicAdd(&s_cnt[key[i] - kmin], 1u);
      else atomicAdd(&cnt[key[i]], 1u);
    }
    __syncthreads();
    for (uint32_t k = threadIdx.x; k < kOrderWindow; k += kOrderThreads) {
      const uint32_t n = s_cnt[k];
      if (n) { atomicAdd(&cnt[kmin + k], n); s_cnt[k] = 0u; }
    }
    __syncthreads();
  }
}
__global__ void __launch_bounds__(kOrderThreads) k_order_fill(const Ctx c, int kind, uint32_t lanes) {
  __shared__ uint32_t s_cnt[kOrderWindow];
  __shared__ uint32_t s_min;
  constexpr uint32_t kNone = 0xFFFFFFFFu;
  const uint32_t n_trk = *c.n_tracklets, n_keys = order_keys((uint32_t)c.n_rows, c.n_tasks);
  uint32_t* cursor = c.order_cnt + (size_t)(2 * kind + 1) * n_keys;
  const uint32_t stagger = order_stagger(c, kind, lanes, n_trk);
  if (n_trk <= lanes) {  // every tracklet starts at once whatever the order: keep the neighbours in (task, row, bin) together
    for (uint32_t t = blockIdx.x * kOrderThreads + threadIdx.x; t < n_trk; t += gridDim.x * kOrderThreads) c.trk_perm[t] = t;
    return;
  }
  for (uint32_t k = threadIdx.x; k < kOrderWindow; k += kOrderThreads) s_cnt[k] = 0u;
  for (uint32_t t0 = blockIdx.x * kOrderChunk; t0 < n_trk; t0 += gridDim.x * kOrderChunk) {
    if (threadIdx.x == 0) s_min = kNone;
    __syncthreads();
    uint32_t key[kOrderItems], rank[kOrderItems];
    uint32_t kmin = kNone;
#pragma unroll
    for (int i = 0; i < kOrderItems; ++i) {
      const uint32_t t = t0 + (uint32_t)i * kOrderThreads + threadIdx.x;
      key[i] = t < n_trk ? order_diagonal(c, c.trk_key[t], stagger) : kNone;
      kmin = min(kmin, key[i]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
    if ((threadIdx.x & 31) == 0) atomicMin(&s_min, kmin);
    __syncthreads();
    kmin = s_min;
#pragma unroll
    for (int i = 0; i < kOrderItems; ++i) {
      rank[i] = 0u;
      if (key[i] == kNone) continue;
      if (key[i] - kmin < kOrderWindow) {
        rank[i] = atomicAdd(&s_cnt[key[i] - kmin], 1u);
      } else {  // beyond the window: straight to global memory
        c.trk_perm[atomicAdd(&cursor[key[i]], 1u)] = t0 + (uint32_t)i * kOrderThreads + threadIdx.x;
        key[i] = kNone;
      }
    }
    __syncthreads();
    for (uint32_t k = threadIdx.x; k < kOrderWindow; k += kOrderThreads) {
      const uint32_t n = s_cnt[k];
      if (n) s_cnt[k] = atomicAdd(&cursor[kmin + k], n);
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kOrderItems; ++i) {
      const uint32_t t = t0 + (uint32_t)i * kOrderThreads + threadIdx.x;
      if (key[i] != kNone) c.trk_perm[s_cnt[key[i] - kmin] + rank[i]] = t;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kOrderItems; ++i)
      if (key[i] != kNone) s_cnt[key[i] - kmin] = 0u;
    __syncthreads();
  }
}
// tracklets per diagonal -> first slot of every diagonal (the counters of the fill pass start there)
__global__ void __launch_bounds__(1024) k_order_scan(const Ctx c, int kind) {
  __shared__ uint32_t s_warp[33];
  const uint32_t n_keys = order_keys((uint32_t)c.n_rows, c.n_tasks);
  const uint32_t* cnt = c.order_cnt + (size_t)(2 * kind) * n_keys;
  uint32_t* first = c.order_cnt + (size_t)(2 * kind + 1) * n_keys;
  uint32_t carry = 0u;
  for (uint32_t k0 = 0u; k0 < n_keys; k0 += 1024u) {
    const uint32_t k = k0 + threadIdx.x;
    const uint32_t v = k < n_keys ? cnt[k] : 0u;
    uint32_t total;
    const uint32_t ex = block_exclusive_scan(v, s_warp, &total);
    if (k < n_keys) first[k] = carry + ex;
    carry += total;
  }
}

// ---------------------------------------------------------------------------
// K1 seed + K2 chain fit.  Every step: transport one row up, update with the chain hit.  The hit two links
// ahead and the (y,z) of the next one are requested before the transport, so no step waits for a load.
// ---------------------------------------------------------------------------
constexpr int kChainSlot16 = kSeedU4;
template <bool COUNT>
__global__ void __launch_bounds__(kTrackletThreads, kFitBlocksPerSm) k_trk_chain(const Ctx c) {
  extern __shared__ __align__(16) float sX[];  // [n_rows] x of the pad rows, then the slots
  constexpr unsigned FULL = 0xffffffffu;
  const int n_rows = c.n_rows, lane = (int)threadIdx.x & 31;
  uint4* slot = reinterpret_cast<uint4*>(sX + ((n_rows + 3) & ~3)) + (size_t)threadIdx.x * kChainSlot16;
  for (int r = (int)threadIdx.x; r < n_rows; r += (int)blockDim.x) sX[r] = c.X[r];
  __syncthreads();
  const uint32_t n_trk = *c.n_tracklets;
  const float a = c.a, max_sin = c.prm.max_sinphi, sy2 = c.sy2, sz2 = c.sz2;
  TrackState S;
  zero_state(S);
  uint32_t t = 0u, t_next = 0u, tr_base = 0u;
  uint32_t* map = c.trk_hits;
  int r0 = 0, row_cur = 0, n_hits = 0;
  int32_t h_cur = -1, h_next = -1, h_last = -1;  // chain hit of the next step, the one after it, the last one fitted
  float2 p_cur = make_float2(0.0f, 0.0f);
  int st = LN_IDLE, pf = PF_NONE;
  TrackletQueue pool;
  queue_open(pool, &c.tickets[2], c.trk_perm, n_trk, lane);
  uint32_t n_steps = 0u, n_chain = 0u;
  while (true) {
    fetch_request<0>(pool, &c.tickets[2], c.trk_perm, (st == LN_IDLE || (st == LN_RUN && h_next < 0)) && pf == PF_NONE,
                         lane, n_trk, pf, t_next, slot, c.trk_seed, sizeof(uint4) * kSeedU4, kChainSlot16);
    if (st == LN_IDLE) {
      if (pf == PF_READY) {
        prefetch_wait();
        const uint4 q0 = slot[0], q1 = slot[1], q2 = slot[2];
        t = t_next;
        const uint32_t tr0 = q0.y;
        const uint32_t task = tr0 / (uint32_t)n_rows;
        r0 = (int)(tr0 - task * (uint32_t)n_rows);
        tr_base = task * (uint32_t)n_rows;
        map = c.trk_hits + (size_t)t * map_stride(n_rows);
        h_last = (int32_t)q0.z;
        h_cur = (int32_t)q0.w;
        h_next = (int32_t)q2.w;
        p_cur = make_float2(__uint_as_float(q2.x), __uint_as_float(q2.y));
        const float y0s = __uint_as_float(q1.x), z0s = __uint_as_float(q1.y);
        const float y1s = __uint_as_float(q1.z), z1s = __uint_as_float(q1.w);
        const float dx = sX[r0 + 1] - sX[r0], dy = y1s - y0s, dz = z1s - z0s;       // K1
        const float ri = 1.0f / sqrtf(dx * dx + dy * dy);
        S.y = y1s; S.z = z1s; S.s = dy * ri; S.t = dz * ri; S.q = 0.0f;
        S.c00 = sy2; S.c10 = 0.0f; S.c11 = sz2; S.c20 = 0.0f; S.c21 = 0.0f; S.c22 = c.prm.c0_sinphi;
        S.c30 = 0.0f; S.c31 = 0.0f; S.c32 = 0.0f; S.c33 = c.prm.c0_dzds;
        S.c40 = 0.0f; S.c41 = 0.0f; S.c42 = 0.0f; S.c43 = 0.0f; S.c44 = c.prm.c0_qpt;
        S.chi2 = 0.0f; S.ndf = -5;
        map[r0] = q0.x;
        map[r0 + 1] = q0.z;
        row_cur = r0 + 1; n_hits = 2;
        if (COUNT) n_chain += 2u;
        st = LN_RUN; pf = PF_NONE;
      } else if (pf == PF_DRAINED) {
        st = LN_EXIT;
      }
    }
    if (pf == PF_ISSUED) pf = PF_READY;
    if (__ballot_sync(FULL, st != LN_EXIT) == 0u) break;
    bool ok = true;
    const bool step = st == LN_RUN && h_cur >= 0;
    int32_t h_n2 = -1;
    float2 p_next = make_float2(0.0f, 0.0f);
    if (step) {                                                        // K2
      if (h_next >= 0) { p_next = c.yz[h_next]; h_n2 = c.clean_up[h_next]; }
      ok = transport(S, sX[row_cur + 1] - sX[row_cur], a, max_sin);
      if (COUNT) ++n_steps;
    }
    __syncwarp();
    if (step && ok) {
      update_hit(S, p_cur.x, p_cur.y, sy2, sz2);
      ++row_cur;
      map[row_cur] = (uint32_t)h_cur;
      ++n_hits;
      if (COUNT) ++n_chain;
      h_last = h_cur;
      h_cur = h_next; p_cur = p_next; h_next = h_n2;
    }
    if (st == LN_RUN && (h_cur < 0 || !ok)) {  // end of the chain, or K2's failed transport (-> K4, no up pass)
      store_rec(c.trk_rec + (size_t)t * kRecFloat4, S, 0.0f, n_hits, r0, row_cur,
                pack_rows(row_cur, row_cur - 1, r0, !ok), tr_base, (uint32_t)h_last, 0u);
      order_note(c, t, tr_base + (uint32_t)row_cur);            // the up pass begins in this row
      st = LN_IDLE;
    }
  }
  if (COUNT) {
    atomicAdd(&c.counters[CN_ROW_STEPS], (unsigned long long)n_steps);
    atomicAdd(&c.counters[CN_CHAIN_HITS], (unsigned long long)n_chain);
  }
}

// ---------------------------------------------------------------------------
// K3 up pass + K4 turn-around.  Every step of the up pass searches; the turn-around is the same step
// shape (transport to lastRow, no search, update with the hit of lastRow), so it runs with the others.
// ---------------------------------------------------------------------------
constexpr int kRecSlot16 = kRecFloat4;
template <bool COUNT>
__global__ void __launch_bounds__(kTrackletThreads, kSearchBlocksPerSm) k_trk_up(const Ctx c) {
  extern __shared__ __align__(16) float sX[];
  constexpr unsigned FULL = 0xffffffffu;
  const int n_rows = c.n_rows, lane = (int)threadIdx.x & 31;
  float4* slot = reinterpret_cast<float4*>(sX + ((n_rows + 3) & ~3)) + (size_t)threadIdx.x * kRecSlot16;
  for (int r = (int)threadIdx.x; r < n_rows; r += (int)blockDim.x) sX[r] = c.X[r];
  __syncthreads();
  const uint32_t n_trk = *c.n_tracklets;
  const float a = c.a, max_sin = c.prm.max_sinphi, sy2 = c.sy2, sz2 = c.sz2;
  const int max_gap = c.prm.max_row_gap;
  TrackState S;
  zero_state(S);
  uint32_t t = 0u, t_next = 0u, tr_base = 0u;
  uint32_t* map = c.trk_hits;
  int r0 = 0, row_cur = 0, first_row = 0, last_row = 0, n_hits = 0, gap = 0;
  int32_t last_hit = -1;
  bool turn = false;  // this lane's next step is the turn-around (its last step here)
  int st = LN_IDLE, pf = PF_NONE;
  TrackletQueue pool;
  queue_open(pool, &c.tickets[3], c.trk_perm, n_trk, lane);
  uint32_t n_steps = 0u, n_search = 0u, n_cand = 0u;
  while (true) {
    if (st == LN_RUN && row_cur + 1 >= n_rows) turn = true;            // K3 ran off the last row
    fetch_request<1>(pool, &c.tickets[3], c.trk_perm, (st == LN_IDLE || (st == LN_RUN && turn)) && pf == PF_NONE, lane,
                         n_trk, pf, t_next, slot, c.trk_rec, sizeof(float4) * kRecFloat4, kRecSlot16);
    if (st == LN_IDLE) {
      if (pf == PF_READY) {
        prefetch_wait();
        uint32_t pack, ia, ib;
        load_rec(slot, S, n_hits, first_row, last_row, pack, tr_base, ia, ib);
        t = t_next;
        row_cur = (int)(pack & 1023u); r0 = (int)((pack >> 20) & 1023u);
        map = c.trk_hits + (size_t)t * map_stride(n_rows);
        last_hit = (int32_t)ia;
        turn = (((pack >> 30) & 1u) != 0u) | (row_cur + 1 >= n_rows);
        gap = 0;
        st = LN_RUN; pf = PF_NONE;
      } else if (pf == PF_DRAINED) {
        st = LN_EXIT;
      }
    }
    if (pf == PF_ISSUED) pf = PF_READY;
    if (__ballot_sync(FULL, st != LN_EXIT) == 0u) break;
    const bool run = st == LN_RUN;
    int rt = 0;
    int32_t hit = -1;
    float2 hp = make_float2(0.0f, 0.0f);
    bool do_search = false, p_turn = false;
    uint32_t ia = kNoHit, ib = kNoHit;  // turn-around: map[lastRow - 1], map[lastRow - 2] for the refit kernel
    RowInfo g;
    g.inv = 0.0f; g.y0 = 0.0f; g.z0 = 0.0f; g.ny_nz = 0u; g.bins_off = 0u; g.row_lo = 0u; g.pad0 = 0u; g.pad1 = 0u;
    if (run) {
      p_turn = turn;
      rt = p_turn ? last_row : row_cur + 1;
      if (p_turn) {
        hp = c.yz[last_hit];
        if (last_row - 1 >= r0) ia = map[last_row - 1];
        if (last_row - 2 >= r0) ib = map[last_row - 2];
      } else {
        g = load_row_info(&c.rowinfo[tr_base + (uint32_t)rt]);
      }
      bool ok = true;
      if (rt != row_cur) {
        ok = transport(S, sX[rt] - sX[row_cur], a, max_sin);
        if (ok) row_cur = rt;
        if (COUNT && !p_turn) ++n_steps;
      }
      if (p_turn) {                                                    // K4: C <- C * turn_cov_scale
        const float f = c.prm.turn_cov_scale;
        S.c00 *= f; S.c10 *= f; S.c11 *= f; S.c20 *= f; S.c21 *= f; S.c22 *= f; S.c30 *= f; S.c31 *= f;
        S.c32 *= f; S.c33 *= f; S.c40 *= f; S.c41 *= f; S.c42 *= f; S.c43 *= f; S.c44 *= f;
        S.chi2 = 0.0f; S.ndf = -5;
        hit = row_cur == last_row ? last_hit : -1;                     // the hit of lastRow opens the down pass
      }
      do_search = ok & !p_turn;
      turn = turn | !ok;                                               // K3: failed transport -> turn-around
    }
    __syncwarp();
    if (do_search) {
      if (COUNT) ++n_search;
      hit = search_row<COUNT>(c, S, g, hp, n_cand);
    }
    __syncwarp();
    if (hit >= 0) update_hit(S, hp.x, hp.y, sy2, sz2);
    __syncwarp();
    if (do_search) {                                                   // K3 bookkeeping
      const bool got = hit >= 0;
      TPC_ST1(map + rt, (uint32_t)hit);                                // -1 = kNoHit
      n_hits += got ? 1 : 0;
      last_row = got ? rt : last_row;
      last_hit = got ? hit : last_hit;
      gap = got ? 0 : gap + 1;
      turn = turn | (gap > max_gap);
    }
    if (p_turn) {
      store_rec(c.trk_rec + (size_t)t * kRecFloat4, S, 0.0f, n_hits, first_row, last_row,
                pack_rows(row_cur, last_row - 1, r0, false), tr_base, ia, ib);
      order_note(c, t, tr_base + (uint32_t)(n_rows - 1 - last_row));  // the refit comes down from lastRow
      st = LN_IDLE;
    }
  }
  if (COUNT) {
    atomicAdd(&c.counters[CN_ROW_STEPS], (unsigned long long)n_steps);
    atomicAdd(&c.counters[CN_SEARCHES], (unsigned long long)n_search);
    atomicAdd(&c.counters[CN_CANDIDATES], (unsigned long long)n_cand);
    atomicAdd(&c.counters[CN_SEARCHES_UP], (unsigned long long)n_search);
    atomicAdd(&c.counters[CN_CANDIDATES_UP], (unsigned long long)n_cand);
  }
}

// ---------------------------------------------------------------------------
// K5, first part: the down pass as long as the row has a hit in the map (no search): transport one row
// down, update with the hit.  Map entry two rows ahead and (y,z) one row ahead are requested before the
// transport.  The lane stops in front of the first row without a hit (a hole of the map, or firstRow - 1)
// or of a transport that fails; k_trk_finish goes on from there.
// ---------------------------------------------------------------------------
template <bool COUNT>
__global__ void __launch_bounds__(kTrackletThreads, kFitBlocksPerSm) k_trk_refit(const Ctx c) {
  extern __shared__ __align__(16) float sX[];
  constexpr unsigned FULL = 0xffffffffu;
  const int n_rows = c.n_rows, lane = (int)threadIdx.x & 31;
  float4* slot = reinterpret_cast<float4*>(sX + ((n_rows + 3) & ~3)) + (size_t)threadIdx.x * kRecSlot16;
  for (int r = (int)threadIdx.x; r < n_rows; r += (int)blockDim.x) sX[r] = c.X[r];
  __syncthreads();
  const uint32_t n_trk = *c.n_tracklets;
  const float a = c.a, max_sin = c.prm.max_sinphi, sy2 = c.sy2, sz2 = c.sz2;
  TrackState S;
  zero_state(S);
  uint32_t t = 0u, t_next = 0u, tr_base = 0u;
  const uint32_t* map = c.trk_hits;
  int r0 = 0, row_cur = 0, first_row = 0, last_row = 0, n_hits = 0, r_down = 0;
  uint32_t m_cur = kNoHit, m_next = kNoHit;  // map[r_down], map[r_down - 1]
  float2 p_cur = make_float2(0.0f, 0.0f);
  int st = LN_IDLE, pf = PF_NONE;
  TrackletQueue pool;
  queue_open(pool, &c.tickets[4], c.trk_perm, n_trk, lane);
  uint32_t n_steps = 0u;
  while (true) {
    fetch_request<2>(pool, &c.tickets[4], c.trk_perm, (st == LN_IDLE || (st == LN_RUN && m_next == kNoHit)) && pf == PF_NONE,
                         lane, n_trk, pf, t_next, slot, c.trk_rec, sizeof(float4) * kRecFloat4, kRecSlot16);
    if (st == LN_IDLE) {
      if (pf == PF_READY) {
        prefetch_wait();
        uint32_t pack;
        load_rec(slot, S, n_hits, first_row, last_row, pack, tr_base, m_cur, m_next);
        t = t_next;
        row_cur = (int)(pack & 1023u); r_down = (int)((pack >> 10) & 1023u) - 1; r0 = (int)((pack >> 20) & 1023u);
        map = c.trk_hits + (size_t)t * map_stride(n_rows);
        if (m_cur != kNoHit) p_cur = c.yz[m_cur];  // needed after the first transport only
        st = LN_RUN; pf = PF_NONE;
      } else if (pf == PF_DRAINED) {
        st = LN_EXIT;
      }
    }
    if (pf == PF_ISSUED) pf = PF_READY;
    if (__ballot_sync(FULL, st != LN_EXIT) == 0u) break;
    bool ok = true;
    const bool step = st == LN_RUN && m_cur != kNoHit;
    uint32_t m_n2 = kNoHit;
    float2 p_next = make_float2(0.0f, 0.0f);
    if (step) {
      if (m_next != kNoHit) p_next = c.yz[m_next];
      if (r_down - 2 >= r0) m_n2 = map[r_down - 2];
      ok = transport(S, sX[r_down] - sX[row_cur], a, max_sin);
    }
    __syncwarp();
    if (step && ok) {
      update_hit(S, p_cur.x, p_cur.y, sy2, sz2);
      if (COUNT) ++n_steps;
      row_cur = r_down;
      --r_down;
      m_cur = m_next; p_cur = p_next; m_next = m_n2;
    }
    if (st == LN_RUN && (m_cur == kNoHit || !ok)) {
      store_rec(c.trk_rec + (size_t)t * kRecFloat4, S, 0.0f, n_hits, first_row, last_row,
                pack_rows(row_cur, r_down, r0, false), tr_base, m_cur, 0u);
      order_note(c, t, tr_base + (uint32_t)(n_rows - 1 - (r_down > 0 ? r_down : 0)));  // goes on from r_down
      st = LN_IDLE;
    }
  }
  if (COUNT) {
    atomicAdd(&c.counters[CN_ROW_STEPS], (unsigned long long)n_steps);
    atomicAdd(&c.counters[CN_REFIT_STEPS], (unsigned long long)n_steps);
  }
}

// ---------------------------------------------------------------------------
// K5, rest: rows below firstRow (every step searches) and what follows a hole of the map inside
// [firstRow, lastRow] (search in the hole, known hits after it); K6 finish (the same step shape: transport to
// firstRow, nothing else).  K7 (ownership) is k_resolve in stage_output.cuh.
// ---------------------------------------------------------------------------
enum Phase { PH_DOWN = 0, PH_FINISH = 1, PH_ENDED = 2, PH_IDLE = 3, PH_EXIT = 4 };
constexpr int kFinishSlot16 = kRecFloat4 + 1;  // the record and the third quarter of the seed record (gid of the start hit)

template <bool COUNT>
__global__ void __launch_bounds__(kTrackletThreads, kSearchBlocksPerSm) k_trk_finish(const Ctx c) {
  extern __shared__ __align__(16) float sX[];
  constexpr unsigned FULL = 0xffffffffu;
  const int n_rows = c.n_rows, lane = (int)threadIdx.x & 31;
  float4* slot = reinterpret_cast<float4*>(sX + ((n_rows + 3) & ~3)) + (size_t)threadIdx.x * kFinishSlot16;
  for (int r = (int)threadIdx.x; r < n_rows; r += (int)blockDim.x) sX[r] = c.X[r];
  __syncthreads();
  const uint32_t n_trk = *c.n_tracklets;
  const float a = c.a, max_sin = c.prm.max_sinphi, sy2 = c.sy2, sz2 = c.sz2;
  const int max_gap = c.prm.max_row_gap;
  [[maybe_unused]] const int min_hits = c.prm.min_track_hits;
  TrackState S;
  zero_state(S);
  uint32_t t = 0u, t_next = 0u, tr_base = 0u, gid0 = 0u;
  uint32_t* map = c.trk_hits;
  int r0 = 0, row_cur = 0, first_row = 0, last_row = 0, n_hits = 0, gap = 0, r_down = 0;
  uint32_t map_next = kNoHit;  // map[r_down], loaded one step ahead
  int phase = PH_IDLE, pf = PF_NONE;
  TrackletQueue pool;
  queue_open(pool, &c.tickets[5], c.trk_perm, n_trk, lane);
  uint32_t n_steps = 0u, n_search = 0u, n_cand = 0u, n_kept = 0u, n_kept_hits = 0u;
  while (true) {
    // (A) tracklets that ended in the last step: the record, and what the ownership kernel (K7) needs
    if (phase == PH_ENDED) {
      store_rec(c.trk_rec + (size_t)t * kRecFloat4, S, sX[row_cur], n_hits, first_row, last_row, 0u, tr_base, 0u, 0u);
      c.trk_meta[t] = make_uint4((uint32_t)n_hits, (uint32_t)first_row | ((uint32_t)last_row << 16), gid0, 0u);
      if (COUNT && n_hits >= min_hits) { ++n_kept; n_kept_hits += (uint32_t)n_hits; }
      phase = PH_IDLE;
    }
    // (B) the next tracklets: requested while the lane runs its finish step, taken over here
    {
      const bool want = (phase == PH_IDLE || phase == PH_FINISH || (phase == PH_DOWN && r_down < 0)) && pf == PF_NONE;
      const unsigned need = __ballot_sync(FULL, want);
      if (need || pool.asked) {
        uint32_t tn = 0u;
        if (queue_step<3>(pool, &c.tickets[5], c.trk_perm, n_trk, need, lane, tn)) {
          if (tn == kQueueEnd) {
            pf = PF_DRAINED;
          } else {
            t_next = tn;
            prefetch_slot(slot, c.trk_rec + (size_t)tn * kRecFloat4, kRecFloat4);
            prefetch_slot(slot + kRecFloat4, c.trk_seed + (size_t)tn * kSeedU4 + 2, 1);
            pf = PF_ISSUED;
          }
        }
      }
    }
    if (phase == PH_IDLE) {
      if (pf == PF_READY) {
        prefetch_wait();
        uint32_t pack, ib;
        load_rec(slot, S, n_hits, first_row, last_row, pack, tr_base, map_next, ib);
        gid0 = __float_as_uint(slot[kRecFloat4].z);
        t = t_next;
        row_cur = (int)(pack & 1023u); r_down = (int)((pack >> 10) & 1023u) - 1; r0 = (int)((pack >> 20) & 1023u);
        map = c.trk_hits + (size_t)t * map_stride(n_rows);
        gap = 0;
        phase = PH_DOWN; pf = PF_NONE;
      } else if (pf == PF_DRAINED) {
        phase = PH_EXIT;
      }
    }
    if (pf == PF_ISSUED) pf = PF_READY;
    if (__ballot_sync(FULL, phase != PH_EXIT) == 0u) break;
    // (C) one row step of every running lane: transport -> choose the hit -> update -> bookkeeping
    int rt = 0;
    int32_t hit = -1;
    float2 hp = make_float2(0.0f, 0.0f);
    bool book = false, do_search = false;
    RowInfo g;
    g.inv = 0.0f; g.y0 = 0.0f; g.z0 = 0.0f; g.ny_nz = 0u; g.bins_off = 0u; g.row_lo = 0u; g.pad0 = 0u; g.pad1 = 0u;
    if (phase <= PH_FINISH) {
      if (phase == PH_DOWN && r_down < 0) phase = PH_FINISH;            // K5 ran off row 0
      const bool p_down = phase == PH_DOWN, p_fin = phase == PH_FINISH;
      rt = p_down ? r_down : first_row;
      const int32_t known = (p_down & (map_next != kNoHit)) ? (int32_t)map_next : -1;
      if (known >= 0) hp = c.yz[known];
      if (p_down) {                                                     // map entry of the row after this one
        const int rn = rt - 1;
        map_next = rn >= r0 ? map[rn] : kNoHit;
      }
      if (p_down && known < 0) g = load_row_info(&c.rowinfo[tr_base + (uint32_t)rt]);
      bool ok = true;
      if (rt != row_cur) {
        ok = transport(S, sX[rt] - sX[row_cur], a, max_sin);
        if (ok) row_cur = rt;
        if (COUNT && p_down) ++n_steps;
      }
      book = ok & p_down;
      do_search = book & (known < 0);
      hit = (book & !do_search) ? known : -1;
      // K6 finish -> ended; failed transport in K5 -> finish
      phase = p_fin ? PH_ENDED : (ok ? phase : PH_FINISH);
    }
    __syncwarp();
    if (do_search) {
      if (COUNT) ++n_search;
      hit = search_row<COUNT>(c, S, g, hp, n_cand);
    }
    __syncwarp();
    if (hit >= 0) update_hit(S, hp.x, hp.y, sy2, sz2);
    __syncwarp();
    if (book) {
      const bool got = hit >= 0;
      const bool gap_row = do_search & (rt < first_row);                // rows whose hits / misses drive the gap
      if (do_search) TPC_ST1(map + rt, (uint32_t)hit);                  // -1 = kNoHit
      n_hits += (do_search & got) ? 1 : 0;
      if (gap_row & got) first_row = rt;
      gap = gap_row ? (got ? 0 : gap + 1) : gap;
      if (gap_row & !got & (gap > max_gap)) phase = PH_FINISH;          // K5 stop
      --r_down;
    }
  }
  if (COUNT) {
    atomicAdd(&c.counters[CN_ROW_STEPS], (unsigned long long)n_steps);
    atomicAdd(&c.counters[CN_SEARCHES], (unsigned long long)n_search);
    atomicAdd(&c.counters[CN_CANDIDATES], (unsigned long long)n_cand);
    atomicAdd(&c.counters[CN_TRACKLETS_KEPT], (unsigned long long)n_kept);
    atomicAdd(&c.counters[CN_TRACKLET_HITS], (unsigned long long)n_kept_hits);
  }
}

}  // namespace tpc
