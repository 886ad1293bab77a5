// a5  tracklet constructor ("Kalman filter for track fitting and
// track following"; L123: "in the track following phase, 1 GPU thread handles 1
// track").  docs/ARITH_SPEC.md sections 5 (track model) and 6 (K1..K7).
//
// One LANE per tracklet, the whole filter state (5 parameters, 15 covariance
// entries, chi2) in registers, in a PERSISTENT kernel: a lane whose tracklet has
// ended takes the next one from a global queue, so the 32 lanes of a warp stay
// busy although tracklets live for 10..320 row steps.  The five passes of SPEC 6
// (chain fit, up pass, turn-around, down pass, finish) are ONE loop whose body is
// a single row step
//     transport -> choose the hit (chain link / row map / search) -> update
// with a per-lane phase, so lanes in different passes execute the same
// instructions.  The row -> hit map of a tracklet is its row of Ctx::trk_hits in
// global memory (idx per pad row or kNoHit): written once per row step, read
// back in the down pass ONE ROW AHEAD, so that together with the chain link and
// the grid header every load a step needs is issued before the transport
// arithmetic and none is waited for.  No shared memory besides the row table:
// the registers alone bound the number of tracklets in flight.
#pragma once
#include "device_common.cuh"

namespace tpc {

constexpr int kTrackletThreads = 128;
constexpr int kTrackletBlocksPerSm = 6;  // registers per thread <= 65536 / (128 * 6) = 85

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
constexpr int kSearchUnroll = 2;

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

enum Phase { PH_CHAIN = 0, PH_UP = 1, PH_TURN = 2, PH_DOWN = 3, PH_FINISH = 4, PH_ENDED = 5, PH_FETCH = 6, PH_EXIT = 7 };

constexpr uint32_t kNoHit = 0xFFFFFFFFu;  // row map entry of a row without a hit
constexpr int kClaimChunks = 5;           // 32-row chunks of a map row claimed per round (159 rows = 5 chunks)

template <bool COUNT>
__global__ void __launch_bounds__(kTrackletThreads, kTrackletBlocksPerSm) k_tracklets(const Ctx c) {
  extern __shared__ __align__(16) float sX[];  // [n_rows] x of the pad rows
  constexpr unsigned FULL = 0xffffffffu;
  const int n_rows = c.n_rows, nthr = (int)blockDim.x, tid = (int)threadIdx.x, lane = tid & 31;
  for (int r = tid; r < n_rows; r += nthr) sX[r] = c.X[r];
  __syncthreads();
  const uint32_t n_trk = *c.n_tracklets;
  const float a = c.a, max_sin = c.prm.max_sinphi, sy2 = c.sy2, sz2 = c.sz2;
  const int max_gap = c.prm.max_row_gap, min_hits = c.prm.min_track_hits;

  TrackState S;
  S.y = S.z = S.s = S.t = S.q = 0.0f;
  S.c00 = S.c10 = S.c11 = S.c20 = S.c21 = S.c22 = S.c30 = S.c31 = S.c32 = S.c33 = 0.0f;
  S.c40 = S.c41 = S.c42 = S.c43 = S.c44 = 0.0f;
  S.chi2 = 0.0f; S.ndf = -5;
  uint32_t t = 0u, tr_base = 0u, gid0 = 0u;
  uint32_t* map = c.trk_hits;  // row map of the running tracklet
  int r0 = 0, row_cur = 0, first_row = 0, last_row = 0, n_hits = 0, gap = 0, r_down = 0;
  int32_t last_hit = -1, next_chain = -1;
  uint32_t map_next = kNoHit;  // down pass: map[r_down], loaded one step ahead
  int phase = PH_FETCH;
  uint32_t n_steps = 0u, n_search = 0u, n_cand = 0u, n_chain = 0u, n_kept = 0u, n_kept_hits = 0u;

  while (true) {
    // (A) tracklets that ended in the last step: the warp claims their hits one tracklet at a time
    //     (K7 ownership, 32 rows of the map per round), the lane stores the record
    unsigned ended = __ballot_sync(FULL, phase == PH_ENDED);
    if (ended) __syncwarp();  // the map rows written by the ended lanes are read by the other lanes below
    while (ended) {
      const int L = __ffs(ended) - 1;
      ended &= ended - 1u;
      const int fn = __shfl_sync(FULL, n_hits, L);
      if (fn >= min_hits) {  // K6, K7: longest tracklet wins, then the smaller start-hit gid
        const uint32_t ft = __shfl_sync(FULL, t, L), fgid0 = __shfl_sync(FULL, gid0, L);
        const int ffirst = __shfl_sync(FULL, first_row, L), flast = __shfl_sync(FULL, last_row, L);
        const unsigned long long key = ((unsigned long long)(uint32_t)fn << 32) | (unsigned long long)(0xFFFFFFFFu - fgid0);
        const uint32_t* fmap = c.trk_hits + (size_t)ft * map_stride(n_rows);
        for (int rb = ffirst; rb <= flast; rb += 32 * kClaimChunks) {  // the map loads of a round together, then the claims
          uint32_t idx[kClaimChunks];
#pragma unroll
          for (int q = 0; q < kClaimChunks; ++q) {
            const int r = rb + 32 * q + lane;
            idx[q] = r <= flast ? fmap[r] : kNoHit;
          }
#pragma unroll
          for (int q = 0; q < kClaimChunks; ++q)
            if (idx[q] != kNoHit) atomicMax(&c.owner[idx[q]], key);
        }
      }
      if (lane == L) {
        float4* rec = c.trk_rec + (size_t)t * kRecFloat4;
        rec[0] = make_float4(sX[row_cur], S.y, S.z, S.s);
        rec[1] = make_float4(S.t, S.q, S.c00, S.c10);
        rec[2] = make_float4(S.c11, S.c20, S.c21, S.c22);
        rec[3] = make_float4(S.c30, S.c31, S.c32, S.c33);
        rec[4] = make_float4(S.c40, S.c41, S.c42, S.c43);
        rec[5] = make_float4(S.c44, S.chi2, __int_as_float(S.ndf), __int_as_float(n_hits));
        rec[6] = make_float4(__int_as_float(first_row), __int_as_float(last_row), 0.0f, 0.0f);
        if (COUNT && n_hits >= min_hits) { ++n_kept; n_kept_hits += (uint32_t)n_hits; }
        phase = PH_FETCH;
      }
    }
    // (B) lanes without a tracklet take the next ones from the queue (K1 seed); the seed record of a4
    //     holds everything the seed needs, so a new tracklet costs one round of loads
    const unsigned need = __ballot_sync(FULL, phase == PH_FETCH);
    if (need) {
      uint32_t base = 0u;
      if (lane == 0) base = atomicAdd(&c.tickets[2], (uint32_t)__popc(need));
      base = __shfl_sync(FULL, base, 0);
      if (phase == PH_FETCH) {
        t = base + (uint32_t)__popc(need & ((1u << lane) - 1u));
        if (t >= n_trk) {
          phase = PH_EXIT;
        } else {
          const uint4* sr = c.trk_seed + (size_t)t * kSeedU4;
          const uint4 q0 = __ldg(sr), q1 = __ldg(sr + 1), q2 = __ldg(sr + 2);
          const uint32_t tr0 = q0.y;
          const uint32_t task = tr0 / (uint32_t)n_rows;
          r0 = (int)(tr0 - task * (uint32_t)n_rows);
          tr_base = task * (uint32_t)n_rows;
          gid0 = q2.z;
          map = c.trk_hits + (size_t)t * map_stride(n_rows);
          const float y0s = __uint_as_float(q1.x), z0s = __uint_as_float(q1.y);
          const float y1s = __uint_as_float(q1.z), z1s = __uint_as_float(q1.w);
          const float dx = sX[r0 + 1] - sX[r0], dy = y1s - y0s, dz = z1s - z0s;
          const float ri = 1.0f / sqrtf(dx * dx + dy * dy);
          S.y = y1s; S.z = z1s; S.s = dy * ri; S.t = dz * ri; S.q = 0.0f;
          S.c00 = sy2; S.c10 = 0.0f; S.c11 = sz2; S.c20 = 0.0f; S.c21 = 0.0f; S.c22 = c.prm.c0_sinphi;
          S.c30 = 0.0f; S.c31 = 0.0f; S.c32 = 0.0f; S.c33 = c.prm.c0_dzds;
          S.c40 = 0.0f; S.c41 = 0.0f; S.c42 = 0.0f; S.c43 = 0.0f; S.c44 = c.prm.c0_qpt;
          S.chi2 = 0.0f; S.ndf = -5;
          map[r0] = q0.x;
          map[r0 + 1] = q0.z;
          row_cur = r0 + 1; first_row = r0; last_row = r0 + 1; n_hits = 2; gap = 0; r_down = 0;
          last_hit = (int32_t)q0.z;
          next_chain = (int32_t)q0.w;
          phase = next_chain >= 0 ? PH_CHAIN : PH_UP;
          if (COUNT) n_chain += 2u;
        }
      }
    }
    if (__ballot_sync(FULL, phase != PH_EXIT) == 0u) break;
    // (C) one row step of every running lane: transport -> choose the hit -> update -> bookkeeping.
    //     The parts are separated by warp barriers so that the lanes run each of them together
    //     whatever their phase is.
    int rt = 0;
    int32_t hit = -1;
    float2 hp = make_float2(0.0f, 0.0f);
    bool book = false, do_search = false;
    RowInfo g;
    g.inv = 0.0f; g.y0 = 0.0f; g.z0 = 0.0f; g.ny_nz = 0u; g.bins_off = 0u; g.row_lo = 0u; g.pad0 = 0u; g.pad1 = 0u;
    if (phase <= PH_FINISH) {
      if (phase == PH_UP && row_cur + 1 >= n_rows) phase = PH_TURN;     // K3 ran off the last row
      if (phase == PH_DOWN && r_down < 0) phase = PH_FINISH;            // K5 ran off row 0
      const bool p_chain = phase == PH_CHAIN, p_turn = phase == PH_TURN, p_down = phase == PH_DOWN;
      rt = phase <= PH_UP ? row_cur + 1 : (p_turn ? last_row : (p_down ? r_down : first_row));
      // Every load of this step whose address does not depend on the transported state is issued here,
      // before the transport: the hit when it is known already (chain link, lastRow hit at the turn, row
      // map entry fetched a step ago), the next chain link, the map entry of the next down row, and the
      // row's grid header when a search may follow.
      const int32_t known = p_chain ? next_chain
                                    : (p_turn ? last_hit : ((p_down & (map_next != kNoHit)) ? (int32_t)map_next : -1));
      if (known >= 0) hp = c.yz[known];
      if (phase == PH_CHAIN) next_chain = c.clean_up[known];            // K2: the link after this one
      if (phase == PH_TURN || phase == PH_DOWN) {                       // map entry of the row after this one
        const int rn = (phase == PH_TURN ? last_row : rt) - 1;
        map_next = rn >= r0 ? map[rn] : kNoHit;
      }
      if (phase == PH_UP || (phase == PH_DOWN && known < 0)) g = load_row_info(&c.rowinfo[tr_base + (uint32_t)rt]);
      bool ok = true;
      if (rt != row_cur) {
        ok = transport(S, sX[rt] - sX[row_cur], a, max_sin);
        if (ok) row_cur = rt;
        if (COUNT && phase != PH_TURN && phase != PH_FINISH) ++n_steps;
      }
      // what the step does next, by phase, without branches (the lanes of a warp are in different passes)
      const bool p_fin = phase == PH_FINISH;
      if (p_turn) {                                                       // K4: C <- C * turn_cov_scale (once per tracklet)
        const float f = c.prm.turn_cov_scale;
        S.c00 *= f; S.c10 *= f; S.c11 *= f; S.c20 *= f; S.c21 *= f; S.c22 *= f; S.c30 *= f; S.c31 *= f;
        S.c32 *= f; S.c33 *= f; S.c40 *= f; S.c41 *= f; S.c42 *= f; S.c43 *= f; S.c44 *= f;
      }
      S.chi2 = p_turn ? 0.0f : S.chi2;
      S.ndf = p_turn ? -5 : S.ndf;
      gap = p_turn ? 0 : gap;
      r_down = p_turn ? last_row - 1 : r_down;
      book = ok & !p_fin & !p_turn;                                       // K2, K3, K5 with the transport done
      do_search = book & ((phase == PH_UP) | (known < 0));                // K3, K5 without a map entry
      // the hit is known: K2, K5 with a map entry, K4 (the lastRow hit opens the down pass)
      hit = ((book & !do_search) | (p_turn & (row_cur == last_row))) ? known : -1;
      // K6 finish -> ended; K4 -> down pass; failed transport: K2/K3 -> turn-around, K5 -> finish
      phase = p_fin ? PH_ENDED : (p_turn ? PH_DOWN : (ok ? phase : (p_down ? PH_FINISH : PH_TURN)));
    }
    __syncwarp();
    if (do_search) {
      if (COUNT) ++n_search;
      hit = search_row<COUNT>(c, S, g, hp, n_cand);
    }
    __syncwarp();
    if (hit >= 0) update_hit(S, hp.x, hp.y, sy2, sz2);
    __syncwarp();
    if (book) {  // chain fit, up pass or down pass, transport done: record the row, count hits and gaps (no branches:
                 // the lanes of a warp are in different passes)
      const bool is_up = phase == PH_UP, is_dn = phase == PH_DOWN, got = hit >= 0;
      const bool decided = !is_dn | do_search;                  // this step decided the row's map entry
      const bool gap_row = is_up | (is_dn & do_search & (rt < first_row));  // rows whose hits / misses drive the gap
      if (decided) map[rt] = (uint32_t)hit;                     // -1 = kNoHit
      n_hits += (decided & got) ? 1 : 0;
      if (COUNT && phase == PH_CHAIN) ++n_chain;
      if (!is_dn & got) { last_row = rt; last_hit = hit; }
      if (gap_row & got & is_dn) first_row = rt;
      gap = gap_row ? (got ? 0 : gap + 1) : gap;
      if (gap_row & !got & (gap > max_gap)) phase = is_up ? PH_TURN : PH_FINISH;   // K3 / K5 stop
      if (phase == PH_CHAIN && next_chain < 0) { phase = PH_UP; gap = 0; }          // K2 -> K3
      r_down -= is_dn ? 1 : 0;
    }
  }
  if (COUNT) {
    atomicAdd(&c.counters[CN_ROW_STEPS], (unsigned long long)n_steps);
    atomicAdd(&c.counters[CN_SEARCHES], (unsigned long long)n_search);
    atomicAdd(&c.counters[CN_CANDIDATES], (unsigned long long)n_cand);
    atomicAdd(&c.counters[CN_CHAIN_HITS], (unsigned long long)n_chain);
    atomicAdd(&c.counters[CN_TRACKLETS_KEPT], (unsigned long long)n_kept);
    atomicAdd(&c.counters[CN_TRACKLET_HITS], (unsigned long long)n_kept_hits);
  }
}

}  // namespace tpc
