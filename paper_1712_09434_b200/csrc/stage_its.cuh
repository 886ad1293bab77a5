// ITS standalone tracker (section 4.2 "Fast ITS standalone tracking").
// docs/ARITH_SPEC.md section 12: SPD tracklets seen under nearly the same angle from the vertex (V1..V5), Kalman
// seed from the vertex and the two SPD clusters (W1..W4), outward pass with the nearest cluster under a strict chi2
// cut, multiple scattering per layer, at least 4 clusters and no two consecutive layers missed (O1..O4), inward
// pass to the vertex plane (N1..N3).  The track model (TRANSPORT, UPDATE) is the TPC tracker's.
//   k_its_pairs      one thread per SPD cluster (both layers): its best partner in the other layer by the plain
//                    loop over that layer's clusters of the event, 128 at a time through shared memory
//   k_its_tracklets  mutual choices become tracklets, numbered in the order of the inner cluster (ordered compaction)
//   k_its_follow     one warp per tracklet: seed, outward pass (every layer search is the plain loop over the
//                    layer's clusters, strided over the lanes, then a warp minimum of (chi2, gid)), inward pass
//   k_its_output     kept tracks are written in tracklet order (ordered compaction)
#pragma once
#include "device_common.cuh"
#include "stage_tracklet.cuh"

namespace tpc {

constexpr int kItsThreads = 128;
constexpr int kItsBlocksPerEvent = 16;  // k_its_pairs: blocks that share the SPD clusters of one event

struct ItsRec;
struct ItsCtx {
  float R[6], sr2[6], sz2[6], ms2[6];
  float a, wphi, wtan, svxy2, svz2;
  tpc_its_params prm;
  const float *x, *y, *z;
  const uint32_t* lo;   // [n_events*6 + 1]
  const float* vtx;     // [n_events][3]
  uint32_t n, n_events, max_tracklets;
  // workspace
  int32_t *best1, *best0;          // [n] partner of a layer-0 / layer-1 cluster (gid) or -1
  uint32_t *tl_a, *tl_b, *tl_ev;   // [max_tracklets]
  uint32_t* n_tracklets;
  unsigned long long *scan_tl, *scan_out;
  uint32_t* tickets;               // [2]
  struct ItsRec* recs;             // [max_tracklets] results parked for the ordered output
  tpc_its_tracks out;
};

// event of SPD cluster gid (layers 0, 1): last e with lo[6e] <= gid
__device__ __forceinline__ uint32_t its_event_of(const ItsCtx& c, uint32_t gid) {
  uint32_t lo = 0u, hi = c.n_events;
  while (hi - lo > 1u) {
    const uint32_t mid = (lo + hi) >> 1;
    if (c.lo[6u * mid] <= gid) lo = mid; else hi = mid;
  }
  return lo;
}

// V1..V5 for one cluster of layer `mine` (0 or 1) against every cluster of the other SPD layer of its event.
__global__ void __launch_bounds__(kItsThreads) k_its_pairs(const ItsCtx c) {
  // partner clusters of the tile, already relative to the vertex: (x, y, r, tan lambda) of V1 - computed once per
  // partner by the thread that stages it, not once per pair
  __shared__ float s_x[kItsThreads], s_y[kItsThreads], s_r[kItsThreads], s_t[kItsThreads];
  const uint32_t e = blockIdx.y;
  const int mine = (int)blockIdx.z;  // 0: threads are layer-0 clusters A, partners B in layer 1; 1: the other way round
  const float vx = c.vtx[3u * e], vy = c.vtx[3u * e + 1u], vz = c.vtx[3u * e + 2u];
  const uint32_t a0 = c.lo[6u * e], a1 = c.lo[6u * e + 1u], b1 = c.lo[6u * e + 2u];
  const uint32_t m0 = mine == 0 ? a0 : a1, m1 = mine == 0 ? a1 : b1;   // my clusters
  const uint32_t p0 = mine == 0 ? a1 : a0, p1 = mine == 0 ? b1 : a1;   // partners
  for (uint32_t base = m0 + blockIdx.x * kItsThreads; base < m1; base += gridDim.x * kItsThreads) {
    const uint32_t me = base + threadIdx.x;
    const bool act = me < m1;
    float mx = 0.f, my = 0.f, mr = 1.f, mt = 0.f;
    if (act) {
      mx = c.x[me] - vx; my = c.y[me] - vy; mr = sqrtf(mx * mx + my * my); mt = (c.z[me] - vz) / mr;   // V1
    }
    int32_t best = -1;
    float m_best = 0.f;
    for (uint32_t t0 = p0; t0 < p1; t0 += kItsThreads) {
      __syncthreads();
      if (t0 + threadIdx.x < p1) {
        const float ox = c.x[t0 + threadIdx.x] - vx, oy = c.y[t0 + threadIdx.x] - vy, orr = sqrtf(ox * ox + oy * oy);   // V1
        s_x[threadIdx.x] = ox; s_y[threadIdx.x] = oy; s_r[threadIdx.x] = orr; s_t[threadIdx.x] = (c.z[t0 + threadIdx.x] - vz) / orr;
      }
      __syncthreads();
      const uint32_t cnt = min((uint32_t)kItsThreads, p1 - t0);
      if (!act) continue;
      for (uint32_t k = 0; k < cnt; ++k) {
        const float ox = s_x[k], oy = s_y[k], orr = s_r[k], ot = s_t[k];
        // A is always the layer-0 cluster, B the layer-1 cluster, whoever the thread is
        const float ax = mine == 0 ? mx : ox, ay = mine == 0 ? my : oy, ra = mine == 0 ? mr : orr, ta = mine == 0 ? mt : ot;
        const float bx = mine == 0 ? ox : mx, by = mine == 0 ? oy : my, rb = mine == 0 ? orr : mr, tb = mine == 0 ? ot : mt;
        const float cd = ax * bx + ay * by;
        if (!(cd > 0.0f && fabsf(tb - ta) <= c.prm.max_dtan)) continue;                        // V3, the parts without a division first
        const float sd = (ax * by - ay * bx) / (ra * rb);                                      // V2
        if (!(fabsf(sd) <= c.prm.max_sinphi_pair)) continue;                                   // V3
        const float m = (sd * sd) * c.wphi + ((tb - ta) * (tb - ta)) * c.wtan;                 // V4
        if (best < 0 || m < m_best) { best = (int32_t)(t0 + k); m_best = m; }                   // V5: ascending gid, ties keep the smaller
      }
    }
    if (act) (mine == 0 ? c.best1 : c.best0)[me] = best;
  }
}

// V5: (A, B) is a tracklet iff each is the other's best; numbered in the order of gid A.
__global__ void __launch_bounds__(kItsThreads) k_its_tracklets(const ItsCtx c) {
  __shared__ uint32_t s_warp[33];
  __shared__ uint32_t s_tile;
  __shared__ unsigned long long s_prefix;
  if (threadIdx.x == 0) s_tile = atomicAdd(&c.tickets[0], 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t gid = tile * kItsThreads + threadIdx.x;
  bool is_tl = false;
  uint32_t e = 0u;
  int32_t b = -1;
  if (gid < c.n) {
    e = its_event_of(c, gid);
    if (gid >= c.lo[6u * e] && gid < c.lo[6u * e + 1u]) {  // a layer-0 cluster
      b = c.best1[gid];
      is_tl = b >= 0 && c.best0[b] == (int32_t)gid;
    }
  }
  uint32_t total;
  const uint32_t excl = block_exclusive_scan(is_tl ? 1u : 0u, s_warp, &total);
  if (threadIdx.x < 32) {
    const unsigned long long p = lookback_exclusive(c.scan_tl, tile, (unsigned long long)total);
    if (threadIdx.x == 0) s_prefix = p;
  }
  __syncthreads();
  const uint32_t pos = (uint32_t)s_prefix + excl;
  if (is_tl && pos < c.max_tracklets) { c.tl_a[pos] = gid; c.tl_b[pos] = (uint32_t)b; c.tl_ev[pos] = e; }
  if (threadIdx.x == 0 && tile == gridDim.x - 1) {
    const unsigned long long all = s_prefix + total;
    *c.n_tracklets = (uint32_t)(all > c.max_tracklets ? c.max_tracklets : all);
    c.out.header[1] = *c.n_tracklets;
    if (all > c.max_tracklets) atomicOr(&c.out.header[2], 1u);
  }
}

__device__ __forceinline__ void its_scatter(const ItsCtx& c, TrackState& S, int l) {
  const float th = c.ms2[l] * (S.q * S.q);
  S.c22 = S.c22 + th * (1.0f - S.s * S.s);
  S.c33 = S.c33 + th * ((1.0f + S.t * S.t) * (1.0f + S.t * S.t));
}

__device__ __forceinline__ void its_put_state(float* d, float x, const TrackState& S) {
  d[0] = x; d[1] = S.y; d[2] = S.z; d[3] = S.s; d[4] = S.t; d[5] = S.q;
  d[6] = S.c00; d[7] = S.c10; d[8] = S.c11; d[9] = S.c20; d[10] = S.c21; d[11] = S.c22; d[12] = S.c30; d[13] = S.c31;
  d[14] = S.c32; d[15] = S.c33; d[16] = S.c40; d[17] = S.c41; d[18] = S.c42; d[19] = S.c43; d[20] = S.c44; d[21] = S.chi2;
}

// Result of one tracklet, parked in the workspace until the ordered output knows its slot.
struct ItsRec {
  float out_state[22], in_state[22];
  float ca, sa;
  int32_t cluster[6];
  int32_t out_ndf, in_ndf;
  uint32_t n_clusters, event, alive, pad;
};

// W1..W4, O1..O4, N1..N3: one WARP per tracklet.  Every lane carries the same filter state (same inputs, same
// arithmetic, same bits); the lanes differ only in the layer searches of O2, where lane j tests the clusters
// j, j + 32, ... of the layer and the warp takes the lexicographic minimum of (chi2, gid).
__global__ void __launch_bounds__(kItsThreads) k_its_follow(const ItsCtx c) {
  constexpr unsigned FULL = 0xffffffffu;
  const uint32_t n_tl = *c.n_tracklets;
  const int lane = (int)threadIdx.x & 31;
  const uint32_t k = blockIdx.x * (kItsThreads / 32) + (threadIdx.x >> 5);
  if (k >= n_tl) return;
  const float a = c.a, max_sin = c.prm.max_sinphi;
  bool alive = true;
  TrackState S, S_out;
  zero_state(S);
  zero_state(S_out);
  float x = 0.0f, x_out = 0.0f;
  int32_t cl[6] = {-1, -1, -1, -1, -1, -1};
  const uint32_t A = c.tl_a[k], B = c.tl_b[k], e = c.tl_ev[k];
  const float vx = c.vtx[3u * e], vy = c.vtx[3u * e + 1u], vz = c.vtx[3u * e + 2u];
  const float ax = c.x[A] - vx, ay = c.y[A] - vy, ra = sqrtf(ax * ax + ay * ay);
  const float bx = c.x[B] - vx, by = c.y[B] - vy, rb = sqrtf(bx * bx + by * by), tb = (c.z[B] - vz) / rb;
  const float ca = bx / rb, sa = by / rb;                                                        // W1
  auto loc_x = [&](uint32_t P) { return (c.x[P] - vx) * ca + (c.y[P] - vy) * sa; };
  auto loc_y = [&](uint32_t P) { return (c.y[P] - vy) * ca - (c.x[P] - vx) * sa; };
  const float ox = -(vx * ca + vy * sa), oy = -(vy * ca - vx * sa);
  const float xa = loc_x(A), ya = loc_y(A), xb = rb;                                             // W2
  const float dab = sqrtf((xb - xa) * (xb - xa) + ya * ya);
  const float kap = -((2.0f * (ya * xb)) / ((ra * rb) * dab));
  S.y = 0.0f; S.z = vz; S.s = -(0.5f * kap) * xb; S.t = tb; S.q = a != 0.0f ? kap / a : 0.0f;    // W3
  S.c00 = c.svxy2; S.c11 = c.svz2; S.c22 = c.prm.c0_sinphi; S.c33 = c.prm.c0_dzds; S.c44 = c.prm.c0_qpt;
  S.chi2 = 0.0f; S.ndf = -5;
  update_hit(S, 0.0f, vz, c.svxy2, c.svz2);                                                      // W4
  auto attach = [&](uint32_t P, int l) {
    const float xp = loc_x(P);
    if (!transport(S, xp - x, a, max_sin)) return false;
    x = xp;
    update_hit(S, loc_y(P), c.z[P], c.sr2[l], c.sz2[l]);
    its_scatter(c, S, l);
    return true;
  };
  cl[0] = (int32_t)A; cl[1] = (int32_t)B;
  alive = attach(A, 0);                                                                          // O1
  if (alive) alive = attach(B, 1);
  int n_cl = 2, miss = 0;
#pragma unroll
  for (int l = 2; l < 6; ++l) {                                                                  // O2
    if (!alive) break;
    const float Rl = c.R[l];
    for (int it = 0; it < 2 && alive; ++it) {
      const float dyo = S.y - oy;
      const float xt = ox + sqrtf(fmaxf(Rl * Rl - dyo * dyo, 0.0f));
      if (it == 1 && xt == x) break;
      alive = transport(S, xt - x, a, max_sin);
      if (alive) x = xt;
    }
    if (!alive) break;
    const float cphi = sqrtf(1.0f - S.s * S.s);
    const float ey = S.c00 + c.sr2[l], ez = S.c11 + c.sz2[l];
    const float tany = S.s / cphi, tanz = S.t / cphi;
    uint32_t best = 0xFFFFFFFFu;
    float chi_best = __int_as_float(0x7f800000);
    // O2 as written is |dx| <= max_dx and chi2 < chi2_max with chi2 = dy^2/ey + dz^2/ez (two IEEE divisions).  The loop
    // visits every cluster of the layer and nearly all of them fail, so the cheap parts come first: the |dx| test and
    // dy^2 <= lim_y and dz^2 <= lim_z with lim_y = chi2_max * ey * (1 + 1e-4) - a NECESSARY condition of chi2 < chi2_max (both
    // terms are >= 0, so each alone is below chi2_max, up to the rounding the margin covers).  Only candidates that
    // pass all three pay for the divisions; those get the exact expression, so the decisions are the oracle's.
    const float max_dx = c.prm.max_dx, chi2_max = c.prm.chi2_max;
    const float lim_y = (chi2_max * ey) * 1.0001f, lim_z = (chi2_max * ez) * 1.0001f;
    // four clusters per lane and iteration: their twelve loads are in flight together (the loop waits for loads)
    for (uint32_t P0 = c.lo[6u * e + l] + (uint32_t)lane, Pe = c.lo[6u * e + l + 1u]; P0 < Pe; P0 += 128u) {
      float px[4], py[4], pz[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t P = P0 + 32u * (uint32_t)k;
        const bool in = P < Pe;
        px[k] = in ? c.x[P] : 0.0f; py[k] = in ? c.y[P] : 0.0f; pz[k] = in ? c.z[P] : 0.0f;
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t P = P0 + 32u * (uint32_t)k;
        const float dx = ((px[k] - vx) * ca + (py[k] - vy) * sa) - x;      // loc_x(P) - x
        const float dy = ((py[k] - vy) * ca - (px[k] - vx) * sa) - (S.y + dx * tany);
        const float dz = pz[k] - (S.z + dx * tanz);
        const float dy2 = dy * dy, dz2 = dz * dz;
        if ((P < Pe) & (fabsf(dx) <= max_dx) & (dy2 <= lim_y) & (dz2 <= lim_z)) {
          const float chi = dy2 / ey + dz2 / ez;
          if (chi < chi2_max && chi < chi_best) { best = P; chi_best = chi; }  // ascending P in a lane: ties keep the smaller gid
        }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {                             // lexicographic minimum of (chi2, gid) over the warp
      const float oc = __shfl_xor_sync(FULL, chi_best, o);
      const uint32_t ob = __shfl_xor_sync(FULL, best, o);
      if (oc < chi_best || (oc == chi_best && ob < best)) { chi_best = oc; best = ob; }
    }
    if (best != 0xFFFFFFFFu) {
      alive = attach(best, l);
      cl[l] = (int32_t)best; ++n_cl; miss = 0;
    } else {
      its_scatter(c, S, l);
      if (++miss == 2) alive = false;
    }
  }
  alive = alive && n_cl >= c.prm.min_clusters;                                                   // O3
  if (alive) {
    S_out = S; x_out = x;                                                                        // O4
    const float f = c.prm.turn_cov_scale;                                                        // N1
    S.c00 *= f; S.c10 *= f; S.c11 *= f; S.c20 *= f; S.c21 *= f; S.c22 *= f; S.c30 *= f; S.c31 *= f;
    S.c32 *= f; S.c33 *= f; S.c40 *= f; S.c41 *= f; S.c42 *= f; S.c43 *= f; S.c44 *= f;
    S.chi2 = 0.0f; S.ndf = -5;
#pragma unroll
    for (int l = 5; l >= 0; --l) {                                                               // N2
      if (cl[l] < 0) continue;
      const uint32_t P = (uint32_t)cl[l];
      const float xp = loc_x(P);
      if (xp != x) {
        if (!transport(S, xp - x, a, max_sin)) break;
        x = xp;
      }
      update_hit(S, loc_y(P), c.z[P], c.sr2[l], c.sz2[l]);
      its_scatter(c, S, l);
    }
    if (x != 0.0f && transport(S, 0.0f - x, a, max_sin)) x = 0.0f;                               // N3
  }
  if (lane == 0) {
    ItsRec& r = c.recs[k];
    r.alive = alive ? 1u : 0u;
    if (alive) {
      its_put_state(r.out_state, x_out, S_out);
      its_put_state(r.in_state, x, S);
      r.ca = ca; r.sa = sa;
#pragma unroll
      for (int l = 0; l < 6; ++l) r.cluster[l] = cl[l];
      r.out_ndf = S_out.ndf; r.in_ndf = S.ndf; r.n_clusters = (uint32_t)n_cl; r.event = e;
    }
  }
}

// kept tracks in tracklet order (ordered compaction): one thread per tracklet copies its parked result
__global__ void __launch_bounds__(kItsThreads) k_its_output(const ItsCtx c) {
  __shared__ uint32_t s_warp[33];
  __shared__ uint32_t s_tile;
  __shared__ unsigned long long s_prefix;
  if (threadIdx.x == 0) s_tile = atomicAdd(&c.tickets[1], 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t n_tl = *c.n_tracklets;
  const uint32_t last_tile = n_tl > 0u ? (n_tl - 1u) / kItsThreads : 0u;
  if (tile > last_tile) return;
  const uint32_t k = tile * kItsThreads + threadIdx.x;
  const bool alive = k < n_tl && c.recs[k].alive != 0u;
  uint32_t total;
  const uint32_t excl = block_exclusive_scan(alive ? 1u : 0u, s_warp, &total);
  if (threadIdx.x < 32) {
    const unsigned long long p = lookback_exclusive(c.scan_out, tile, (unsigned long long)total);
    if (threadIdx.x == 0) s_prefix = p;
  }
  __syncthreads();
  const uint32_t slot = (uint32_t)s_prefix + excl;
  const tpc_its_tracks& o = c.out;
  if (alive) {
    if (slot < o.capacity) {
      const ItsRec& r = c.recs[k];
      o.event[slot] = r.event; o.n_clusters[slot] = r.n_clusters;
      for (int l = 0; l < 6; ++l) o.cluster[(size_t)slot * 6 + l] = r.cluster[l];
      o.frame[2 * slot] = r.ca; o.frame[2 * slot + 1] = r.sa;
      for (int j = 0; j < 22; ++j) { o.out_state[(size_t)slot * 22 + j] = r.out_state[j]; o.in_state[(size_t)slot * 22 + j] = r.in_state[j]; }
      o.out_ndf[slot] = r.out_ndf; o.in_ndf[slot] = r.in_ndf;
    } else {
      atomicOr(&o.header[2], 2u);
    }
  }
  if (threadIdx.x == 0 && tile == last_tile) o.header[0] = (uint32_t)s_prefix + total;
}

}  // namespace tpc
