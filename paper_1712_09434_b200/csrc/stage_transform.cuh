// Cluster transformation (PAPER.md L77 footnote 1: "convert the raw TPC clusters from
// TPC pad row, TPC pad, and time coordinates into x, y, and z coordinates taking into account the calibration";
// L101, L213: the map is the default or the fed-back calibration, the cluster index does not change).
// docs/ARITH_SPEC.md section 10, X1..X4: nominal pad/time geometry plus a bilinear (dy, dz) map per (sector,row).
//
// Pure streaming work: 8 bytes in, 8 bytes out per cluster, the 6 MB map stays in L2.  One block per 4096
// consecutive clusters (whole 16-byte groups: float4 loads of pad/time, float4 stores of y/z); the (task,row)
// of a cluster comes from the row offsets of the chunk, staged in shared memory once per block together with
// the pad row and the sector of every staged row (no division per cluster); the first row of the chunk is found
// by warp 0 with 32 probes per round.
#pragma once
#include "device_common.cuh"

namespace tpc {

#ifndef TPC_XF_THREADS
#define TPC_XF_THREADS 256
#endif
#ifndef TPC_XF_CHUNK
#define TPC_XF_CHUNK 4096
#endif
#ifndef TPC_XF_MINBLOCKS
#define TPC_XF_MINBLOCKS 6  // 40 registers; (chunk, blocks/SM): (2048, -) 0.24 ms, (4096, 6) 0.20, (8192, 6) 0.20 (but 8192 clusters of a sparse event span more rows than are staged)
#endif
constexpr int kXfThreads = TPC_XF_THREADS;
constexpr uint32_t kXfChunk = TPC_XF_CHUNK;  // clusters per block: whole float4 groups per thread
constexpr int kXfRows = 256;         // row offsets of the chunk kept in shared memory

struct TransformCtx {
  int32_t n_sectors, n_rows, my, mz;
  float z_max, t0, v_drift, kz;
  const float* pitch;   // [n_rows] X1
  const float* centre;  // [n_rows] 0.5f*(float)(n_pads-1)
  const float* ky;      // [n_rows] (float)(MY-1)/(float)(n_pads-1)
  const float* map;     // [n_sectors][n_rows][MZ][MY][2]
  const float *pad, *time;
  const uint32_t* row_off;
  uint32_t n, n_tr;
  float *y, *z;
};

// (task,row) index tr -> row | sector << 10 (n_rows <= 1024): computed once per staged row, not per cluster
__device__ __forceinline__ uint32_t row_sector(const TransformCtx& c, uint32_t tr) {
  const uint32_t nr = (uint32_t)c.n_rows, ns = (uint32_t)c.n_sectors;
  const uint32_t task = tr / nr;
  return (tr - task * nr) | ((task % ns) << 10);
}
// X1..X4 for one cluster of pad row `row` in sector `sec`, both packed as row_sector() gives them
__device__ __forceinline__ float2 transform_one(const TransformCtx& c, uint32_t rs, float pad, float time) {
  const uint32_t nr = (uint32_t)c.n_rows, ns = (uint32_t)c.n_sectors;
  const uint32_t row = rs & 1023u, sec = rs >> 10;
  const float y0 = (pad - __ldg(c.centre + row)) * __ldg(c.pitch + row);   // X1
  const float zd = (time - c.t0) * c.v_drift;                               // X2
  const float z0 = 2u * sec < ns ? c.z_max - zd : zd - c.z_max;
  float u = pad * __ldg(c.ky + row), v = time * c.kz;                       // X3
  u = fminf(fmaxf(u, 0.0f), (float)(c.my - 1));
  v = fminf(fmaxf(v, 0.0f), (float)(c.mz - 1));
  const int iu = min((int)u, c.my - 2), iv = min((int)v, c.mz - 2);
  const float fu = u - (float)iu, fv = v - (float)iv;
  const float2* m = reinterpret_cast<const float2*>(c.map) + ((size_t)(sec * nr + row) * c.mz + iv) * c.my + iu;
  const float2 m00 = __ldg(m), m01 = __ldg(m + 1), m10 = __ldg(m + c.my), m11 = __ldg(m + c.my + 1);
  const float ay = m00.x + fu * (m01.x - m00.x), by = m10.x + fu * (m11.x - m10.x);
  const float az = m00.y + fu * (m01.y - m00.y), bz = m10.y + fu * (m11.y - m10.y);
  return make_float2(y0 + (ay + fv * (by - ay)), z0 + (az + fv * (bz - az)));   // X4
}

__global__ void __launch_bounds__(kXfThreads, TPC_XF_MINBLOCKS) k_transform(const TransformCtx c) {
  __shared__ uint32_t s_rowoff[kXfRows + 1];
  __shared__ uint32_t s_rowsec[kXfRows + 1];  // row | sector << 10 of the staged rows
  __shared__ uint32_t s_tr;
  const uint32_t i0 = blockIdx.x * kXfChunk, i1 = min(i0 + kXfChunk, c.n);
  if (threadIdx.x < 32u) {  // last (task,row) with row_off <= i0: warp 0 probes 32 places per round (4 rounds for 10^5 rows)
    const uint32_t lane = threadIdx.x;
    uint32_t lo = 0u, hi = c.n_tr;  // row_off[lo] <= i0 < row_off[hi]
    while (hi - lo > 1u) {
      const uint32_t step = (hi - lo + 31u) / 32u;
      const uint64_t p64 = (uint64_t)lo + (uint64_t)(lane + 1u) * step;
      const uint32_t p = p64 < (uint64_t)hi ? (uint32_t)p64 : hi;
      const bool le = p < hi && c.row_off[p] <= i0;   // monotone in the lane: true for a prefix of the lanes
      const uint32_t k = (uint32_t)__popc(__ballot_sync(0xffffffffu, le));
      const uint32_t new_hi = (uint64_t)lo + (uint64_t)(k + 1u) * step < (uint64_t)hi ? lo + (k + 1u) * step : hi;
      lo = lo + k * step;
      hi = new_hi;
    }
    if (lane == 0u) s_tr = lo;
  }
  __syncthreads();
  const uint32_t tr0 = s_tr;
  for (uint32_t j = threadIdx.x; j <= (uint32_t)kXfRows; j += kXfThreads) {
    const uint32_t tr = min(tr0 + j, c.n_tr);
    s_rowoff[j] = c.row_off[tr];
    s_rowsec[j] = row_sector(c, min(tr, c.n_tr - 1u));
  }
  __syncthreads();
  // staged rows the chunk really spans (a chunk of a central event holds 5 rows): the searches below are short
  __shared__ uint32_t s_span;
  if (threadIdx.x == 0) {
    uint32_t k = 1u;
    while (k < (uint32_t)kXfRows && s_rowoff[k] < i1) ++k;
    s_span = k;  // s_rowoff[k] >= i1, or k == kXfRows
  }
  __syncthreads();
  const uint32_t span = s_span;
  const bool staged = s_rowoff[span] >= i1;  // else: more than kXfRows (mostly empty) rows, global search
  auto row_slot = [&](uint32_t i) -> uint32_t {  // last staged row j with s_rowoff[j] <= i
    uint32_t lo = 0u, hi = span;
    while (hi - lo > 1u) {
      const uint32_t mid = (lo + hi) >> 1;
      if (s_rowoff[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
  };
  auto tr_global = [&](uint32_t i) -> uint32_t {
    uint32_t lo = tr0, hi = c.n_tr;
    while (hi - lo > 1u) {
      const uint32_t mid = (lo + hi) >> 1;
      if (c.row_off[mid] <= i) lo = mid; else hi = mid;
    }
    return lo;
  };
  for (uint32_t g = i0 + 4u * threadIdx.x; g < i1; g += 4u * kXfThreads) {
    const uint32_t n_el = min(4u, i1 - g);
    uint32_t rs[4];
    if (staged) {  // the four clusters are consecutive: one search; a group inside one row (nearly all) needs no more
      uint32_t j = row_slot(g);
      if (j + 1u >= span || s_rowoff[j + 1u] >= g + 4u) {
        rs[0] = rs[1] = rs[2] = rs[3] = s_rowsec[j];
      } else {  // the group crosses row ends (empty rows too): step over them
#pragma unroll
        for (uint32_t k = 0; k < 4u; ++k) {
          while (j + 1u < span && s_rowoff[j + 1u] <= g + k) ++j;
          rs[k] = s_rowsec[j];
        }
      }
    } else {
#pragma unroll
      for (uint32_t k = 0; k < 4u; ++k) rs[k] = row_sector(c, tr_global(min(g + k, i1 - 1u)));
    }
    if (n_el == 4u) {  // a whole 16-byte group (cudaMalloc'ed arrays: chunk starts are 16-byte aligned)
      const float4 p = __ldg(reinterpret_cast<const float4*>(c.pad + g));
      const float4 t = __ldg(reinterpret_cast<const float4*>(c.time + g));
      const float2 r0 = transform_one(c, rs[0], p.x, t.x), r1 = transform_one(c, rs[1], p.y, t.y);
      const float2 r2 = transform_one(c, rs[2], p.z, t.z), r3 = transform_one(c, rs[3], p.w, t.w);
      *reinterpret_cast<float4*>(c.y + g) = make_float4(r0.x, r1.x, r2.x, r3.x);
      *reinterpret_cast<float4*>(c.z + g) = make_float4(r0.y, r1.y, r2.y, r3.y);
    } else {
      for (uint32_t k = 0; k < n_el; ++k) {
        const float2 r = transform_one(c, rs[k], c.pad[g + k], c.time[g + k]);
        c.y[g + k] = r.x; c.z[g + k] = r.y;
      }
    }
  }
}

}  // namespace tpc
