// Frame slicer ("slice the time frames along the time / beam axis,
// process the slices individually, and merge the track segments afterwards").  docs/ARITH_SPEC.md section 11, SLICE:
// clusters of whole frames, sorted by (frame, sector, row), are re-sorted by (frame, slice, sector, row) - stable
// inside a row - with the slice from the fp32 formula; src_index keeps the identity of every cluster (L213).
//   k_slice_count    one warp per input (task,row): clusters per slice -> counts of the output rows
//   k_slice_scan     exclusive scan of the output row counts (one block) -> row_offsets_out
//   k_slice_scatter  one warp per input (task,row): 32 clusters at a time, the rank of a cluster among those of its
//                    slice by __match_any_sync, running counts per slice in shared memory: a stable partition
#pragma once
#include "device_common.cuh"

namespace tpc {

constexpr int kSliceThreads = 128;  // 4 warps = 4 input rows per block
constexpr int kMaxSlices = 256;

struct SliceCtx {
  const float *y, *z;
  const uint32_t* row_off_in;   // [n_tr_in + 1]
  uint32_t n, n_tr_in;          // n_tr_in = n_tasks_in * n_rows
  int32_t n_sectors, n_rows, n_slices;
  float inv_len;
  float *y_out, *z_out;
  uint32_t *src_index, *row_off_out;  // [n], [n_tr_in * n_slices + 1]
  uint32_t* counts;                   // workspace [n_tr_in * n_slices + 1]
};

__device__ __forceinline__ uint32_t slice_of(const SliceCtx& c, float zeta) {
  return (uint32_t)fminf(fmaxf(fabsf(zeta) * c.inv_len, 0.0f), (float)(c.n_slices - 1));
}
// output (task,row) of input (task,row) tr and slice s
__device__ __forceinline__ uint32_t slice_out_tr(const SliceCtx& c, uint32_t tr, uint32_t s) {
  const uint32_t nr = (uint32_t)c.n_rows, ns = (uint32_t)c.n_sectors;
  const uint32_t task = tr / nr, row = tr - task * nr, frame = task / ns, sec = task - frame * ns;
  return ((frame * (uint32_t)c.n_slices + s) * ns + sec) * nr + row;
}

__global__ void __launch_bounds__(kSliceThreads) k_slice_count(const SliceCtx c) {
  __shared__ uint32_t s_cnt[kSliceThreads / 32][kMaxSlices];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t tr = blockIdx.x * (kSliceThreads / 32) + warp;
  if (tr >= c.n_tr_in) return;
  for (int s = lane; s < c.n_slices; s += 32) s_cnt[warp][s] = 0u;
  __syncwarp();
  for (uint32_t i = c.row_off_in[tr] + lane, e = c.row_off_in[tr + 1]; i < e; i += 32) atomicAdd(&s_cnt[warp][slice_of(c, c.z[i])], 1u);
  __syncwarp();
  for (int s = lane; s < c.n_slices; s += 32) c.counts[slice_out_tr(c, tr, (uint32_t)s)] = s_cnt[warp][s];
}

__global__ void __launch_bounds__(1024) k_slice_scan(const SliceCtx c) {
  __shared__ uint32_t s_warp[33];
  const uint32_t n = c.n_tr_in * (uint32_t)c.n_slices + 1u, per = (n + 1023u) / 1024u;
  const uint32_t b0 = min(threadIdx.x * per, n), b1 = min(b0 + per, n);
  uint32_t sum = 0u;
  for (uint32_t k = b0; k < b1; ++k) sum += k + 1u < n ? c.counts[k] : 0u;
  uint32_t total;
  uint32_t run = block_exclusive_scan(sum, s_warp, &total);
  for (uint32_t k = b0; k < b1; ++k) { c.row_off_out[k] = run; run += k + 1u < n ? c.counts[k] : 0u; }
}

__global__ void __launch_bounds__(kSliceThreads) k_slice_scatter(const SliceCtx c) {
  __shared__ uint32_t s_pos[kSliceThreads / 32][kMaxSlices];  // next output position of every slice of this row
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t tr = blockIdx.x * (kSliceThreads / 32) + warp;
  if (tr >= c.n_tr_in) return;
  for (int s = lane; s < c.n_slices; s += 32) s_pos[warp][s] = c.row_off_out[slice_out_tr(c, tr, (uint32_t)s)];
  __syncwarp();
  const uint32_t lo = c.row_off_in[tr], hi = c.row_off_in[tr + 1];
  for (uint32_t i0 = lo; i0 < hi; i0 += 32) {  // 32 consecutive clusters: input order is kept inside every slice
    const uint32_t i = i0 + lane;
    const bool act = i < hi;
    const float zz = act ? c.z[i] : 0.0f;
    const uint32_t s = act ? slice_of(c, zz) : 0xFFFFFFFFu;
    const unsigned same = __match_any_sync(0xffffffffu, s);
    const uint32_t rank = __popc(same & ((1u << lane) - 1u));
    uint32_t base = 0u;
    if (act) base = s_pos[warp][s];
    __syncwarp();
    if (act && rank == 0u) s_pos[warp][s] = base + __popc(same);
    __syncwarp();
    if (act) {
      const uint32_t k = base + rank;
      c.y_out[k] = c.y[i];
      c.z_out[k] = zz;
      c.src_index[k] = i;
    }
  }
}

}  // namespace tpc
