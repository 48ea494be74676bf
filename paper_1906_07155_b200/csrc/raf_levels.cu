// raf_levels.cu -- K1: level assignment + per-level histogram + stable bucketing.
// (north_star "level-assignment and RoI-bucketing kernel".)
//
// One CTA of 1024 threads walks the RoIs in chunks of 1024, in order.  Stability comes from the
// order: position = offset[level] + (#RoIs of that level in earlier chunks) + (rank inside the
// chunk, from warp ballots + a scan over the 32 warp counts).  K <= 8192 in every BASELINE config
// (<= 8 chunks); the bytes are negligible (20 B/RoI in, 8 B/RoI out), the cost is launch latency.
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

constexpr int kLevelThreads = 1024;

__global__ void __launch_bounds__(kLevelThreads, 1)
assign_levels_kernel(const float* __restrict__ rois, int K, int L, float finest_scale,
                     int32_t* __restrict__ levels, int32_t* __restrict__ counts,
                     int32_t* __restrict__ perm) {
  __shared__ int s_hist[kMaxLevels];
  __shared__ int s_base[kMaxLevels];            // next free slot of each level
  __shared__ int s_warp[kMaxLevels][32];        // per-warp count of each level in this chunk
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid < kMaxLevels) s_hist[tid] = 0;
  __syncthreads();

  // pass 1: levels + histogram
  for (int k = tid; k < K; k += kLevelThreads) {
    const float* r = rois + 5 * (int64_t)k;
    const int lv = level_of(r[1], r[2], r[3], r[4], L, finest_scale);
    if (levels) levels[k] = lv;
    atomicAdd(&s_hist[lv], 1);
  }
  __syncthreads();
  if (tid == 0) {
    int run = 0;
    for (int l = 0; l < L; ++l) {
      if (counts) counts[l] = s_hist[l];
      s_base[l] = run;
      run += s_hist[l];
    }
  }
  if (!perm) return;
  __syncthreads();

  // pass 2: stable positions, chunk by chunk
  for (int k0 = 0; k0 < K; k0 += kLevelThreads) {
    const int k = k0 + tid;
    int lv = -1;
    if (k < K) {
      const float* r = rois + 5 * (int64_t)k;
      lv = level_of(r[1], r[2], r[3], r[4], L, finest_scale);
    }
    int rank_in_warp = 0;
    for (int l = 0; l < L; ++l) {
      const unsigned m = __ballot_sync(0xffffffffu, lv == l);
      if (lane == 0) s_warp[l][warp] = __popc(m);
      if (lv == l) rank_in_warp = __popc(m & ((1u << lane) - 1u));
    }
    __syncthreads();
    if (lv >= 0) {
      int before = 0;
      for (int w = 0; w < warp; ++w) before += s_warp[lv][w];
      perm[s_base[lv] + before + rank_in_warp] = k;
    }
    __syncthreads();
    if (tid < L) {
      int tot = 0;
      for (int w = 0; w < 32; ++w) tot += s_warp[tid][w];
      s_base[tid] += tot;
    }
    __syncthreads();
  }
}

int launch_assign_levels(const float* rois, int K, int L, float finest_scale, int32_t* levels,
                         int32_t* counts, int32_t* perm, cudaStream_t stream) {
  assign_levels_kernel<<<1, kLevelThreads, 0, stream>>>(rois, K, L, finest_scale, levels, counts,
                                                        perm);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

}  // namespace raf
