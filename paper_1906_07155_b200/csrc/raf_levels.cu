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

// ---------------------------------------------------------------------------------------------
// Stable bucketing by (level, image): key = level * N + batch_idx.  Feeds the pull backward
// (raf_backward_pull.cu), whose tiles walk the RoIs of their own (level, image) in ascending k --
// a fixed order, hence bit-reproducible sums.  RoIs with an invalid batch index are dropped.
//   bperm[K]      RoI indices grouped by key, ascending k inside a key
//   boff[NK + 1]  start of every key's group (NK = L * N)
//   bwin[K]       (optional) in bperm order: conservative window {ymin, ymax, xmin, xmax} of the
//                 pixels the RoI's samples can touch on its level (empty: ymin > ymax)
// One CTA, 32 warps; warp w owns the contiguous RoI range [w*q, (w+1)*q).  cnt[w][key] first
// counts, then (after a scan over keys, warps minor) holds the next free slot of (key, warp):
// warp-private rows, so neither atomics nor block barriers inside the walks.
// ---------------------------------------------------------------------------------------------

// Pixels an axis can touch: samples are monotone in (bin, i) up to rounding, so the first and the
// last sample (with slack for that rounding) bound all of them; a sample at v touches
// floor(max(v,0)) and the next pixel (clamped to n-1); samples outside [-1, n] touch nothing.
__device__ __forceinline__ void axis_window(float start, float bin, int P, int g, int n, int& lo, int& hi) {
  const float va = sample_coord(start, bin, 0, 0, g), vb = sample_coord(start, bin, P - 1, g - 1, g);
  const float slack = 0.01f + 1e-6f * fmaxf(fabsf(va), fabsf(vb));
  const float vlo = fminf(va, vb) - slack, vhi = fmaxf(va, vb) + slack;
  lo = 0x7fffffff; hi = -1;
  if (!(vlo <= vhi) || vhi < -1.0f || vlo > (float)n) return;   // NaN or entirely outside
  lo = (int)fminf(fmaxf(vlo, 0.0f), (float)(n - 1));
  hi = min(n - 1, (int)fminf(fmaxf(vhi, 0.0f), (float)(n - 1)) + 1);
}

__global__ void __launch_bounds__(kLevelThreads, 1)
bucket_rois_kernel(const LevelsParam lv, const RoiArgs a, int32_t* __restrict__ bperm,
                   int32_t* __restrict__ boff, int4* __restrict__ bwin) {
  extern __shared__ int s_cnt[];  // [32][NK + 1] then [NK + 1] totals/offsets
  const int K = a.K, L = lv.L, N = lv.n;
  const int NK = L * N, NK1 = NK + 1;
  int* s_tot = s_cnt + 32 * NK1;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int q = ((K + 31) / 32 + 31) & ~31;  // per-warp range, multiple of 32
  const int lo = warp * q, hi = min(K, lo + q);
  for (int i = tid; i < 32 * NK1 + NK1; i += kLevelThreads) s_cnt[i] = 0;
  __syncthreads();

  auto key_of = [&](int k) -> int {
    if (k >= hi) return -1;
    const float* r = a.rois + 5 * (int64_t)k;
    const int b = batch_index_of(r[0], N);
    if (b < 0) return NK;  // dropped
    return level_of(r[1], r[2], r[3], r[4], L, a.finest_scale) * N + b;
  };

  int* mine = s_cnt + warp * NK1;
  for (int k0 = lo; k0 < hi; k0 += 32) {
    const int key = key_of(k0 + lane);
    const unsigned peers = __match_any_sync(0xffffffffu, key);
    if (key >= 0 && lane == __ffs(peers) - 1) mine[key] += __popc(peers);
    __syncwarp();
  }
  __syncthreads();

  // totals per key
  for (int key = tid; key < NK1; key += kLevelThreads) {
    int t = 0;
    for (int w = 0; w < 32; ++w) t += s_cnt[w * NK1 + key];
    s_tot[key] = t;
  }
  __syncthreads();
  if (warp == 0) {  // exclusive scan of the totals over keys, 32 at a time
    int carry = 0;
    for (int base = 0; base < NK1; base += 32) {
      const int key = base + lane;
      const int v = key < NK1 ? s_tot[key] : 0;
      int incl = v;
      for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
      }
      if (key < NK1) s_tot[key] = carry + incl - v;
      carry += __shfl_sync(0xffffffffu, incl, 31);
    }
  }
  __syncthreads();
  for (int key = tid; key < NK1; key += kLevelThreads) {
    if (key <= NK) boff[key] = s_tot[key];  // boff[NK] = number of kept RoIs
    int run = s_tot[key];
    for (int w = 0; w < 32; ++w) {
      const int c = s_cnt[w * NK1 + key];
      s_cnt[w * NK1 + key] = run;
      run += c;
    }
  }
  __syncthreads();

  for (int k0 = lo; k0 < hi; k0 += 32) {
    const int k = k0 + lane;
    const int key = key_of(k);
    const unsigned peers = __match_any_sync(0xffffffffu, key);
    const int base = (key >= 0) ? mine[key] : 0;
    __syncwarp();
    if (key >= 0 && key < NK) {
      const int p = base + __popc(peers & ((1u << lane) - 1u));
      bperm[p] = k;
      if (bwin) {
        const float* r = a.rois + 5 * (int64_t)k;
        const int level = key / N;
        const RoiGeom geo = roi_geom(r[1], r[2], r[3], r[4], lv.scale[level], a.PH, a.PW, a.sampling_ratio, a.aligned);
        int4 w;
        axis_window(geo.sy, geo.bh, a.PH, a.sampling_ratio, lv.h[level], w.x, w.y);
        axis_window(geo.sx, geo.bw, a.PW, a.sampling_ratio, lv.w[level], w.z, w.w);
        if (w.x > w.y || w.z > w.w) w = make_int4(0x7fffffff, -1, 0x7fffffff, -1);
        bwin[p] = w;
      }
    }
    if (key >= 0 && lane == __ffs(peers) - 1) mine[key] = base + __popc(peers);
    __syncwarp();
  }
}

size_t bucket_smem_bytes(int L, int N) { return (size_t)33 * ((size_t)L * N + 1) * sizeof(int); }

int launch_bucket_rois(const LevelsParam& lv, const RoiArgs& a, int32_t* bperm, int32_t* boff, int4* bwin,
                       cudaStream_t stream) {
  const size_t smem = bucket_smem_bytes(lv.L, lv.n);
  if (smem > 200 * 1024) return RAF_ERR_UNSUPPORTED;
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(bucket_rois_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return RAF_ERR_CUDA;
  bucket_rois_kernel<<<1, kLevelThreads, smem, stream>>>(lv, a, bperm, boff, bwin);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

int launch_assign_levels(const float* rois, int K, int L, float finest_scale, int32_t* levels,
                         int32_t* counts, int32_t* perm, cudaStream_t stream) {
  assign_levels_kernel<<<1, kLevelThreads, 0, stream>>>(rois, K, L, finest_scale, levels, counts,
                                                        perm);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

}  // namespace raf
