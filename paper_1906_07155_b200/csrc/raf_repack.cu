// raf_repack.cu -- NCHW <-> channels-last repack: "any NCHW -> channel-last
// repack counted in the timing" (north_star).  One batched matrix transpose, src[b][R][S] -> dst[b][S][R],
// through 64 x 64 shared-memory tiles (both the reads and the writes are coalesced along the fast
// dimension).  A level [N, C, H, W] contiguous is the matrix C x (H*W) per image; an output / grad_out
// tensor [K, C, PH, PW] is C x (PH*PW) per RoI.  Used only when the caller passes RAF_REPACK together with
// a workspace that has room for the channels-last copies (roi_align_fpn_repack_bytes).
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

constexpr int kTrTile = 64;   // 64 x 64 elements per CTA: 16 KB (fp32) in flight per CTA before the barrier

template <typename T>
__global__ void __launch_bounds__(256)
transpose_kernel(const T* __restrict__ src, T* __restrict__ dst, int R, int S, int tiles_r, int tiles_s) {
  __shared__ T tile[kTrTile][kTrTile + 1];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8 threads
  const int64_t bid = blockIdx.x;
  const int64_t per = (int64_t)tiles_r * tiles_s;
  const int64_t b = bid / per;
  const int rem = (int)(bid - b * per);
  const int tr = rem / tiles_s, ts = rem - tr * tiles_s;
  const int r0 = tr * kTrTile, s0 = ts * kTrTile;
  const T* sp = src + b * (int64_t)R * S;
  T* dp = dst + b * (int64_t)R * S;
#pragma unroll
  for (int i = ty; i < kTrTile; i += 8) {
    const int r = r0 + i;
#pragma unroll
    for (int h = 0; h < kTrTile; h += 32) {
      const int s = s0 + h + tx;
      if (r < R && s < S) tile[i][h + tx] = sp[(int64_t)r * S + s];
    }
  }
  __syncthreads();
#pragma unroll
  for (int i = ty; i < kTrTile; i += 8) {
    const int s = s0 + i;
#pragma unroll
    for (int h = 0; h < kTrTile; h += 32) {
      const int r = r0 + h + tx;
      if (r < R && s < S) dp[(int64_t)s * R + r] = tile[h + tx][i];
    }
  }
}

// src[batch][R][S] -> dst[batch][S][R]; esz = 2 or 4 bytes per element.
int launch_transpose(const void* src, void* dst, int64_t batch, int R, int S, size_t esz, cudaStream_t stream) {
  if (batch <= 0 || R <= 0 || S <= 0) return RAF_OK;
  const int tiles_r = (R + kTrTile - 1) / kTrTile, tiles_s = (S + kTrTile - 1) / kTrTile;
  const int64_t blocks = batch * tiles_r * tiles_s;
  if (blocks >= ((int64_t)1 << 31)) return RAF_ERR_UNSUPPORTED;
  if (esz == 4)
    transpose_kernel<uint32_t><<<(unsigned)blocks, 256, 0, stream>>>((const uint32_t*)src, (uint32_t*)dst, R, S, tiles_r, tiles_s);
  else
    transpose_kernel<uint16_t><<<(unsigned)blocks, 256, 0, stream>>>((const uint16_t*)src, (uint16_t*)dst, R, S, tiles_r, tiles_s);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

}  // namespace raf
