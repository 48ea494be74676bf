// raf_backward.cu -- K3: multi-level RoIAlign backward scatter.
//
//   gF_l[b,c,y,x] += sum over (k,ph,pw,iy,ix) of  w_tap * gout[k,c,ph,pw] / count
//
// Exact transpose of the forward: same sample coordinates, same weights (bit-identical, see
// raf_device.cuh), invalid samples skipped.  This file holds the ATOMIC variant:
//  * bwd_cl_kernel       channels-last: one CTA per RoI, sample tables in shared memory, threads
//                        laid out (4-channel group, bin); every tap is ONE 16-byte fp32 vector
//                        reduction `red.global.add.v4.f32` (north_star), a warp covers 512 B.
//  * bwd_generic_kernel  any strides / adaptive sampling: scalar atomicAdd per tap.
// Summation order across RoIs is whatever the L2 atomics see (several results are correct;
// tolerance reading S11).  The deterministic pull variant (the default) lives in raf_backward_pull.cu.
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

constexpr int kTableB = 64;

struct AxisEntryB {
  int lo, hi;
  float wl, wh;
};

// Load 4 consecutive channels of grad_out as fp32.
template <typename T> __device__ __forceinline__ float4 load4(const T* p);
template <> __device__ __forceinline__ float4 load4<float>(const float* p) {
  return __ldg(reinterpret_cast<const float4*>(p));
}
template <> __device__ __forceinline__ float4 load4<__half>(const __half* p) {
  const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
  const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
  return make_float4(a.x, a.y, b.x, b.y);
}
template <> __device__ __forceinline__ float4 load4<__nv_bfloat16>(const __nv_bfloat16* p) {
  const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
  return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u),
                     __uint_as_float(r.y << 16), __uint_as_float(r.y & 0xffff0000u));
}

template <typename T, int G>
__global__ void __launch_bounds__(256)
bwd_cl_kernel(const LevelsParam lv, const RoiArgs a, const T* __restrict__ gout, int64_t gs_k,
              int64_t gs_h, int64_t gs_w) {
  __shared__ AxisEntryB s_y[kTableB], s_x[kTableB];
  __shared__ float s_inv_count;
  __shared__ int s_b;

  const int k = blockIdx.x;
  const int tid = threadIdx.y * blockDim.x + threadIdx.x;
  const int g = (G > 0) ? G : a.sampling_ratio;
  const int ny = a.PH * g, nx = a.PW * g;
  const float* r = a.rois + 5 * (int64_t)k;
  const float r0 = __ldg(r), x1 = __ldg(r + 1), y1 = __ldg(r + 2), x2 = __ldg(r + 3), y2 = __ldg(r + 4);
  const int level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);
  const int b0 = batch_index_of(r0, lv.n);
  if (b0 < 0) return;  // uniform across the CTA: no gradient (reading S17)

  if (tid < ny + nx) {
    const RoiGeom geo = roi_geom(x1, y1, x2, y2, lv.scale[level], a.PH, a.PW, g, a.aligned);
    const bool isy = tid < ny;
    const int s = isy ? tid : tid - ny;
    const int p = s / g, i = s - p * g;
    const float v = isy ? sample_coord(geo.sy, geo.bh, p, i, g) : sample_coord(geo.sx, geo.bw, p, i, g);
    const AxisTap t = axis_tap(v, isy ? lv.h[level] : lv.w[level]);
    const int stride = (int)(isy ? lv.sh[level] : lv.sw[level]);
    AxisEntryB e;
    e.lo = t.valid ? t.lo * stride : -1;  // -1 marks an invalid sample
    e.hi = t.hi * stride;
    e.wl = t.wl;
    e.wh = t.wh;
    if (isy) s_y[s] = e; else s_x[s] = e;
    if (tid == 0) { s_inv_count = geo.inv_count; s_b = b0; }
  }
  __syncthreads();

  const float inv_count = s_inv_count;
  const int C4 = lv.c >> 2;
  const int nbins = a.PH * a.PW;
  const T* gout_k = gout + (int64_t)k * gs_k;
  float* base = reinterpret_cast<float*>(const_cast<void*>(lv.data[level])) + (int64_t)b0 * lv.sn[level];

  for (int bin = threadIdx.y; bin < nbins; bin += blockDim.y) {
    const int ph = bin / a.PW, pw = bin - ph * a.PW;
    for (int c4 = threadIdx.x; c4 < C4; c4 += blockDim.x) {
      float4 go = load4<T>(gout_k + ph * gs_h + pw * gs_w + c4 * 4);
      go.x *= inv_count; go.y *= inv_count; go.z *= inv_count; go.w *= inv_count;
      float* bc = base + c4 * 4;
#pragma unroll(G > 0 ? G : 1)
      for (int iy = 0; iy < g; ++iy) {
        const AxisEntryB ey = s_y[ph * g + iy];
        if (ey.lo < 0) continue;
#pragma unroll(G > 0 ? G : 1)
        for (int ix = 0; ix < g; ++ix) {
          const AxisEntryB ex = s_x[pw * g + ix];
          if (ex.lo < 0) continue;
          const float w1 = __fmul_rn(ey.wh, ex.wh), w2 = __fmul_rn(ey.wh, ex.wl);
          const float w3 = __fmul_rn(ey.wl, ex.wh), w4 = __fmul_rn(ey.wl, ex.wl);
          red_add_v4(bc + ey.lo + ex.lo, w1 * go.x, w1 * go.y, w1 * go.z, w1 * go.w);
          red_add_v4(bc + ey.lo + ex.hi, w2 * go.x, w2 * go.y, w2 * go.z, w2 * go.w);
          red_add_v4(bc + ey.hi + ex.lo, w3 * go.x, w3 * go.y, w3 * go.z, w3 * go.w);
          red_add_v4(bc + ey.hi + ex.hi, w4 * go.x, w4 * go.y, w4 * go.z, w4 * go.w);
        }
      }
    }
  }
}

template <typename T>
__global__ void __launch_bounds__(256)
bwd_generic_kernel(const LevelsParam lv, const RoiArgs a, const T* __restrict__ gout, int64_t gs_k,
                   int64_t gs_c, int64_t gs_h, int64_t gs_w, int64_t total) {
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int pw = (int)(idx % a.PW);
    const int ph = (int)((idx / a.PW) % a.PH);
    const int c = (int)((idx / ((int64_t)a.PW * a.PH)) % lv.c);
    const int k = (int)(idx / ((int64_t)a.PW * a.PH * lv.c));
    const float* r = a.rois + 5 * (int64_t)k;
    const float x1 = r[1], y1 = r[2], x2 = r[3], y2 = r[4];
    const int b = batch_index_of(r[0], lv.n);
    if (b < 0) continue;
    const int level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);
    const RoiGeom geo = roi_geom(x1, y1, x2, y2, lv.scale[level], a.PH, a.PW, a.sampling_ratio, a.aligned);
    const int H = lv.h[level], W = lv.w[level];
    const int64_t sh = lv.sh[level], sw = lv.sw[level];
    float* G_ = reinterpret_cast<float*>(const_cast<void*>(lv.data[level])) + b * lv.sn[level] + c * lv.sc[level];
    const float go = Elem<T>::to_f32(gout[k * gs_k + c * gs_c + ph * gs_h + pw * gs_w]) * geo.inv_count;
    for (int iy = 0; iy < geo.gh; ++iy) {
      const AxisTap ty = axis_tap(sample_coord(geo.sy, geo.bh, ph, iy, geo.gh), H);
      if (!ty.valid) continue;
      for (int ix = 0; ix < geo.gw; ++ix) {
        const AxisTap tx = axis_tap(sample_coord(geo.sx, geo.bw, pw, ix, geo.gw), W);
        if (!tx.valid) continue;
        atomicAdd(G_ + ty.lo * sh + tx.lo * sw, __fmul_rn(ty.wh, tx.wh) * go);
        atomicAdd(G_ + ty.lo * sh + tx.hi * sw, __fmul_rn(ty.wh, tx.wl) * go);
        atomicAdd(G_ + ty.hi * sh + tx.lo * sw, __fmul_rn(ty.wl, tx.wh) * go);
        atomicAdd(G_ + ty.hi * sh + tx.hi * sw, __fmul_rn(ty.wl, tx.wl) * go);
      }
    }
  }
}

__global__ void __launch_bounds__(256)
zero_level_kernel(float* __restrict__ data, int c, int h, int w, int64_t sn, int64_t sc, int64_t sh,
                  int64_t sw, int64_t total) {
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int x = (int)(idx % w);
    const int y = (int)((idx / w) % h);
    const int ch = (int)((idx / ((int64_t)w * h)) % c);
    const int n = (int)(idx / ((int64_t)w * h * c));
    data[n * sn + ch * sc + y * sh + x * sw] = 0.0f;
  }
}

int launch_zero_level(float* data, int n, int c, int h, int w, int64_t sn, int64_t sc, int64_t sh,
                      int64_t sw, cudaStream_t stream) {
  const int64_t total = (int64_t)n * c * h * w;
  const int64_t blocks = (total + 255) / 256;
  const int grid = (int)(blocks < (int64_t)148 * 32 ? blocks : (int64_t)148 * 32);
  zero_level_kernel<<<grid, 256, 0, stream>>>(data, c, h, w, sn, sc, sh, sw, total);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

template <typename T>
static int backward_typed(const LevelsParam& lv, const RoiArgs& a, const void* gout,
                          const int64_t* gs, bool channels_last, cudaStream_t stream) {
  const T* go = reinterpret_cast<const T*>(gout);
  const int g = a.sampling_ratio;
  if (channels_last && g > 0 && a.PH * g <= kTableB && a.PW * g <= kTableB) {
    const int C4 = lv.c / 4;
    int bx = 1;
    while (bx < C4 && bx < 256) bx <<= 1;
    const dim3 block(bx, 256 / bx);
    if (g == 2)
      bwd_cl_kernel<T, 2><<<a.K, block, 0, stream>>>(lv, a, go, gs[0], gs[2], gs[3]);
    else
      bwd_cl_kernel<T, 0><<<a.K, block, 0, stream>>>(lv, a, go, gs[0], gs[2], gs[3]);
  } else {
    const int64_t total = (int64_t)a.K * lv.c * a.PH * a.PW;
    const int64_t blocks = (total + 255) / 256;
    const int grid = (int)(blocks < (int64_t)148 * 64 ? blocks : (int64_t)148 * 64);
    bwd_generic_kernel<T><<<grid, 256, 0, stream>>>(lv, a, go, gs[0], gs[1], gs[2], gs[3], total);
  }
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

int launch_backward_atomic(const LevelsParam& glv, raf_dtype gout_dtype, const RoiArgs& a,
                           const void* grad_out, const int64_t* gout_strides, bool channels_last,
                           cudaStream_t stream) {
  switch (gout_dtype) {
    case RAF_F32: return backward_typed<float>(glv, a, grad_out, gout_strides, channels_last, stream);
    case RAF_F16: return backward_typed<__half>(glv, a, grad_out, gout_strides, channels_last, stream);
    case RAF_BF16: return backward_typed<__nv_bfloat16>(glv, a, grad_out, gout_strides, channels_last, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
