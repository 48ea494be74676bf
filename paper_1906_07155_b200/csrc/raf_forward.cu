// raf_forward.cu -- K2: multi-level RoIAlign forward gather.
//
//   out[k,c,ph,pw] = (1/count) * sum_{iy,ix} bilinear(F_{level_k}[b_k,c], y(ph,iy), x(pw,ix))
//
// Two kernels:
//  * fwd_cl_kernel   channels-last fast path: one CTA per RoI.  The RoI's level, image and its
//                    per-axis sample tables (pixel offsets + bilinear weights, computed ONCE per
//                    sample and reused by every channel -- north_star) are staged in shared memory;
//                    then threads are laid out (channel-vector, bin): each 128-bit load covers 4
//                    fp32 / 8 half channels of one tap, a warp reads 512 contiguous bytes.
//  * fwd_generic_kernel  any strides / any C / adaptive sampling: one thread per output element.
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

constexpr int kTable = 64;  // max samples per axis (out_size * sampling_ratio) of the fast path

struct AxisEntry {
  int lo, hi;     // element offsets of the two taps (already multiplied by the axis stride)
  float wl, wh;   // weights of hi / lo; both 0 when the sample is outside the map (reading S6)
};

template <typename T, int G>
__global__ void __launch_bounds__(256)
fwd_cl_kernel(const LevelsParam lv, const RoiArgs a, T* __restrict__ out, int64_t os_k, int64_t os_h,
              int64_t os_w) {
  using V = Vec16<T>;
  constexpr int VN = V::N;
  __shared__ AxisEntry s_y[kTable], s_x[kTable];
  __shared__ float s_inv_count;
  __shared__ int s_level, s_b;

  const int k = blockIdx.x;
  const int tid = threadIdx.y * blockDim.x + threadIdx.x;
  const int g = (G > 0) ? G : a.sampling_ratio;
  const int ny = a.PH * g, nx = a.PW * g;
  const float* r = a.rois + 5 * (int64_t)k;
  const float r0 = __ldg(r), x1 = __ldg(r + 1), y1 = __ldg(r + 2), x2 = __ldg(r + 3), y2 = __ldg(r + 4);
  const int level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);

  if (tid < ny + nx) {
    const RoiGeom geo = roi_geom(x1, y1, x2, y2, lv.scale[level], a.PH, a.PW, g, a.aligned);
    const bool isy = tid < ny;
    const int s = isy ? tid : tid - ny;
    const int p = s / g, i = s - p * g;
    const float v = isy ? sample_coord(geo.sy, geo.bh, p, i, g) : sample_coord(geo.sx, geo.bw, p, i, g);
    const AxisTap t = axis_tap(v, isy ? lv.h[level] : lv.w[level]);
    const int stride = (int)(isy ? lv.sh[level] : lv.sw[level]);
    AxisEntry e;
    e.lo = t.lo * stride;
    e.hi = t.hi * stride;
    e.wl = t.valid ? t.wl : 0.0f;
    e.wh = t.valid ? t.wh : 0.0f;
    if (isy) s_y[s] = e; else s_x[s] = e;
    if (tid == 0) {
      s_inv_count = geo.inv_count;
      s_level = level;
      s_b = batch_index_of(r0, lv.n);
    }
  }
  __syncthreads();

  const int b = s_b;
  const float inv_count = s_inv_count;
  const int CV = lv.c / VN;
  const int nbins = a.PH * a.PW;
  T* out_k = out + (int64_t)k * os_k;
  const T* base = (b >= 0) ? reinterpret_cast<const T*>(lv.data[level]) + (int64_t)b * lv.sn[level] : nullptr;

  for (int bin = threadIdx.y; bin < nbins; bin += blockDim.y) {
    const int ph = bin / a.PW, pw = bin - ph * a.PW;
    for (int cv = threadIdx.x; cv < CV; cv += blockDim.x) {
      float acc[VN];
#pragma unroll
      for (int j = 0; j < VN; ++j) acc[j] = 0.0f;
      if (b >= 0) {
        const T* bc = base + cv * VN;
#pragma unroll(G > 0 ? G : 1)
        for (int iy = 0; iy < g; ++iy) {
          const AxisEntry ey = s_y[ph * g + iy];
#pragma unroll(G > 0 ? G : 1)
          for (int ix = 0; ix < g; ++ix) {
            const AxisEntry ex = s_x[pw * g + ix];
            const float w1 = __fmul_rn(ey.wh, ex.wh), w2 = __fmul_rn(ey.wh, ex.wl);
            const float w3 = __fmul_rn(ey.wl, ex.wh), w4 = __fmul_rn(ey.wl, ex.wl);
            float v1[VN], v2[VN], v3[VN], v4[VN];
            V::load(bc + ey.lo + ex.lo, v1);
            V::load(bc + ey.lo + ex.hi, v2);
            V::load(bc + ey.hi + ex.lo, v3);
            V::load(bc + ey.hi + ex.hi, v4);
#pragma unroll
            for (int j = 0; j < VN; ++j)
              acc[j] += w1 * v1[j] + w2 * v2[j] + w3 * v3[j] + w4 * v4[j];
          }
        }
      }
#pragma unroll
      for (int j = 0; j < VN; ++j) acc[j] *= inv_count;
      V::store(out_k + ph * os_h + pw * os_w + cv * VN, acc);
    }
  }
}

template <typename T>
__global__ void __launch_bounds__(256)
fwd_generic_kernel(const LevelsParam lv, const RoiArgs a, T* __restrict__ out, int64_t os_k,
                   int64_t os_c, int64_t os_h, int64_t os_w, int64_t total) {
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int pw = (int)(idx % a.PW);
    const int ph = (int)((idx / a.PW) % a.PH);
    const int c = (int)((idx / ((int64_t)a.PW * a.PH)) % lv.c);
    const int k = (int)(idx / ((int64_t)a.PW * a.PH * lv.c));
    const float* r = a.rois + 5 * (int64_t)k;
    const float x1 = r[1], y1 = r[2], x2 = r[3], y2 = r[4];
    const int level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);
    const int b = batch_index_of(r[0], lv.n);
    float acc = 0.0f;
    if (b >= 0) {
      const RoiGeom geo = roi_geom(x1, y1, x2, y2, lv.scale[level], a.PH, a.PW, a.sampling_ratio, a.aligned);
      const int H = lv.h[level], W = lv.w[level];
      const int64_t sh = lv.sh[level], sw = lv.sw[level];
      const T* F = reinterpret_cast<const T*>(lv.data[level]) + b * lv.sn[level] + c * lv.sc[level];
      for (int iy = 0; iy < geo.gh; ++iy) {
        const AxisTap ty = axis_tap(sample_coord(geo.sy, geo.bh, ph, iy, geo.gh), H);
        if (!ty.valid) continue;
        for (int ix = 0; ix < geo.gw; ++ix) {
          const AxisTap tx = axis_tap(sample_coord(geo.sx, geo.bw, pw, ix, geo.gw), W);
          if (!tx.valid) continue;
          const float w1 = __fmul_rn(ty.wh, tx.wh), w2 = __fmul_rn(ty.wh, tx.wl);
          const float w3 = __fmul_rn(ty.wl, tx.wh), w4 = __fmul_rn(ty.wl, tx.wl);
          acc += w1 * Elem<T>::to_f32(F[ty.lo * sh + tx.lo * sw]) + w2 * Elem<T>::to_f32(F[ty.lo * sh + tx.hi * sw]) +
                 w3 * Elem<T>::to_f32(F[ty.hi * sh + tx.lo * sw]) + w4 * Elem<T>::to_f32(F[ty.hi * sh + tx.hi * sw]);
        }
      }
      acc *= geo.inv_count;
    }
    out[k * os_k + c * os_c + ph * os_h + pw * os_w] = Elem<T>::from_f32(acc);
  }
}

template <typename T>
static int forward_typed(const LevelsParam& lv, const RoiArgs& a, void* out, const int64_t* os,
                         bool channels_last, cudaStream_t stream) {
  T* o = reinterpret_cast<T*>(out);
  const int g = a.sampling_ratio;
  if (channels_last && g > 0 && a.PH * g <= kTable && a.PW * g <= kTable) {
    const int CV = lv.c / Vec16<T>::N;
    int bx = 1;
    while (bx < CV && bx < 256) bx <<= 1;
    const dim3 block(bx, 256 / bx);
    const dim3 grid(a.K);
    if (g == 2)
      fwd_cl_kernel<T, 2><<<grid, block, 0, stream>>>(lv, a, o, os[0], os[2], os[3]);
    else
      fwd_cl_kernel<T, 0><<<grid, block, 0, stream>>>(lv, a, o, os[0], os[2], os[3]);
  } else {
    const int64_t total = (int64_t)a.K * lv.c * a.PH * a.PW;
    const int64_t blocks = (total + 255) / 256;
    const int grid = (int)(blocks < (int64_t)148 * 64 ? blocks : (int64_t)148 * 64);
    fwd_generic_kernel<T><<<grid, 256, 0, stream>>>(lv, a, o, os[0], os[1], os[2], os[3], total);
  }
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

int launch_forward(const LevelsParam& lv, raf_dtype dtype, const RoiArgs& a, void* out,
                   const int64_t* out_strides, bool channels_last, cudaStream_t stream) {
  switch (dtype) {
    case RAF_F32: return forward_typed<float>(lv, a, out, out_strides, channels_last, stream);
    case RAF_F16: return forward_typed<__half>(lv, a, out, out_strides, channels_last, stream);
    case RAF_BF16: return forward_typed<__nv_bfloat16>(lv, a, out, out_strides, channels_last, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
