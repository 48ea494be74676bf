// raf_deform.cu -- multi-level (FPN) deformable RoI pooling, forward and backward ("DCN [8]: deformable
// convolution and deformable RoI pooling").  SURVEY.md 8(f) item 4; readings D1-D5 in
// RoIAlign (half-pixel shift, no minimum size) whose bin (ph, pw) is moved by
//     ox = (gamma * rw) * offset[k,0,ph,pw],   oy = (gamma * rh) * offset[k,1,ph,pw]      (feature pixels)
// i.e. sample (iy, ix) sits at the C3 coordinate plus ONE more fp32 addition; every sample then follows the C3
// tap rule (outside [-1,H] x [-1,W] -> 0, clamped at the borders); out = sum / count.  Backward: the exact
// transpose for the features (fp32 atomics), and for the offsets the derivative of the forward where it exists
// (a sample contributes hy*(F[yl,xh]-F[yl,xl]) + ly*(F[yh,xh]-F[yh,xl]) along x unless its x is clamped).
//
// Coordinates are formed with the explicitly rounded intrinsics of raf_device.cuh, in the oracle's order, so the
// taps and weights are bit-identical to the CPU checker (its fp32 "spec" mode); sums are fp32.  One thread per output
// element; with channels-last features consecutive lanes take consecutive channels of the same bin, so every
// tap is one coalesced load per warp and the offset gradient of a bin is reduced over the warp before it is
// added (one atomic per warp instead of one per channel).
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

struct DeformBin {
  float sx, sy, bw, bh, ox, oy, inv_count, grw, grh;   // grw = gamma * rw, grh = gamma * rh
  int gh, gw;
};

__device__ __forceinline__ DeformBin deform_bin(const float* __restrict__ r, float scale, int PH, int PW, int g,
                                                const float* __restrict__ offset, float gamma, int k, int ph, int pw) {
  const float x1 = __ldg(r + 1), y1 = __ldg(r + 2), x2 = __ldg(r + 3), y2 = __ldg(r + 4);
  DeformBin d;
  d.sx = __fsub_rn(__fmul_rn(x1, scale), 0.5f);
  d.sy = __fsub_rn(__fmul_rn(y1, scale), 0.5f);
  const float rw = __fsub_rn(__fsub_rn(__fmul_rn(x2, scale), 0.5f), d.sx);
  const float rh = __fsub_rn(__fsub_rn(__fmul_rn(y2, scale), 0.5f), d.sy);
  d.bw = __fdiv_rn(rw, (float)PW);
  d.bh = __fdiv_rn(rh, (float)PH);
  d.gh = sampling_grid(g, d.bh);
  d.gw = sampling_grid(g, d.bw);
  const int cnt = d.gh * d.gw;
  d.inv_count = 1.0f / (float)(cnt > 1 ? cnt : 1);
  d.grw = __fmul_rn(gamma, rw);
  d.grh = __fmul_rn(gamma, rh);
  const float dx = offset ? __ldg(offset + (((int64_t)k * 2 + 0) * PH + ph) * PW + pw) : 0.0f;
  const float dy = offset ? __ldg(offset + (((int64_t)k * 2 + 1) * PH + ph) * PW + pw) : 0.0f;
  d.ox = __fmul_rn(d.grw, dx);
  d.oy = __fmul_rn(d.grh, dy);
  return d;
}

__device__ __forceinline__ void deform_index(int64_t idx, int C, int PH, int PW, bool chan_fastest, int& k, int& c, int& ph,
                                             int& pw) {
  if (chan_fastest) {
    c = (int)(idx % C);
    pw = (int)((idx / C) % PW);
    ph = (int)((idx / ((int64_t)C * PW)) % PH);
    k = (int)(idx / ((int64_t)C * PW * PH));
  } else {
    pw = (int)(idx % PW);
    ph = (int)((idx / PW) % PH);
    c = (int)((idx / ((int64_t)PW * PH)) % C);
    k = (int)(idx / ((int64_t)PW * PH * C));
  }
}

template <typename T, bool kChanFastest>
__global__ void __launch_bounds__(256)
deform_fwd_kernel(const LevelsParam lv, const float* __restrict__ rois, const float* __restrict__ offset, float gamma, int PH,
                  int PW, int g, float finest_scale, T* __restrict__ out, int64_t os_k, int64_t os_c, int64_t os_h,
                  int64_t os_w, int64_t total) {
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    int k, c, ph, pw;
    deform_index(idx, lv.c, PH, PW, kChanFastest, k, c, ph, pw);
    const float* r = rois + 5 * (int64_t)k;
    const int b = batch_index_of(__ldg(r), lv.n);
    float acc = 0.0f;
    if (b >= 0) {
      const int level = level_of(__ldg(r + 1), __ldg(r + 2), __ldg(r + 3), __ldg(r + 4), lv.L, finest_scale);
      const DeformBin d = deform_bin(r, lv.scale[level], PH, PW, g, offset, gamma, k, ph, pw);
      const int H = lv.h[level], W = lv.w[level];
      const int64_t sh = lv.sh[level], sw = lv.sw[level];
      const T* F = reinterpret_cast<const T*>(lv.data[level]) + b * lv.sn[level] + c * lv.sc[level];
      for (int iy = 0; iy < d.gh; ++iy) {
        const AxisTap ty = axis_tap(__fadd_rn(sample_coord(d.sy, d.bh, ph, iy, d.gh), d.oy), H);
        if (!ty.valid) continue;
        for (int ix = 0; ix < d.gw; ++ix) {
          const AxisTap tx = axis_tap(__fadd_rn(sample_coord(d.sx, d.bw, pw, ix, d.gw), d.ox), W);
          if (!tx.valid) continue;
          const float w1 = __fmul_rn(ty.wh, tx.wh), w2 = __fmul_rn(ty.wh, tx.wl);
          const float w3 = __fmul_rn(ty.wl, tx.wh), w4 = __fmul_rn(ty.wl, tx.wl);
          acc += w1 * Elem<T>::to_f32(__ldg(F + ty.lo * sh + tx.lo * sw)) + w2 * Elem<T>::to_f32(__ldg(F + ty.lo * sh + tx.hi * sw)) +
                 w3 * Elem<T>::to_f32(__ldg(F + ty.hi * sh + tx.lo * sw)) + w4 * Elem<T>::to_f32(__ldg(F + ty.hi * sh + tx.hi * sw));
        }
      }
      acc *= d.inv_count;
    }
    out[k * os_k + c * os_c + ph * os_h + pw * os_w] = Elem<T>::from_f32(acc);
  }
}

// feats: the forward's features (read for the offset gradient); glv.data[l] == nullptr: no feature gradient.
template <typename T, bool kChanFastest>
__global__ void __launch_bounds__(256)
deform_bwd_kernel(const LevelsParam lv, const LevelsParam glv, bool want_feats, const float* __restrict__ rois,
                  const float* __restrict__ offset, float gamma, int PH, int PW, int g, float finest_scale,
                  const T* __restrict__ gout, int64_t gs_k, int64_t gs_c, int64_t gs_h, int64_t gs_w,
                  float* __restrict__ grad_offset, int64_t total, bool warp_reduce) {
  const int64_t span = (int64_t)gridDim.x * blockDim.x;
  const int64_t rounds = (total + span - 1) / span;   // every thread runs every round: the warp reductions stay convergent
  for (int64_t rd = 0; rd < rounds; ++rd) {
    const int64_t idx = rd * span + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = idx < total;
    int k = 0, c = 0, ph = 0, pw = 0;
    float gx = 0.0f, gy = 0.0f;
    bool valid = false;
    if (live) {
      deform_index(idx, lv.c, PH, PW, kChanFastest, k, c, ph, pw);
      const float* r = rois + 5 * (int64_t)k;
      const int b = batch_index_of(__ldg(r), lv.n);
      if (b >= 0) {
        valid = true;
        const int level = level_of(__ldg(r + 1), __ldg(r + 2), __ldg(r + 3), __ldg(r + 4), lv.L, finest_scale);
        const DeformBin d = deform_bin(r, lv.scale[level], PH, PW, g, offset, gamma, k, ph, pw);
        const int H = lv.h[level], W = lv.w[level];
        const float go = Elem<T>::to_f32(__ldg(gout + k * gs_k + c * gs_c + ph * gs_h + pw * gs_w)) * d.inv_count;
        const T* F = reinterpret_cast<const T*>(lv.data[level]) + b * lv.sn[level] + c * lv.sc[level];
        const int64_t fsh = lv.sh[level], fsw = lv.sw[level];
        float* G = want_feats ? reinterpret_cast<float*>(const_cast<void*>(glv.data[level])) + b * glv.sn[level] + c * glv.sc[level]
                              : nullptr;
        const int64_t gsh = glv.sh[level], gsw = glv.sw[level];
        float ax = 0.0f, ay = 0.0f;
        for (int iy = 0; iy < d.gh; ++iy) {
          const float yv = __fadd_rn(sample_coord(d.sy, d.bh, ph, iy, d.gh), d.oy);
          const AxisTap ty = axis_tap(yv, H);
          if (!ty.valid) continue;
          const bool yin = yv > 0.0f && ty.lo < ty.hi;
          for (int ix = 0; ix < d.gw; ++ix) {
            const float xv = __fadd_rn(sample_coord(d.sx, d.bw, pw, ix, d.gw), d.ox);
            const AxisTap tx = axis_tap(xv, W);
            if (!tx.valid) continue;
            const bool xin = xv > 0.0f && tx.lo < tx.hi;
            if (G) {
              atomicAdd(G + ty.lo * gsh + tx.lo * gsw, __fmul_rn(ty.wh, tx.wh) * go);
              atomicAdd(G + ty.lo * gsh + tx.hi * gsw, __fmul_rn(ty.wh, tx.wl) * go);
              atomicAdd(G + ty.hi * gsh + tx.lo * gsw, __fmul_rn(ty.wl, tx.wh) * go);
              atomicAdd(G + ty.hi * gsh + tx.hi * gsw, __fmul_rn(ty.wl, tx.wl) * go);
            }
            if (grad_offset) {
              const float f1 = Elem<T>::to_f32(__ldg(F + ty.lo * fsh + tx.lo * fsw)), f2 = Elem<T>::to_f32(__ldg(F + ty.lo * fsh + tx.hi * fsw));
              const float f3 = Elem<T>::to_f32(__ldg(F + ty.hi * fsh + tx.lo * fsw)), f4 = Elem<T>::to_f32(__ldg(F + ty.hi * fsh + tx.hi * fsw));
              if (xin) ax += ty.wh * (f2 - f1) + ty.wl * (f4 - f3);
              if (yin) ay += tx.wh * (f3 - f1) + tx.wl * (f4 - f2);
            }
          }
        }
        gx = go * ax * d.grw;
        gy = go * ay * d.grh;
      }
    }
    if (!grad_offset) continue;
    if (warp_reduce) {   // channel fastest and C % 32 == 0: the 32 lanes of a warp hold 32 channels of ONE bin
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        gx += __shfl_xor_sync(0xffffffffu, gx, o);
        gy += __shfl_xor_sync(0xffffffffu, gy, o);
      }
      if ((threadIdx.x & 31) == 0 && live && valid) {
        atomicAdd(grad_offset + (((int64_t)k * 2 + 0) * PH + ph) * PW + pw, gx);
        atomicAdd(grad_offset + (((int64_t)k * 2 + 1) * PH + ph) * PW + pw, gy);
      }
    } else if (live && valid) {
      atomicAdd(grad_offset + (((int64_t)k * 2 + 0) * PH + ph) * PW + pw, gx);
      atomicAdd(grad_offset + (((int64_t)k * 2 + 1) * PH + ph) * PW + pw, gy);
    }
  }
}

static int deform_grid(int64_t total) {
  const int64_t blocks = (total + 255) / 256;
  return (int)(blocks < (int64_t)148 * 64 ? blocks : (int64_t)148 * 64);
}

template <typename T>
static int deform_fwd_typed(const LevelsParam& lv, const float* rois, int K, const float* offset, float gamma, int PH, int PW,
                            int g, float fs, void* out, const int64_t* os, bool chan_fastest, cudaStream_t stream) {
  const int64_t total = (int64_t)K * lv.c * PH * PW;
  T* o = reinterpret_cast<T*>(out);
  if (chan_fastest)
    deform_fwd_kernel<T, true><<<deform_grid(total), 256, 0, stream>>>(lv, rois, offset, gamma, PH, PW, g, fs, o, os[0], os[1], os[2], os[3], total);
  else
    deform_fwd_kernel<T, false><<<deform_grid(total), 256, 0, stream>>>(lv, rois, offset, gamma, PH, PW, g, fs, o, os[0], os[1], os[2], os[3], total);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

template <typename T>
static int deform_bwd_typed(const LevelsParam& lv, const LevelsParam& glv, bool want_feats, const float* rois, int K,
                            const float* offset, float gamma, int PH, int PW, int g, float fs, const void* gout,
                            const int64_t* gs, float* grad_offset, bool chan_fastest, cudaStream_t stream) {
  const int64_t total = (int64_t)K * lv.c * PH * PW;
  const T* go = reinterpret_cast<const T*>(gout);
  const bool warp_reduce = chan_fastest && lv.c % 32 == 0;
  if (chan_fastest)
    deform_bwd_kernel<T, true><<<deform_grid(total), 256, 0, stream>>>(lv, glv, want_feats, rois, offset, gamma, PH, PW, g, fs, go, gs[0], gs[1],
                                                                       gs[2], gs[3], grad_offset, total, warp_reduce);
  else
    deform_bwd_kernel<T, false><<<deform_grid(total), 256, 0, stream>>>(lv, glv, want_feats, rois, offset, gamma, PH, PW, g, fs, go, gs[0], gs[1],
                                                                        gs[2], gs[3], grad_offset, total, false);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

int launch_deform_forward(const LevelsParam& lv, raf_dtype dtype, const float* rois, int K, const float* offset, float gamma,
                          int PH, int PW, int g, float fs, void* out, const int64_t* os, bool chan_fastest, cudaStream_t stream) {
  switch (dtype) {
    case RAF_F32: return deform_fwd_typed<float>(lv, rois, K, offset, gamma, PH, PW, g, fs, out, os, chan_fastest, stream);
    case RAF_F16: return deform_fwd_typed<__half>(lv, rois, K, offset, gamma, PH, PW, g, fs, out, os, chan_fastest, stream);
    case RAF_BF16: return deform_fwd_typed<__nv_bfloat16>(lv, rois, K, offset, gamma, PH, PW, g, fs, out, os, chan_fastest, stream);
  }
  return RAF_ERR_DTYPE;
}

int launch_deform_backward(const LevelsParam& lv, const LevelsParam& glv, bool want_feats, raf_dtype dtype, const float* rois,
                           int K, const float* offset, float gamma, int PH, int PW, int g, float fs, const void* gout,
                           const int64_t* gs, float* grad_offset, bool chan_fastest, cudaStream_t stream) {
  switch (dtype) {
    case RAF_F32: return deform_bwd_typed<float>(lv, glv, want_feats, rois, K, offset, gamma, PH, PW, g, fs, gout, gs, grad_offset, chan_fastest, stream);
    case RAF_F16: return deform_bwd_typed<__half>(lv, glv, want_feats, rois, K, offset, gamma, PH, PW, g, fs, gout, gs, grad_offset, chan_fastest, stream);
    case RAF_BF16: return deform_bwd_typed<__nv_bfloat16>(lv, glv, want_feats, rois, K, offset, gamma, PH, PW, g, fs, gout, gs, grad_offset, chan_fastest, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
