// raf_pool.cu -- multi-level (FPN) RoIPool-max forward / backward: the max variant of the "RoIPooling-like
// operators" the RoIExtractor applies (section 3.1; the RoI pooling layer of Fast R-CNN,
// PAPER.md:39).  SURVEY.md 8(f) item 1; readings P1-P4 in DESIGN.md 3b.
//
//   P1  window of bin (ph, pw): sw = roundf(x1*scale) ... ; rw = max(ew - sw + 1, 1); bw = rw / PW (fp32);
//       ws = clamp(floorf(pw*bw) + sw, 0, W), we = clamp(ceilf((pw+1)*bw) + sw, 0, W); rows likewise
//   P2  out = max of F over the window (0 when the window is empty or the batch index invalid)
//   P3  argmax = y*W + x of the FIRST maximum in row-major order (-1: none); NaN never wins
//   P4  backward: grad[level_k][b_k][c][argmax] += grad_out[k,c,ph,pw]
//
// Everything that decides an index is fp32 with explicitly rounded operations in the order written, so the
// windows (hence argmax and the values, which are copies of inputs) are bit-identical to the oracle's.
// One thread per output element; with channels-last features consecutive lanes take consecutive channels
// of the same bin, so every window pixel is one coalesced load per warp.  The backward scatters with
// `red.global.add.f32` (channels pick different pixels, so there is no vector form).
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

struct PoolWindow {
  int hs, he, ws, we;
};

__device__ __forceinline__ PoolWindow pool_window(float x1, float y1, float x2, float y2, float scale, int PH, int PW,
                                                  int ph, int pw, int H, int W) {
  const int sw = (int)roundf(__fmul_rn(x1, scale)), sh = (int)roundf(__fmul_rn(y1, scale));
  const int ew = (int)roundf(__fmul_rn(x2, scale)), eh = (int)roundf(__fmul_rn(y2, scale));
  const int rw = max(ew - sw + 1, 1), rh = max(eh - sh + 1, 1);
  const float bw = __fdiv_rn((float)rw, (float)PW), bh = __fdiv_rn((float)rh, (float)PH);
  PoolWindow o;
  o.hs = min(max((int)floorf(__fmul_rn((float)ph, bh)) + sh, 0), H);
  o.he = min(max((int)ceilf(__fmul_rn((float)(ph + 1), bh)) + sh, 0), H);
  o.ws = min(max((int)floorf(__fmul_rn((float)pw, bw)) + sw, 0), W);
  o.we = min(max((int)ceilf(__fmul_rn((float)(pw + 1), bw)) + sw, 0), W);
  return o;
}

// kChanFastest: idx = ((k*PH + ph)*PW + pw)*C + c (channels-last memory: a warp reads consecutive channels);
// else idx = ((k*C + c)*PH + ph)*PW + pw.
template <typename T, bool kChanFastest>
__global__ void __launch_bounds__(256)
pool_fwd_kernel(const LevelsParam lv, const float* __restrict__ rois, int PH, int PW, float finest_scale,
                T* __restrict__ out, int32_t* __restrict__ argmax, int64_t os_k, int64_t os_c, int64_t os_h, int64_t os_w,
                int64_t total) {
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    int k, c, ph, pw;
    if (kChanFastest) {
      c = (int)(idx % lv.c);
      pw = (int)((idx / lv.c) % PW);
      ph = (int)((idx / ((int64_t)lv.c * PW)) % PH);
      k = (int)(idx / ((int64_t)lv.c * PW * PH));
    } else {
      pw = (int)(idx % PW);
      ph = (int)((idx / PW) % PH);
      c = (int)((idx / ((int64_t)PW * PH)) % lv.c);
      k = (int)(idx / ((int64_t)PW * PH * lv.c));
    }
    const float* r = rois + 5 * (int64_t)k;
    const float r0 = __ldg(r), x1 = __ldg(r + 1), y1 = __ldg(r + 2), x2 = __ldg(r + 3), y2 = __ldg(r + 4);
    const int level = level_of(x1, y1, x2, y2, lv.L, finest_scale);
    const int b = batch_index_of(r0, lv.n);
    float best = 0.0f;
    int arg = -1;
    if (b >= 0) {
      const int H = lv.h[level], W = lv.w[level];
      const PoolWindow w = pool_window(x1, y1, x2, y2, lv.scale[level], PH, PW, ph, pw, H, W);
      const T* F = reinterpret_cast<const T*>(lv.data[level]) + b * lv.sn[level] + c * lv.sc[level];
      const int64_t sh = lv.sh[level], sw = lv.sw[level];
      for (int y = w.hs; y < w.he; ++y)
        for (int x = w.ws; x < w.we; ++x) {
          const float v = Elem<T>::to_f32(__ldg(F + y * sh + x * sw));
          if (v != v) continue;   // NaN never wins
          if (arg < 0 || v > best) { best = v; arg = y * W + x; }
        }
    }
    const int64_t o = k * os_k + c * os_c + ph * os_h + pw * os_w;
    out[o] = Elem<T>::from_f32(arg >= 0 ? best : 0.0f);   // a copy of an input element: exact
    if (argmax) argmax[o] = arg;
  }
}

template <typename T, bool kChanFastest>
__global__ void __launch_bounds__(256)
pool_bwd_kernel(const LevelsParam lv, const float* __restrict__ rois, int PH, int PW, float finest_scale,
                const T* __restrict__ gout, const int32_t* __restrict__ argmax, int64_t gs_k, int64_t gs_c, int64_t gs_h,
                int64_t gs_w, int64_t total) {
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    int k, c, ph, pw;
    if (kChanFastest) {
      c = (int)(idx % lv.c);
      pw = (int)((idx / lv.c) % PW);
      ph = (int)((idx / ((int64_t)lv.c * PW)) % PH);
      k = (int)(idx / ((int64_t)lv.c * PW * PH));
    } else {
      pw = (int)(idx % PW);
      ph = (int)((idx / PW) % PH);
      c = (int)((idx / ((int64_t)PW * PH)) % lv.c);
      k = (int)(idx / ((int64_t)PW * PH * lv.c));
    }
    const int64_t o = k * gs_k + c * gs_c + ph * gs_h + pw * gs_w;
    const int a = __ldg(argmax + o);
    if (a < 0) continue;
    const float* r = rois + 5 * (int64_t)k;
    const int b = batch_index_of(__ldg(r), lv.n);
    if (b < 0) continue;
    const int level = level_of(__ldg(r + 1), __ldg(r + 2), __ldg(r + 3), __ldg(r + 4), lv.L, finest_scale);
    const int W = lv.w[level];
    if (a >= lv.h[level] * W) continue;   // not an index of this level: ignore (memory safety)
    float* G = reinterpret_cast<float*>(const_cast<void*>(lv.data[level])) + b * lv.sn[level] + c * lv.sc[level] +
               (a / W) * lv.sh[level] + (a % W) * lv.sw[level];
    atomicAdd(G, Elem<T>::to_f32(__ldg(gout + o)));
  }
}

static int pool_grid(int64_t total) {
  const int64_t blocks = (total + 255) / 256;
  return (int)(blocks < (int64_t)148 * 64 ? blocks : (int64_t)148 * 64);
}

template <typename T>
static int pool_fwd_typed(const LevelsParam& lv, const float* rois, int K, int PH, int PW, float fs, void* out,
                          int32_t* argmax, const int64_t* os, bool chan_fastest, cudaStream_t stream) {
  const int64_t total = (int64_t)K * lv.c * PH * PW;
  T* o = reinterpret_cast<T*>(out);
  if (chan_fastest)
    pool_fwd_kernel<T, true><<<pool_grid(total), 256, 0, stream>>>(lv, rois, PH, PW, fs, o, argmax, os[0], os[1], os[2], os[3], total);
  else
    pool_fwd_kernel<T, false><<<pool_grid(total), 256, 0, stream>>>(lv, rois, PH, PW, fs, o, argmax, os[0], os[1], os[2], os[3], total);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

template <typename T>
static int pool_bwd_typed(const LevelsParam& lv, const float* rois, int K, int PH, int PW, float fs, const void* gout,
                          const int32_t* argmax, const int64_t* gs, bool chan_fastest, cudaStream_t stream) {
  const int64_t total = (int64_t)K * lv.c * PH * PW;
  const T* g = reinterpret_cast<const T*>(gout);
  if (chan_fastest)
    pool_bwd_kernel<T, true><<<pool_grid(total), 256, 0, stream>>>(lv, rois, PH, PW, fs, g, argmax, gs[0], gs[1], gs[2], gs[3], total);
  else
    pool_bwd_kernel<T, false><<<pool_grid(total), 256, 0, stream>>>(lv, rois, PH, PW, fs, g, argmax, gs[0], gs[1], gs[2], gs[3], total);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

int launch_pool_forward(const LevelsParam& lv, raf_dtype dtype, const float* rois, int K, int PH, int PW, float fs,
                        void* out, int32_t* argmax, const int64_t* os, bool chan_fastest, cudaStream_t stream) {
  switch (dtype) {
    case RAF_F32: return pool_fwd_typed<float>(lv, rois, K, PH, PW, fs, out, argmax, os, chan_fastest, stream);
    case RAF_F16: return pool_fwd_typed<__half>(lv, rois, K, PH, PW, fs, out, argmax, os, chan_fastest, stream);
    case RAF_BF16: return pool_fwd_typed<__nv_bfloat16>(lv, rois, K, PH, PW, fs, out, argmax, os, chan_fastest, stream);
  }
  return RAF_ERR_DTYPE;
}

int launch_pool_backward(const LevelsParam& glv, raf_dtype dtype, const float* rois, int K, int PH, int PW, float fs,
                         const void* gout, const int32_t* argmax, const int64_t* gs, bool chan_fastest, cudaStream_t stream) {
  switch (dtype) {
    case RAF_F32: return pool_bwd_typed<float>(glv, rois, K, PH, PW, fs, gout, argmax, gs, chan_fastest, stream);
    case RAF_F16: return pool_bwd_typed<__half>(glv, rois, K, PH, PW, fs, gout, argmax, gs, chan_fastest, stream);
    case RAF_BF16: return pool_bwd_typed<__nv_bfloat16>(glv, rois, K, PH, PW, fs, gout, argmax, gs, chan_fastest, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
