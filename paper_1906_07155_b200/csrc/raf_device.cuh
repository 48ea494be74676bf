// raf_device.cuh -- device-side arithmetic shared by the raf kernels (sm_100a).
//
// Everything that decides WHERE a sample lands is done with explicitly rounded fp32 intrinsics
// (__fmul_rn / __fadd_rn / __fsub_rn / __fdiv_rn / __fsqrt_rn): ptxas may not contract them into
// FMAs, so sample coordinates and bilinear weights are bit-identical to the canonical operation
// order of SURVEY.md 8(c) C1/C3 (reading S9; H1: a contracted `sx + pw*bw` alone moves 1.4 % of
// outputs outside the forward tolerance).  Accumulation order is free and uses FMAs.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/raf.h"

namespace raf {

constexpr int kMaxLevels = 8;
constexpr int kMaxAdaptiveGrid = 1024;  // implementation cap on the adaptive sampling grid per axis

// Device-side copy of the level descriptors (passed by value as a kernel parameter).
struct LevelsParam {
  const void* data[kMaxLevels];
  int64_t sn[kMaxLevels], sc[kMaxLevels], sh[kMaxLevels], sw[kMaxLevels];
  int32_t h[kMaxLevels], w[kMaxLevels];
  float scale[kMaxLevels];
  int32_t n, c, L;
};

// C1: level = #{ j in [1,L-1] : t >= 2^j }, t = sqrt(w*h)/finest_scale + 1e-6f, fp32 step by step.
__device__ __forceinline__ int level_of(float x1, float y1, float x2, float y2, int L,
                                        float finest_scale) {
  const float w = __fsub_rn(x2, x1);
  const float h = __fsub_rn(y2, y1);
  const float a = __fmul_rn(w, h);
  const float s = __fsqrt_rn(a);
  const float q = __fdiv_rn(s, finest_scale);
  const float t = __fadd_rn(q, 1e-6f);
  int level = 0;
  float p = 2.0f;
  for (int j = 1; j < L; ++j) {
    level += (t >= p) ? 1 : 0;  // NaN compares false -> level 0 (reading S4)
    p *= 2.0f;
  }
  return level;
}

// Reading S17: batch index must be an integer in [0,N); returns -1 otherwise.
__device__ __forceinline__ int batch_index_of(float f, int N) {
  if (!(f >= 0.0f) || !(f < (float)N)) return -1;
  const int i = (int)f;
  return ((float)i == f) ? i : -1;
}

// Samples per bin along one axis: the fixed grid, or (reading S7, sampling_ratio == 0) ceil(bin size),
// 0 for a non-positive / NaN bin size, capped at kMaxAdaptiveGrid.
__device__ __forceinline__ int sampling_grid(int sampling_ratio, float bin) {
  if (sampling_ratio > 0) return sampling_ratio;
  const float c = ceilf(bin);
  return (c >= (float)kMaxAdaptiveGrid) ? kMaxAdaptiveGrid : ((c >= 1.0f) ? (int)c : 0);
}

// C3, first block: geometry of one RoI on its level.
struct RoiGeom {
  float sx, sy, bw, bh;
  int gh, gw;
  float inv_count;  // 1 / max(gh*gw, 1)
};

__device__ __forceinline__ RoiGeom roi_geom(float x1, float y1, float x2, float y2, float scale,
                                            int PH, int PW, int sampling_ratio, int aligned) {
  RoiGeom g;
  const float off = aligned ? 0.5f : 0.0f;
  const float sx = __fsub_rn(__fmul_rn(x1, scale), off);
  const float sy = __fsub_rn(__fmul_rn(y1, scale), off);
  const float ex = __fsub_rn(__fmul_rn(x2, scale), off);
  const float ey = __fsub_rn(__fmul_rn(y2, scale), off);
  float rw = __fsub_rn(ex, sx);
  float rh = __fsub_rn(ey, sy);
  if (!aligned) {
    if (!(rw >= 1.0f)) rw = 1.0f;
    if (!(rh >= 1.0f)) rh = 1.0f;
  }
  g.sx = sx;
  g.sy = sy;
  g.bw = __fdiv_rn(rw, (float)PW);
  g.bh = __fdiv_rn(rh, (float)PH);
  g.gh = sampling_grid(sampling_ratio, g.bh);
  g.gw = sampling_grid(sampling_ratio, g.bw);
  const int cnt = g.gh * g.gw;
  g.inv_count = 1.0f / (float)(cnt > 1 ? cnt : 1);
  return g;
}

// C3: start + p*bin + ((i + 0.5)*bin)/grid, each operation rounded, in that order.
__device__ __forceinline__ float sample_coord(float start, float bin, int p, int i, int grid) {
  const float a = __fadd_rn(start, __fmul_rn((float)p, bin));
  const float d = __fdiv_rn(__fmul_rn((float)i + 0.5f, bin), (float)grid);
  return __fadd_rn(a, d);
}

// One axis of a bilinear sample (C3, second block): the two taps and their weights.
struct AxisTap {
  int lo, hi;    // pixel indices
  float wl, wh;  // weight of `hi` (= fractional part l) and of `lo` (= 1 - l)
  int valid;     // 0 when the coordinate lies outside [-1, n] (reading S6) or is NaN
};

__device__ __forceinline__ AxisTap axis_tap(float v, int n) {
  AxisTap t;
  t.valid = (v >= -1.0f) && (v <= (float)n);  // false for NaN
  if (v <= 0.0f || !t.valid) v = 0.0f;
  int lo = (int)v;
  int hi;
  if (lo >= n - 1) {
    lo = hi = n - 1;
    v = (float)lo;
  } else {
    hi = lo + 1;
  }
  t.lo = lo;
  t.hi = hi;
  t.wl = __fsub_rn(v, (float)lo);
  t.wh = __fsub_rn(1.0f, t.wl);
  return t;
}

// ---- element type helpers ------------------------------------------------------------------------
template <typename T> struct Elem;
template <> struct Elem<float> {
  static __device__ __forceinline__ float to_f32(float v) { return v; }
  static __device__ __forceinline__ float from_f32(float v) { return v; }
};
template <> struct Elem<__half> {
  static __device__ __forceinline__ float to_f32(__half v) { return __half2float(v); }
  static __device__ __forceinline__ __half from_f32(float v) { return __float2half_rn(v); }
};
template <> struct Elem<__nv_bfloat16> {
  static __device__ __forceinline__ float to_f32(__nv_bfloat16 v) { return __bfloat162float(v); }
  static __device__ __forceinline__ __nv_bfloat16 from_f32(float v) { return __float2bfloat16_rn(v); }
};

// 16-byte vector of T, widened to fp32 lanes.
template <typename T> struct Vec16;
template <> struct Vec16<float> {
  static constexpr int N = 4;
  static __device__ __forceinline__ void load(const float* p, float (&v)[4]) {
    const float4 r = __ldg(reinterpret_cast<const float4*>(p));
    v[0] = r.x; v[1] = r.y; v[2] = r.z; v[3] = r.w;
  }
  static __device__ __forceinline__ void store(float* p, const float (&v)[4]) {
    *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
  }
};
template <> struct Vec16<__half> {
  static constexpr int N = 8;
  static __device__ __forceinline__ void load(const __half* p, float (&v)[8]) {
    const uint4 r = __ldg(reinterpret_cast<const uint4*>(p));
    const __half2* h = reinterpret_cast<const __half2*>(&r);
#pragma unroll
    for (int i = 0; i < 4; ++i) { const float2 f = __half22float2(h[i]); v[2 * i] = f.x; v[2 * i + 1] = f.y; }
  }
  static __device__ __forceinline__ uint4 load_raw(const __half* p) { return __ldg(reinterpret_cast<const uint4*>(p)); }
  static __device__ __forceinline__ void widen(const uint4& r, float (&v)[8]) {
    const __half2* h = reinterpret_cast<const __half2*>(&r);
#pragma unroll
    for (int i = 0; i < 4; ++i) { const float2 f = __half22float2(h[i]); v[2 * i] = f.x; v[2 * i + 1] = f.y; }
  }
  static __device__ __forceinline__ void store(__half* p, const float (&v)[8]) {
    uint4 r;
    __half2* h = reinterpret_cast<__half2*>(&r);
#pragma unroll
    for (int i = 0; i < 4; ++i) h[i] = __floats2half2_rn(v[2 * i], v[2 * i + 1]);
    *reinterpret_cast<uint4*>(p) = r;
  }
};
template <> struct Vec16<__nv_bfloat16> {
  static constexpr int N = 8;
  static __device__ __forceinline__ void load(const __nv_bfloat16* p, float (&v)[8]) {
    const uint4 r = __ldg(reinterpret_cast<const uint4*>(p));
    const uint32_t* u = reinterpret_cast<const uint32_t*>(&r);
#pragma unroll
    for (int i = 0; i < 4; ++i) {  // bf16 -> fp32 is a 16-bit shift
      v[2 * i] = __uint_as_float(u[i] << 16);
      v[2 * i + 1] = __uint_as_float(u[i] & 0xffff0000u);
    }
  }
  static __device__ __forceinline__ uint4 load_raw(const __nv_bfloat16* p) { return __ldg(reinterpret_cast<const uint4*>(p)); }
  static __device__ __forceinline__ void widen(const uint4& r, float (&v)[8]) {
    const uint32_t* u = reinterpret_cast<const uint32_t*>(&r);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      v[2 * i] = __uint_as_float(u[i] << 16);
      v[2 * i + 1] = __uint_as_float(u[i] & 0xffff0000u);
    }
  }
  static __device__ __forceinline__ void store(__nv_bfloat16* p, const float (&v)[8]) {
    uint4 r;
    __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&r);
#pragma unroll
    for (int i = 0; i < 4; ++i) h[i] = __floats2bfloat162_rn(v[2 * i], v[2 * i + 1]);
    *reinterpret_cast<uint4*>(p) = r;
  }
};

// 4 consecutive gradient channels of type G (the gradient pyramid is fp32, or -- roi_align_fpn_backward_ex -- the
// 16-bit type of grad_out: sums are formed in fp32 registers and rounded once when they are stored).
template <typename G> struct Grad4;
template <> struct Grad4<float> {
  static __device__ __forceinline__ float4 load(const float* p) { return *reinterpret_cast<const float4*>(p); }
  static __device__ __forceinline__ void store(float* p, const float4& v) { *reinterpret_cast<float4*>(p) = v; }
};
template <> struct Grad4<__half> {
  static __device__ __forceinline__ float4 load(const __half* p) {
    const uint2 r = *reinterpret_cast<const uint2*>(p);
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
    return make_float4(a.x, a.y, b.x, b.y);
  }
  static __device__ __forceinline__ void store(__half* p, const float4& v) {
    uint2 r;
    *reinterpret_cast<__half2*>(&r.x) = __floats2half2_rn(v.x, v.y);
    *reinterpret_cast<__half2*>(&r.y) = __floats2half2_rn(v.z, v.w);
    *reinterpret_cast<uint2*>(p) = r;
  }
};
template <> struct Grad4<__nv_bfloat16> {
  static __device__ __forceinline__ float4 load(const __nv_bfloat16* p) {
    const uint2 r = *reinterpret_cast<const uint2*>(p);
    return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u),
                       __uint_as_float(r.y << 16), __uint_as_float(r.y & 0xffff0000u));
  }
  static __device__ __forceinline__ void store(__nv_bfloat16* p, const float4& v) {
    uint2 r;
    *reinterpret_cast<__nv_bfloat162*>(&r.x) = __floats2bfloat162_rn(v.x, v.y);
    *reinterpret_cast<__nv_bfloat162*>(&r.y) = __floats2bfloat162_rn(v.z, v.w);
    *reinterpret_cast<uint2*>(p) = r;
  }
};

// fp32 vector reduction into global memory (sm_90+): one L2 atomic transaction for 16 bytes.
__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c),
               "f"(d)
               : "memory");
}

}  // namespace raf
