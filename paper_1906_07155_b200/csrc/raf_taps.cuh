// raf_taps.cuh -- merged separable bilinear taps of one output bin along one axis, shared by the forward
// (raf_forward.cu) and the fused gather + FC kernel (raf_fc.cu): the two produce bit-identical feature values.
#pragma once
#include "raf_device.cuh"

namespace raf {

// One merged bilinear tap of an output bin along one axis: element offset of the pixel (already
// multiplied by the axis stride) and its weight (y taps carry 1/count).
struct FwdTap {
  int off;
  float w;
};

// Merged taps of bin `bin` of one axis into tab[0..2g) (shared memory); returns the count.
// Equal pixels are merged (weights summed in sample order); invalid samples (reading S6) give no tap.
__device__ __forceinline__ int fwd_bin_taps(float start, float bsz, int bin, int g, int n, int stride,
                                            float scale_w, FwdTap* tab) {
  int cnt = 0;
  if (g <= 2) {   // usual case: merge in registers
    int pix[4] = {-1, -1, -1, -1};
    float w[4] = {0.f, 0.f, 0.f, 0.f};
    auto add = [&](int p, float v) {
      bool found = false;
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (q < cnt && pix[q] == p) { w[q] += v; found = true; }
      if (!found) {
#pragma unroll
        for (int q = 0; q < 4; ++q)
          if (q == cnt) { pix[q] = p; w[q] = v; }
        ++cnt;
      }
    };
    for (int i = 0; i < g; ++i) {
      const AxisTap t = axis_tap(sample_coord(start, bsz, bin, i, g), n);
      if (!t.valid) continue;
      add(t.lo, t.wh * scale_w);
      add(t.hi, t.wl * scale_w);
    }
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if (q < 2 * g) { tab[q].off = (q < cnt ? pix[q] : 0) * stride; tab[q].w = w[q]; }
    return cnt;
  }
  for (int i = 0; i < g; ++i) {
    const AxisTap t = axis_tap(sample_coord(start, bsz, bin, i, g), n);
    if (!t.valid) continue;
    const int po[2] = {t.lo * stride, t.hi * stride};
    const float pw[2] = {t.wh * scale_w, t.wl * scale_w};
    for (int h = 0; h < 2; ++h) {
      int q = 0;
      while (q < cnt && tab[q].off != po[h]) ++q;
      if (q < cnt) tab[q].w += pw[h];
      else { tab[cnt].off = po[h]; tab[cnt].w = pw[h]; ++cnt; }
    }
  }
  return cnt;
}

}  // namespace raf
