// raf_ref.cpp -- CPU ORACLE for multi-level (FPN) RoIAlign forward / backward.
//
// THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
// table or helper with the CUDA path (paper_1906_07155_b200/csrc/) and neither imports the other.
//
// What it follows.  The paper (section 3.1 "RoIExtractor ... extracts RoI-wise
// features from a single or multiple feature maps with RoIPooling-like operators ... from the
// corresponding level of feature pyramids ... SingleRoIExtractor") only NAMES the operation; the
// arithmetic is BASELINE.json `north_star` plus the public definition of RoIAlign (Mask R-CNN, the
// paper's ref [13]) as restated in SURVEY.md section 8(c), points C1..C5.  Every
// function below cites the point it follows.  Readings of silent points: DESIGN.md section 3.
//
// It is the definition written out: one loop nest per output element, no blocking, no fusion,
// no reordering.  Two numeric modes (reading S9):
//   coord_f32 = 1  "spec mode": sample coordinates and bilinear weights in fp32, each operation
//                  individually rounded in the canonical order (compile with -ffp-contract=off);
//                  products and sums in double.
//   coord_f32 = 0  "f64 mode": the same formulas entirely in double (used for closed-form pins).
// No excess precision or contraction: built for x86-64 SSE2 with -ffp-contract=off, no -ffast-math
// (oracle/build.py; tests assert the flags).
// Features, grad_out and results are double, logical NCHW / [K,C,PH,PW] contiguous; callers widen
// fp16/bf16/fp32 inputs exactly before calling.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"): worked level values, constant / affine /
// integer-aligned closed forms, edge rule, adjoint identity, dense-operator brute force, an
// independent library routine on the single-level case, and the worked example of SURVEY 8(c).
// Nothing here is "parity unpinned".
#include <cmath>
#include <cstdint>
#include <cstring>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

// One pyramid level, host memory, double, contiguous logical [N,C,H,W].
typedef struct {
  double* data;
  int32_t n, c, h, w;
  float spatial_scale;  // 1/stride of the level
} raf_ref_level;

// ---------------------------------------------------------------------------------------------
// C1: level assignment.  fp32, every operation individually rounded:
//   w = x2-x1; h = y2-y1; a = w*h; s = sqrt(a); q = s/finest_scale; t = q + 1e-6f;
//   level = #{ j in [1, L-1] : t >= 2^j }.
// Equals clamp(floor(log2 t), 0, L-1) with an exact log2 (reading S2); NaN -> 0 (reading S4).
// ---------------------------------------------------------------------------------------------
int32_t raf_ref_level_of(const float* roi, int L, float finest_scale) {
  float w = roi[3] - roi[1];
  float h = roi[4] - roi[2];
  float a = w * h;
  float s = sqrtf(a);
  float q = s / finest_scale;
  float t = q + 1e-6f;
  int32_t level = 0;
  float pow2 = 2.0f;
  for (int j = 1; j <= L - 1; ++j) {
    if (t >= pow2) level += 1;
    pow2 = pow2 * 2.0f;  // exact
  }
  return level;
}

// ---------------------------------------------------------------------------------------------
// C1 + C2: levels[K], counts[L], perm[K] (stable bucketing: perm lists the RoIs of level 0 in
// ascending k, then level 1, ...).
// ---------------------------------------------------------------------------------------------
int roi_fpn_assign_levels_ref(const float* rois, int K, int L, float finest_scale,
                              int32_t* levels, int32_t* counts, int32_t* perm) {
  if (K < 0 || L < 1) return -2;
  for (int l = 0; l < L; ++l) counts[l] = 0;
  for (int k = 0; k < K; ++k) {
    levels[k] = raf_ref_level_of(rois + 5 * (int64_t)k, L, finest_scale);
    counts[levels[k]] += 1;
  }
  int32_t pos = 0;
  for (int l = 0; l < L; ++l)
    for (int k = 0; k < K; ++k)
      if (levels[k] == l) perm[pos++] = k;
  return 0;
}

}  // extern "C"

namespace {

// Geometry of one RoI on its level (C3, first block).  R = float (spec mode) or double (f64 mode).
template <typename R>
struct RoiGeom {
  R sx, sy, bw, bh;
  int gh, gw, count;
};

template <typename R>
RoiGeom<R> roi_geom(const float* roi, float spatial_scale, int PH, int PW, int sampling_ratio,
                    int aligned) {
  RoiGeom<R> g;
  const R scale = (R)spatial_scale;
  const R off = aligned ? (R)0.5 : (R)0.0;
  R sx = (R)roi[1] * scale;  sx = sx - off;   // mul, then sub
  R sy = (R)roi[2] * scale;  sy = sy - off;
  R ex = (R)roi[3] * scale;  ex = ex - off;
  R ey = (R)roi[4] * scale;  ey = ey - off;
  R rw = ex - sx;
  R rh = ey - sy;
  if (!aligned) {                                       // reading S5
    if (!(rw >= (R)1.0)) rw = (R)1.0;
    if (!(rh >= (R)1.0)) rh = (R)1.0;
  }
  R bw = rw / (R)PW;
  R bh = rh / (R)PH;
  g.sx = sx; g.sy = sy; g.bw = bw; g.bh = bh;
  if (sampling_ratio > 0) {
    g.gh = sampling_ratio; g.gw = sampling_ratio;
  } else {                                              // reading S7: adaptive
    g.gh = (int)std::ceil((R)bh);
    g.gw = (int)std::ceil((R)bw);
  }
  int cnt = g.gh * g.gw;
  g.count = cnt > 1 ? cnt : 1;
  if (g.gh <= 0 || g.gw <= 0) g.count = 1;
  return g;
}

// Sample coordinate (C3): start + p*bin + ((i + 0.5)*bin)/grid, in that order.
template <typename R>
R sample_coord(R start, R bin, int p, int i, int grid) {
  R a = (R)p * bin;
  R b = start + a;
  R c = ((R)i + (R)0.5) * bin;
  R d = c / (R)grid;
  R e = b + d;
  return e;
}

// The four taps of one bilinear sample (C3, second block).  Returns false when the sample lies
// outside [-1,H] x [-1,W] (reading S6: it then contributes 0 but still counts in `count`).
template <typename R>
struct Taps {
  int yl, yh, xl, xh;
  R w1, w2, w3, w4;  // (yl,xl) (yl,xh) (yh,xl) (yh,xh)
};

template <typename R>
bool bilinear_taps(R y, R x, int H, int W, Taps<R>* t) {
  if (y < (R)-1.0 || y > (R)H || x < (R)-1.0 || x > (R)W) return false;
  if (!(y == y) || !(x == x)) return false;  // NaN coordinates contribute nothing
  if (y <= (R)0) y = (R)0;
  if (x <= (R)0) x = (R)0;
  int yl = (int)y, xl = (int)x, yh, xh;
  if (yl >= H - 1) { yl = yh = H - 1; y = (R)yl; } else { yh = yl + 1; }
  if (xl >= W - 1) { xl = xh = W - 1; x = (R)xl; } else { xh = xl + 1; }
  R ly = y - (R)yl;
  R lx = x - (R)xl;
  R hy = (R)1.0 - ly;
  R hx = (R)1.0 - lx;
  R w1 = hy * hx;
  R w2 = hy * lx;
  R w3 = ly * hx;
  R w4 = ly * lx;
  t->yl = yl; t->yh = yh; t->xl = xl; t->xh = xh;
  t->w1 = w1; t->w2 = w2; t->w3 = w3; t->w4 = w4;
  return true;
}

// Reading S17: batch index must be an integer in [0, N); otherwise zero row / no gradient.
bool batch_index_of(const float* roi, int N, int* b) {
  float f = roi[0];
  if (!(f >= 0.0f) || !(f < (float)N)) return false;
  int i = (int)f;
  if ((float)i != f) return false;
  *b = i;
  return true;
}

// C3 + C5: forward for RoI k on its level.  out_k: [C,PH,PW] doubles.
template <typename R>
void forward_one(const raf_ref_level& lv, const float* roi, int PH, int PW, int sampling_ratio,
                 int aligned, double* out_k) {
  const int C = lv.c, H = lv.h, W = lv.w;
  for (int64_t i = 0; i < (int64_t)C * PH * PW; ++i) out_k[i] = 0.0;
  int b;
  if (!batch_index_of(roi, lv.n, &b)) return;
  RoiGeom<R> g = roi_geom<R>(roi, lv.spatial_scale, PH, PW, sampling_ratio, aligned);
  for (int c = 0; c < C; ++c) {
    const double* F = lv.data + ((int64_t)b * C + c) * H * W;
    for (int ph = 0; ph < PH; ++ph)
      for (int pw = 0; pw < PW; ++pw) {
        double sum = 0.0;
        for (int iy = 0; iy < g.gh; ++iy) {
          R y = sample_coord<R>(g.sy, g.bh, ph, iy, g.gh);
          for (int ix = 0; ix < g.gw; ++ix) {
            R x = sample_coord<R>(g.sx, g.bw, pw, ix, g.gw);
            Taps<R> t;
            if (!bilinear_taps<R>(y, x, H, W, &t)) continue;
            sum += (double)t.w1 * F[(int64_t)t.yl * W + t.xl] +
                   (double)t.w2 * F[(int64_t)t.yl * W + t.xh] +
                   (double)t.w3 * F[(int64_t)t.yh * W + t.xl] +
                   (double)t.w4 * F[(int64_t)t.yh * W + t.xh];
          }
        }
        out_k[((int64_t)c * PH + ph) * PW + pw] = sum / (double)g.count;
      }
  }
}

// C4: backward (exact transpose) for RoI k, channel range [c0,c1).  Adds into grad (and abs-sum S).
template <typename R>
void backward_one(const raf_ref_level& glv, double* S, const float* roi, int PH, int PW,
                  int sampling_ratio, int aligned, const double* gout_k, int c0, int c1) {
  const int C = glv.c, H = glv.h, W = glv.w;
  int b;
  if (!batch_index_of(roi, glv.n, &b)) return;
  RoiGeom<R> g = roi_geom<R>(roi, glv.spatial_scale, PH, PW, sampling_ratio, aligned);
  for (int c = c0; c < c1; ++c) {
    const int64_t plane = ((int64_t)b * C + c) * H * W;
    double* G = glv.data + plane;
    double* Sa = S ? S + plane : nullptr;
    for (int ph = 0; ph < PH; ++ph)
      for (int pw = 0; pw < PW; ++pw) {
        const double go = gout_k[((int64_t)c * PH + ph) * PW + pw] / (double)g.count;
        for (int iy = 0; iy < g.gh; ++iy) {
          R y = sample_coord<R>(g.sy, g.bh, ph, iy, g.gh);
          for (int ix = 0; ix < g.gw; ++ix) {
            R x = sample_coord<R>(g.sx, g.bw, pw, ix, g.gw);
            Taps<R> t;
            if (!bilinear_taps<R>(y, x, H, W, &t)) continue;
            const int64_t i1 = (int64_t)t.yl * W + t.xl, i2 = (int64_t)t.yl * W + t.xh;
            const int64_t i3 = (int64_t)t.yh * W + t.xl, i4 = (int64_t)t.yh * W + t.xh;
            const double v1 = (double)t.w1 * go, v2 = (double)t.w2 * go;
            const double v3 = (double)t.w3 * go, v4 = (double)t.w4 * go;
            G[i1] += v1; G[i2] += v2; G[i3] += v3; G[i4] += v4;
            if (Sa) { Sa[i1] += std::fabs(v1); Sa[i2] += std::fabs(v2);
                      Sa[i3] += std::fabs(v3); Sa[i4] += std::fabs(v4); }
          }
        }
      }
  }
}

bool levels_consistent(const raf_ref_level* lv, int L) {
  if (!lv || L < 1) return false;
  for (int l = 0; l < L; ++l) {
    if (!lv[l].data || lv[l].n < 1 || lv[l].c < 1 || lv[l].h < 1 || lv[l].w < 1) return false;
    if (lv[l].n != lv[0].n || lv[l].c != lv[0].c) return false;
  }
  return true;
}

}  // namespace

extern "C" {

// ---------------------------------------------------------------------------------------------
// C5: forward over the pyramid.  out: double [K,C,PH,PW] contiguous, row k in ORIGINAL RoI order.
// Parallel over RoIs (rows are independent) when built with OpenMP.
// ---------------------------------------------------------------------------------------------
int roi_align_fpn_forward_ref(const raf_ref_level* feats, int L, const float* rois, int K,
                              int out_h, int out_w, int sampling_ratio, int aligned,
                              float finest_scale, int coord_f32, double* out) {
  if (!levels_consistent(feats, L) || K < 0 || out_h < 1 || out_w < 1 || sampling_ratio < 0)
    return -2;
  const int64_t row = (int64_t)feats[0].c * out_h * out_w;
#pragma omp parallel for schedule(dynamic, 4)
  for (int k = 0; k < K; ++k) {
    const float* roi = rois + 5 * (int64_t)k;
    const int l = raf_ref_level_of(roi, L, finest_scale);
    if (coord_f32)
      forward_one<float>(feats[l], roi, out_h, out_w, sampling_ratio, aligned, out + row * k);
    else
      forward_one<double>(feats[l], roi, out_h, out_w, sampling_ratio, aligned, out + row * k);
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------
// C4: backward over the pyramid.  grad_feats[l].data: double [N,C,H_l,W_l]; overwritten unless
// `accumulate`.  abs_sum (optional, same shapes, one pointer per level) receives
// S = sum |w * gout / count| per element (tolerance scale of reading S11); always overwritten.
// Parallel over channels (channel planes are disjoint, so race-free and order-preserving per
// element: RoIs are visited in ascending k for every element).
// ---------------------------------------------------------------------------------------------
int roi_align_fpn_backward_ref(const raf_ref_level* grad_feats, double* const* abs_sum, int L,
                               const double* grad_out, const float* rois, int K, int out_h,
                               int out_w, int sampling_ratio, int aligned, float finest_scale,
                               int coord_f32, int accumulate) {
  if (!levels_consistent(grad_feats, L) || K < 0 || out_h < 1 || out_w < 1 || sampling_ratio < 0)
    return -2;
  const int C = grad_feats[0].c;
  for (int l = 0; l < L; ++l) {
    const int64_t n = (int64_t)grad_feats[l].n * C * grad_feats[l].h * grad_feats[l].w;
    if (!accumulate) std::memset(grad_feats[l].data, 0, sizeof(double) * n);
    if (abs_sum && abs_sum[l]) std::memset(abs_sum[l], 0, sizeof(double) * n);
  }
  const int64_t row = (int64_t)C * out_h * out_w;
#pragma omp parallel for schedule(dynamic, 1)
  for (int c = 0; c < C; ++c) {
    for (int k = 0; k < K; ++k) {
      const float* roi = rois + 5 * (int64_t)k;
      const int l = raf_ref_level_of(roi, L, finest_scale);
      double* S = (abs_sum && abs_sum[l]) ? abs_sum[l] : nullptr;
      if (coord_f32)
        backward_one<float>(grad_feats[l], S, roi, out_h, out_w, sampling_ratio, aligned,
                            grad_out + row * k, c, c + 1);
      else
        backward_one<double>(grad_feats[l], S, roi, out_h, out_w, sampling_ratio, aligned,
                             grad_out + row * k, c, c + 1);
    }
  }
  return 0;
}

// ---------------------------------------------------------------------------------------------
// Sample enumeration (C3) exposed for tests: marks every (y,x) a RoI touches on its level in
// mask_l [N,H_l,W_l] (uint8) -- the "union of touched pixels" U of SURVEY 8(d) -- spec mode.
// ---------------------------------------------------------------------------------------------
int roi_align_fpn_footprint_ref(uint8_t* const* masks, const raf_ref_level* shapes, int L,
                                const float* rois, int K, int out_h, int out_w,
                                int sampling_ratio, int aligned, float finest_scale) {
  if (K < 0 || L < 1) return -2;
  for (int k = 0; k < K; ++k) {
    const float* roi = rois + 5 * (int64_t)k;
    const int l = raf_ref_level_of(roi, L, finest_scale);
    const int H = shapes[l].h, W = shapes[l].w;
    int b;
    if (!batch_index_of(roi, shapes[l].n, &b)) continue;
    RoiGeom<float> g = roi_geom<float>(roi, shapes[l].spatial_scale, out_h, out_w,
                                       sampling_ratio, aligned);
    uint8_t* M = masks[l] + (int64_t)b * H * W;
    for (int ph = 0; ph < out_h; ++ph)
      for (int pw = 0; pw < out_w; ++pw)
        for (int iy = 0; iy < g.gh; ++iy)
          for (int ix = 0; ix < g.gw; ++ix) {
            float y = sample_coord<float>(g.sy, g.bh, ph, iy, g.gh);
            float x = sample_coord<float>(g.sx, g.bw, pw, ix, g.gw);
            Taps<float> t;
            if (!bilinear_taps<float>(y, x, H, W, &t)) continue;
            M[(int64_t)t.yl * W + t.xl] = 1; M[(int64_t)t.yl * W + t.xh] = 1;
            M[(int64_t)t.yh * W + t.xl] = 1; M[(int64_t)t.yh * W + t.xh] = 1;
          }
  }
  return 0;
}

int raf_ref_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
