// ops_ref.cpp -- CPU ORACLE for the SURVEY 8(f) "next" operations around the RoIAlign hot path:
//   * multi-level (FPN) RoIPool-max forward / backward  ("RoIPooling-like operators", section
//     3.1 RoIExtractor; the max variant is the RoI pooling layer of Fast R-CNN);
//   * greedy NMS and Soft-NMS on boxes ("Soft NMS [1]: an alternative to NMS"; "All basic
//     bbox and mask operations run on GPUs");
//   * deformable RoI pooling forward / backward ("DCN [8]: deformable convolution and deformable RoI pooling",
//     PAPER.md:57-58): RoIAlign whose bins are shifted by per-bin offsets (readings D1-D5).
//
// THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load it.  It shares no code, header, table or helper with the
// CUDA path (paper_1906_07155_b200/csrc/) and neither imports the other.
//
// The paper gives no formula for any of these; the readings are listed in DESIGN.md section 3b (P1-P4,
// N1-N6).  Each function below is its definition written out: one loop nest, no blocking, no fusion.
// Arithmetic that decides an INTEGER (a quantised bin edge, a suppression, a selection) is fp32 with every
// operation individually rounded, in the order written (built with -ffp-contract=off, no fast-math), so that
// the CUDA path can take the same decision in the same precision; values are compared, never transformed.
//
// Pins (tests/test_oracle_ops.py, -m "not gpu"): RoIPool -- constant map, monotone ramp (closed form: value
// at the last pixel of the bin), integer-aligned identity crop, empty bins, an independent library routine
// (torchvision.ops.roi_pool, CPU float64) on the single-level case, backward = scatter of grad_out to the
// recorded argmax (mass conservation, brute force).  NMS -- hand-worked 5-box example, threshold edge,
// permutation invariance, brute-force O(n^2) restatement on tiny inputs via the library routine
// torchvision.ops.nms, idempotence.  Soft-NMS -- hand-worked 3-box example (linear and Gaussian), reduction
// to a score sort when no boxes overlap.  Deformable RoI pooling -- zero offsets == the RoIAlign oracle
// (oracle/raf_ref.cpp, itself pinned) bit for bit; a uniform offset == RoIAlign of the translated box (f64
// mode, 1e-12); an offset on one bin changes that bin only; adjoint identity for the feature gradient;
// central finite differences of the f64 forward for the offset gradient; constant map -> zero offset
// gradient.  Nothing here is "parity unpinned".
#include <cfloat>
#include <cmath>
#include <cstdint>
#include <cstring>

extern "C" {

typedef struct {
  double* data;          // [N,C,H,W] contiguous (features: read; gradients: written)
  int32_t n, c, h, w;
  float spatial_scale;
} ops_ref_level;

// C1 of the RoIAlign path (same rule, restated: the level map is shared by every RoI extractor).
static int32_t level_of(const float* roi, int L, float finest_scale) {
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
    pow2 = pow2 * 2.0f;
  }
  return level;
}

static int batch_index_of(float f, int N) {   // reading S17
  if (!(f >= 0.0f) || !(f < (float)N)) return -1;
  int i = (int)f;
  return ((float)i == f) ? i : -1;
}

// P1: quantised window of bin (ph, pw) of a RoI on a level of size H x W (fp32, each op rounded):
//   sw = roundf(x1*scale) ... ;  rw = max(ew - sw + 1, 1);  bw = (float)rw / (float)PW;
//   ws = clamp((int)floorf((float)pw * bw) + sw, 0, W);  we = clamp((int)ceilf((float)(pw+1) * bw) + sw, 0, W)
static void pool_window(const float* roi, float scale, int PH, int PW, int ph, int pw, int H, int W,
                        int* hs, int* he, int* ws, int* we) {
  const int sw = (int)roundf(roi[1] * scale), sh = (int)roundf(roi[2] * scale);
  const int ew = (int)roundf(roi[3] * scale), eh = (int)roundf(roi[4] * scale);
  int rw = ew - sw + 1, rh = eh - sh + 1;
  if (rw < 1) rw = 1;
  if (rh < 1) rh = 1;
  const float bw = (float)rw / (float)PW, bh = (float)rh / (float)PH;
  int a = (int)floorf((float)ph * bh) + sh, b = (int)ceilf((float)(ph + 1) * bh) + sh;
  *hs = a < 0 ? 0 : (a > H ? H : a);
  *he = b < 0 ? 0 : (b > H ? H : b);
  a = (int)floorf((float)pw * bw) + sw;
  b = (int)ceilf((float)(pw + 1) * bw) + sw;
  *ws = a < 0 ? 0 : (a > W ? W : a);
  *we = b < 0 ? 0 : (b > W ? W : b);
}

// P2 + P3: out[k,c,ph,pw] = max of F over the bin's window (0 for an empty window or an invalid batch
// index); argmax[k,c,ph,pw] = y*W + x of the FIRST maximum in row-major order (-1 when there is none).
// NaN never wins a comparison.
int roi_pool_fpn_forward_ref(const ops_ref_level* feats, int L, const float* rois, int K, int PH, int PW,
                             float finest_scale, double* out, int32_t* argmax) {
  const int C = feats[0].c;
  for (int k = 0; k < K; ++k) {
    const float* roi = rois + 5 * (int64_t)k;
    const int l = level_of(roi, L, finest_scale);
    const ops_ref_level& lv = feats[l];
    const int b = batch_index_of(roi[0], lv.n);
    for (int c = 0; c < C; ++c)
      for (int ph = 0; ph < PH; ++ph)
        for (int pw = 0; pw < PW; ++pw) {
          const int64_t o = (((int64_t)k * C + c) * PH + ph) * PW + pw;
          double best = 0.0;
          int32_t arg = -1;
          if (b >= 0) {
            int hs, he, ws, we;
            pool_window(roi, lv.spatial_scale, PH, PW, ph, pw, lv.h, lv.w, &hs, &he, &ws, &we);
            const double* F = lv.data + ((int64_t)b * C + c) * lv.h * lv.w;
            for (int y = hs; y < he; ++y)
              for (int x = ws; x < we; ++x) {
                const double v = F[(int64_t)y * lv.w + x];
                if (v != v) continue;                       // NaN
                if (arg < 0 || v > best) { best = v; arg = y * lv.w + x; }
              }
          }
          out[o] = arg >= 0 ? best : 0.0;
          if (argmax) argmax[o] = arg;
        }
  }
  return 0;
}

// P4: backward = transpose of the selection: grad[level_k][b_k][c][argmax] += grad_out[k,c,ph,pw].
// The gradient pyramid must hold its starting values (zeros in overwrite mode).
int roi_pool_fpn_backward_ref(const ops_ref_level* grads, int L, const double* grad_out, const int32_t* argmax,
                              const float* rois, int K, int PH, int PW, float finest_scale) {
  const int C = grads[0].c;
  for (int k = 0; k < K; ++k) {
    const float* roi = rois + 5 * (int64_t)k;
    const int l = level_of(roi, L, finest_scale);
    const ops_ref_level& lv = grads[l];
    const int b = batch_index_of(roi[0], lv.n);
    if (b < 0) continue;
    for (int c = 0; c < C; ++c)
      for (int p = 0; p < PH * PW; ++p) {
        const int64_t o = ((int64_t)k * C + c) * PH * PW + p;
        if (argmax[o] >= 0) lv.data[((int64_t)b * C + c) * lv.h * lv.w + argmax[o]] += grad_out[o];
      }
  }
  return 0;
}

// N2: IoU of two boxes (x1,y1,x2,y2), continuous coordinates (no "+1"), fp32, each op rounded:
//   iw = max(min(ax2,bx2) - max(ax1,bx1), 0);  ih likewise;  inter = iw*ih;
//   ua = (area_a + area_b) - inter;  iou = inter / ua        (0/0 = NaN: compares false everywhere)
float ops_ref_iou(const float* a, const float* b) {
  float iw = fminf(a[2], b[2]) - fmaxf(a[0], b[0]);
  float ih = fminf(a[3], b[3]) - fmaxf(a[1], b[1]);
  if (!(iw > 0.0f)) iw = 0.0f;
  if (!(ih > 0.0f)) ih = 0.0f;
  const float inter = iw * ih;
  const float aa = (a[2] - a[0]) * (a[3] - a[1]);
  const float ab = (b[2] - b[0]) * (b[3] - b[1]);
  const float ua = (aa + ab) - inter;
  return inter / ua;
}

// N1: order[] = indices by descending score, ties by ascending index (stable).  Plain insertion sort.
static void order_by_score(const float* scores, int n, int32_t* order) {
  for (int i = 0; i < n; ++i) {
    int j = i;
    while (j > 0 && scores[order[j - 1]] < scores[i]) { order[j] = order[j - 1]; --j; }
    order[j] = i;
  }
}

// N3: greedy NMS.  keep[] receives the kept indices in descending-score order; returns their number.
// A box is suppressed by an earlier KEPT box when iou > iou_threshold (strict).
int nms_ref(const float* boxes, const float* scores, int n, float iou_threshold, int32_t* keep) {
  if (n <= 0) return 0;
  int32_t* order = new int32_t[n];
  unsigned char* dead = new unsigned char[n];
  std::memset(dead, 0, n);
  order_by_score(scores, n, order);
  int nk = 0;
  for (int i = 0; i < n; ++i) {
    const int a = order[i];
    if (dead[a]) continue;
    keep[nk++] = a;
    for (int j = i + 1; j < n; ++j) {
      const int b = order[j];
      if (!dead[b] && ops_ref_iou(boxes + 4 * (int64_t)a, boxes + 4 * (int64_t)b) > iou_threshold) dead[b] = 1;
    }
  }
  delete[] order;
  delete[] dead;
  return nk;
}

// N4-N6: Soft-NMS.  Repeatedly take the remaining box of highest current score (ties: lowest index), emit
// it with that score, and decay the score of every other remaining box b by
//   method 1 (linear):    s_b *= (iou > iou_threshold ? 1 - iou : 1)
//   method 2 (Gaussian):  s_b *= exp(-(iou*iou) / sigma)
// (fp32, each op rounded; expf of the C library); boxes whose score falls below min_score are dropped.
// keep[] / new_scores[] in selection order; returns the number emitted.
int soft_nms_ref(const float* boxes, const float* scores, int n, float iou_threshold, float sigma,
                 float min_score, int method, int32_t* keep, float* new_scores) {
  if (n <= 0) return 0;
  float* s = new float[n];
  unsigned char* gone = new unsigned char[n];
  for (int i = 0; i < n; ++i) { s[i] = scores[i]; gone[i] = !(scores[i] >= min_score); }
  int nk = 0;
  for (;;) {
    int m = -1;
    for (int i = 0; i < n; ++i)
      if (!gone[i] && (m < 0 || s[i] > s[m])) m = i;
    if (m < 0) break;
    keep[nk] = m;
    new_scores[nk] = s[m];
    ++nk;
    gone[m] = 1;
    for (int i = 0; i < n; ++i) {
      if (gone[i]) continue;
      const float iou = ops_ref_iou(boxes + 4 * (int64_t)m, boxes + 4 * (int64_t)i);
      float f = 1.0f;
      if (method == 1) { if (iou > iou_threshold) f = 1.0f - iou; }
      else { const float q = iou * iou; f = expf(-(q / sigma)); if (!(iou == iou)) f = 1.0f; }
      s[i] = s[i] * f;
      if (!(s[i] >= min_score)) gone[i] = 1;
    }
  }
  delete[] s;
  delete[] gone;
  return nk;
}


}  // extern "C" (the templates below have C++ linkage; the two entry points re-open it)

// ---- Deformable RoI pooling (D1-D5) --------------------------------------------------
// D1: the RoI on its level as in C3 with the half-pixel shift and no minimum size ("aligned"):
//       sx = x1*scale - 0.5, ex = x2*scale - 0.5, rw = ex - sx, bw = rw / PW   (rows likewise); level by C1.
// D2: grid per axis g = sampling_ratio, or (sampling_ratio == 0) ceil(bin size), 0 for a non-positive size;
//       count = max(gh*gw, 1).
// D3: bin (ph, pw) of RoI k is shifted by  ox = (gamma*rw) * offset[k,0,ph,pw],  oy = (gamma*rh) * offset[k,1,ph,pw]
//       (feature pixels; plane 0 = x, plane 1 = y; a NULL offset tensor = zeros); sample (iy, ix) sits at
//       x = [(sx + pw*bw) + ((ix + 0.5)*bw)/gw] + ox,  y likewise  -- the C3 coordinate, then ONE more addition.
//       Spec mode: all of this in fp32, each operation rounded, in this order; f64 mode: in double.
// D4: every sample is a C3 bilinear sample (outside [-1,H] x [-1,W] -> contributes 0, count unchanged; clamped
//       at 0 and at the last pixel); out = sum / count.
// D5: backward.  Features: the exact transpose.  Offsets: the derivative of D3-D4 where it exists,
//       d out / d offset_x = (gamma*rw) / count * sum_samples d val / d x,   d val / d x = (hy*(F[yl,xh]-F[yl,xl]) +
//       ly*(F[yh,xh]-F[yh,xl])) for a valid sample whose x is not clamped (0 < x < W-1), 0 otherwise (the forward is
//       constant in x there); y likewise.
template <typename R>
struct DeformTap {   // one axis of one sample
  int lo, hi;
  R wl, wh;      // weight of hi (fraction l) and of lo (1 - l)
  bool valid;    // inside [-1, n]
  bool inner;    // 0 < v < n-1 and lo < hi: the forward depends on v here
};

template <typename R>
static DeformTap<R> deform_axis(R v, int n) {
  DeformTap<R> t;
  t.valid = (v >= (R)-1) && (v <= (R)n);
  t.inner = t.valid && (v > (R)0);
  if (!(v > (R)0)) v = (R)0;
  int lo = t.valid ? (int)v : 0;
  int hi;
  if (lo >= n - 1) { lo = hi = n - 1; v = (R)lo; t.inner = false; }
  else hi = lo + 1;
  t.lo = lo; t.hi = hi;
  t.wl = v - (R)lo;
  t.wh = (R)1 - t.wl;
  return t;
}

template <typename R>
struct DeformGeom { R sx, sy, rw, rh, bw, bh; int gh, gw; int count; };

template <typename R>
static DeformGeom<R> deform_geom(const float* roi, float scale, int PH, int PW, int sampling_ratio) {
  DeformGeom<R> g;
  const R sc = (R)scale, half = (R)0.5;
  g.sx = (R)roi[1] * sc - half; g.sy = (R)roi[2] * sc - half;
  const R ex = (R)roi[3] * sc - half, ey = (R)roi[4] * sc - half;
  g.rw = ex - g.sx; g.rh = ey - g.sy;
  g.bw = g.rw / (R)PW; g.bh = g.rh / (R)PH;
  auto grid = [&](R b) -> int {
    if (sampling_ratio > 0) return sampling_ratio;
    const R c = std::ceil(b);
    return (c >= (R)1) ? (int)c : 0;
  };
  g.gh = grid(g.bh); g.gw = grid(g.bw);
  const int cnt = g.gh * g.gw;
  g.count = cnt > 1 ? cnt : 1;
  return g;
}

template <typename R>
static R deform_coord(R start, R bin, int p, int i, int grid, R shift) {
  const R a = start + (R)p * bin;
  const R d = (((R)i + (R)0.5) * bin) / (R)grid;
  return (a + d) + shift;
}

template <typename R>
static int deform_forward(const ops_ref_level* feats, int L, const float* rois, int K, const float* offset, float gamma,
                          int PH, int PW, int sampling_ratio, float finest_scale, double* out) {
  const int C = feats[0].c;
  for (int k = 0; k < K; ++k) {
    const float* roi = rois + 5 * (int64_t)k;
    const int l = level_of(roi, L, finest_scale);
    const ops_ref_level& lv = feats[l];
    const int b = batch_index_of(roi[0], lv.n);
    const DeformGeom<R> g = deform_geom<R>(roi, lv.spatial_scale, PH, PW, sampling_ratio);
    for (int c = 0; c < C; ++c)
      for (int ph = 0; ph < PH; ++ph)
        for (int pw = 0; pw < PW; ++pw) {
          double acc = 0.0;
          if (b >= 0) {
            const R dx = offset ? (R)offset[(((int64_t)k * 2 + 0) * PH + ph) * PW + pw] : (R)0;
            const R dy = offset ? (R)offset[(((int64_t)k * 2 + 1) * PH + ph) * PW + pw] : (R)0;
            const R ox = ((R)gamma * g.rw) * dx, oy = ((R)gamma * g.rh) * dy;
            const double* F = lv.data + ((int64_t)b * C + c) * lv.h * lv.w;
            for (int iy = 0; iy < g.gh; ++iy) {
              const DeformTap<R> ty = deform_axis<R>(deform_coord<R>(g.sy, g.bh, ph, iy, g.gh, oy), lv.h);
              if (!ty.valid) continue;
              for (int ix = 0; ix < g.gw; ++ix) {
                const DeformTap<R> tx = deform_axis<R>(deform_coord<R>(g.sx, g.bw, pw, ix, g.gw, ox), lv.w);
                if (!tx.valid) continue;
                const R w1 = ty.wh * tx.wh, w2 = ty.wh * tx.wl, w3 = ty.wl * tx.wh, w4 = ty.wl * tx.wl;
                acc += (double)w1 * F[(int64_t)ty.lo * lv.w + tx.lo] + (double)w2 * F[(int64_t)ty.lo * lv.w + tx.hi] +
                       (double)w3 * F[(int64_t)ty.hi * lv.w + tx.lo] + (double)w4 * F[(int64_t)ty.hi * lv.w + tx.hi];
              }
            }
          }
          out[(((int64_t)k * C + c) * PH + ph) * PW + pw] = acc / (double)g.count;
        }
  }
  return 0;
}

extern "C" int deform_roi_pool_fpn_forward_ref(const ops_ref_level* feats, int L, const float* rois, int K, const float* offset,
                                    float gamma, int PH, int PW, int sampling_ratio, float finest_scale, int f64_mode,
                                    double* out) {
  return f64_mode ? deform_forward<double>(feats, L, rois, K, offset, gamma, PH, PW, sampling_ratio, finest_scale, out)
                  : deform_forward<float>(feats, L, rois, K, offset, gamma, PH, PW, sampling_ratio, finest_scale, out);
}

template <typename R>
static int deform_backward(const ops_ref_level* feats, const ops_ref_level* grads, int L, const double* grad_out,
                           const float* rois, int K, const float* offset, float gamma, int PH, int PW, int sampling_ratio,
                           float finest_scale, double* grad_offset) {
  const int C = feats[0].c;
  if (grad_offset) memset(grad_offset, 0, sizeof(double) * (size_t)K * 2 * PH * PW);
  for (int k = 0; k < K; ++k) {
    const float* roi = rois + 5 * (int64_t)k;
    const int l = level_of(roi, L, finest_scale);
    const ops_ref_level& lv = feats[l];
    const int b = batch_index_of(roi[0], lv.n);
    if (b < 0) continue;
    const DeformGeom<R> g = deform_geom<R>(roi, lv.spatial_scale, PH, PW, sampling_ratio);
    for (int c = 0; c < C; ++c)
      for (int ph = 0; ph < PH; ++ph)
        for (int pw = 0; pw < PW; ++pw) {
          const double go = grad_out[(((int64_t)k * C + c) * PH + ph) * PW + pw] / (double)g.count;
          const R dx = offset ? (R)offset[(((int64_t)k * 2 + 0) * PH + ph) * PW + pw] : (R)0;
          const R dy = offset ? (R)offset[(((int64_t)k * 2 + 1) * PH + ph) * PW + pw] : (R)0;
          const R ox = ((R)gamma * g.rw) * dx, oy = ((R)gamma * g.rh) * dy;
          const double* F = lv.data + ((int64_t)b * C + c) * lv.h * lv.w;
          double* G = grads ? grads[l].data + ((int64_t)b * C + c) * lv.h * lv.w : nullptr;
          double gx = 0.0, gy = 0.0;
          for (int iy = 0; iy < g.gh; ++iy) {
            const DeformTap<R> ty = deform_axis<R>(deform_coord<R>(g.sy, g.bh, ph, iy, g.gh, oy), lv.h);
            if (!ty.valid) continue;
            for (int ix = 0; ix < g.gw; ++ix) {
              const DeformTap<R> tx = deform_axis<R>(deform_coord<R>(g.sx, g.bw, pw, ix, g.gw, ox), lv.w);
              if (!tx.valid) continue;
              const int64_t i1 = (int64_t)ty.lo * lv.w + tx.lo, i2 = (int64_t)ty.lo * lv.w + tx.hi;
              const int64_t i3 = (int64_t)ty.hi * lv.w + tx.lo, i4 = (int64_t)ty.hi * lv.w + tx.hi;
              if (G) {
                G[i1] += (double)(ty.wh * tx.wh) * go; G[i2] += (double)(ty.wh * tx.wl) * go;
                G[i3] += (double)(ty.wl * tx.wh) * go; G[i4] += (double)(ty.wl * tx.wl) * go;
              }
              if (tx.inner) gx += (double)ty.wh * (F[i2] - F[i1]) + (double)ty.wl * (F[i4] - F[i3]);
              if (ty.inner) gy += (double)tx.wh * (F[i3] - F[i1]) + (double)tx.wl * (F[i4] - F[i2]);
            }
          }
          if (grad_offset) {
            grad_offset[(((int64_t)k * 2 + 0) * PH + ph) * PW + pw] += go * gx * (double)((R)gamma * g.rw);
            grad_offset[(((int64_t)k * 2 + 1) * PH + ph) * PW + pw] += go * gy * (double)((R)gamma * g.rh);
          }
        }
  }
  return 0;
}

extern "C" {
// grads (may be NULL: offsets only) must hold their starting values; grad_offset [K,2,PH,PW] (may be NULL) is overwritten.
int deform_roi_pool_fpn_backward_ref(const ops_ref_level* feats, const ops_ref_level* grads, int L, const double* grad_out,
                                     const float* rois, int K, const float* offset, float gamma, int PH, int PW,
                                     int sampling_ratio, float finest_scale, int f64_mode, double* grad_offset) {
  return f64_mode ? deform_backward<double>(feats, grads, L, grad_out, rois, K, offset, gamma, PH, PW, sampling_ratio,
                                            finest_scale, grad_offset)
                  : deform_backward<float>(feats, grads, L, grad_out, rois, K, offset, gamma, PH, PW, sampling_ratio,
                                           finest_scale, grad_offset);
}

}  // extern "C"
