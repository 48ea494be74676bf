// ops_ref.cpp -- CPU ORACLE for the SURVEY 8(f) "next" operations around the RoIAlign hot path:
//   * multi-level (FPN) RoIPool-max forward / backward  ("RoIPooling-like operators", section
//     3.1 RoIExtractor; the max variant is the RoI pooling layer of Fast R-CNN);
//   * greedy NMS and Soft-NMS on boxes ("Soft NMS [1]: an alternative to NMS"; "All basic
//     bbox and mask operations run on GPUs").
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
// to a score sort when no boxes overlap.  Nothing here is "parity unpinned".
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

}  // extern "C"
