// raf_api.cu -- the C ABI of libraf.so (include/raf.h): argument validation, layout
// classification and kernel dispatch.  No allocation, no synchronisation, no device->host copy
// (except the documented *_host entry points, which copy between caller-owned buffers).
#include <atomic>
#include <cstdlib>
#include <cstring>

#include "raf_device.cuh"
#include "raf_host.h"
#include "raf_pull_prep.cuh"

namespace raf {

static std::atomic<uint64_t> g_launches{0};
void count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }
constexpr int kBoffInts = 2048;  // boff[L*N + 1]; larger L*N falls back to the atomic backward
static size_t esize(raf_dtype d) { return d == RAF_F32 ? 4 : 2; }

static int check_levels(const raf_level* lv, int L) {
  if (!lv) return RAF_ERR_NULL;
  if (L < 1 || L > kMaxLevels) return RAF_ERR_SHAPE;
  for (int l = 0; l < L; ++l) {
    if (!lv[l].data) return RAF_ERR_NULL;
    if (lv[l].n < 1 || lv[l].c < 1 || lv[l].h < 1 || lv[l].w < 1) return RAF_ERR_SHAPE;
    if (lv[l].n != lv[0].n || lv[l].c != lv[0].c) return RAF_ERR_SHAPE;
    if (lv[l].sn <= 0 || lv[l].sc <= 0 || lv[l].sh <= 0 || lv[l].sw <= 0) return RAF_ERR_STRIDE;
    if (!(lv[l].spatial_scale > 0.0f)) return RAF_ERR_SHAPE;
  }
  return RAF_OK;
}

static int check_common(const float* rois, int K, int out_h, int out_w, int sampling_ratio) {
  if (K < 0 || out_h < 1 || out_h > 32 || out_w < 1 || out_w > 32) return RAF_ERR_SHAPE;
  if (sampling_ratio < 0 || sampling_ratio > 16) return RAF_ERR_SHAPE;
  if (K > 0 && !rois) return RAF_ERR_NULL;
  return RAF_OK;
}

static void fill_param(const raf_level* lv, int L, LevelsParam* p) {
  std::memset(p, 0, sizeof(*p));
  p->n = lv[0].n; p->c = lv[0].c; p->L = L;
  for (int l = 0; l < L; ++l) {
    p->data[l] = lv[l].data;
    p->sn[l] = lv[l].sn; p->sc[l] = lv[l].sc; p->sh[l] = lv[l].sh; p->sw[l] = lv[l].sw;
    p->h[l] = lv[l].h; p->w[l] = lv[l].w; p->scale[l] = lv[l].spatial_scale;
  }
}

// Channels-last fast-path eligibility: unit channel stride, `vec`-element (16-byte for the
// features, see callers) aligned pixel vectors, in-image offsets that fit int32.
static bool levels_vectorizable(const raf_level* lv, int L, int vec, size_t elem) {
  for (int l = 0; l < L; ++l) {
    if (lv[l].sc != 1 || lv[l].c % vec) return false;
    if (lv[l].sn % vec || lv[l].sh % vec || lv[l].sw % vec) return false;
    if (((uintptr_t)lv[l].data) % (vec * elem)) return false;
    const int64_t span = (int64_t)(lv[l].h - 1) * lv[l].sh + (int64_t)(lv[l].w - 1) * lv[l].sw + lv[l].c;
    if (span >= ((int64_t)1 << 31)) return false;
  }
  return true;
}

// (the stride of an extent-1 dimension is never used: frameworks report arbitrary values there)
static bool tensor_vectorizable(const void* p, const int64_t* s, int vec, size_t elem, int K, int PH, int PW) {
  return s[1] == 1 && (K <= 1 || s[0] % vec == 0) && (PH <= 1 || s[2] % vec == 0) && (PW <= 1 || s[3] % vec == 0) &&
         ((uintptr_t)p) % (vec * elem) == 0;
}

// A level is one dense block when its strides are a permutation of a packed layout.
static bool level_dense(const raf_level& v) {
  int64_t ext[4] = {v.n, v.c, v.h, v.w}, st[4] = {v.sn, v.sc, v.sh, v.sw};
  for (int i = 0; i < 4; ++i)
    for (int j = i + 1; j < 4; ++j)
      if (st[j] < st[i] || (st[j] == st[i] && ext[j] < ext[i])) {
        std::swap(st[i], st[j]); std::swap(ext[i], ext[j]);
      }
  int64_t run = 1;
  for (int i = 0; i < 4; ++i) {
    if (ext[i] == 1) continue;
    if (st[i] != run) return false;
    run *= ext[i];
  }
  return true;
}

// Dense NCHW (strides of extent-1 dimensions are not looked at).
static bool level_nchw(const raf_level& v) {
  return (v.w <= 1 || v.sw == 1) && (v.h <= 1 || v.sh == v.w) && (v.c <= 1 || v.sc == (int64_t)v.h * v.w) &&
         (v.n <= 1 || v.sn == (int64_t)v.c * v.h * v.w);
}
static bool tensor_nchw(int K, int C, int PH, int PW, const int64_t* s) {
  return (PW <= 1 || s[3] == 1) && (PH <= 1 || s[2] == PW) && (C <= 1 || s[1] == (int64_t)PH * PW) &&
         (K <= 1 || s[0] == (int64_t)C * PH * PW);
}

}  // namespace raf

using namespace raf;

extern "C" {

// Workspace carve-up (pull backward): [hdr 256 B][bperm K int32][boff kBoffInts int32][bwin K int4][bgeo K float4][taps].
struct WsLayout {
  size_t hdr, bperm, boff, bwin, bgeo, taps, total;
};
static WsLayout ws_layout(int K, int out_h, int out_w, int sampling_ratio) {
  const size_t k = K > 0 ? (size_t)K : 0;
  const size_t g = sampling_ratio > 0 ? (size_t)sampling_ratio : 0;
  WsLayout w;
  w.hdr = 0;
  w.bperm = 256;
  w.boff = w.bperm + align256(4 * k);
  w.bwin = w.boff + align256(4 * (size_t)kBoffInts);
  w.bgeo = w.bwin + align256(16 * k);
  w.taps = w.bgeo + align256(16 * k);
  w.total = w.taps + align256(k * (size_t)(out_h + out_w) * 2 * g * sizeof(PullTap)) + 256;
  return w;
}

// The pull backward's prep tables can be built for these arguments (layout-independent part of the
// pull eligibility; the forward uses the same test before it writes them into the workspace).
static bool prep_possible(const raf_level* lv, int L, int sampling_ratio) {
  if (sampling_ratio < 0 || (int64_t)L * lv[0].n + 1 > kBoffInts) return false;   // (0 = adaptive: buckets only)
  if (bucket_smem_bytes(L, lv[0].n) > 200 * 1024) return false;
  if ((size_t)(kMaxLevels + 1) * ((size_t)L * lv[0].n + 1) * sizeof(int) > 200 * 1024) return false;
  for (int l = 0; l < L; ++l)   // tap tables keep pixel indices in 24 bits
    if (lv[l].h >= 0xffffff || lv[l].w >= 0xffffff) return false;
  return true;
}

// 64-bit FNV-1a over the arguments the prep tables depend on.
static void fnv(uint64_t& h, const void* p, size_t n) {
  const unsigned char* b = (const unsigned char*)p;
  for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ull; }
}
static PrepFingerprint prep_fingerprint(const raf_level* lv, int L, const float* rois, int K, int out_h, int out_w,
                                        int sampling_ratio, int aligned, float finest_scale) {
  uint64_t h = 1469598103934665603ull;
  for (int l = 0; l < L; ++l) {
    fnv(h, &lv[l].h, sizeof(int32_t)); fnv(h, &lv[l].w, sizeof(int32_t));
    fnv(h, &lv[l].spatial_scale, sizeof(float));
  }
  PrepFingerprint f;
  f.v[0] = 0x52414632u;   // "RAF2": table format
  f.v[1] = (uint32_t)K;
  f.v[2] = (uint32_t)out_h | ((uint32_t)out_w << 8) | ((uint32_t)sampling_ratio << 16) | ((uint32_t)(aligned ? 1 : 0) << 24) |
           ((uint32_t)L << 25);
  std::memcpy(&f.v[3], &finest_scale, 4);
  f.v[4] = (uint32_t)lv[0].n;
  f.v[5] = (uint32_t)(h ^ (h >> 32));
  const uint64_t rp = (uint64_t)(uintptr_t)rois;
  f.v[6] = (uint32_t)rp;
  f.v[7] = (uint32_t)(rp >> 32);
  return f;
}

static PullPrepOut prep_out(void* ws, int K, int out_h, int out_w, int sampling_ratio, const PrepFingerprint& fp) {
  const WsLayout w = ws_layout(K, out_h, out_w, sampling_ratio);
  char* base = reinterpret_cast<char*>(ws);
  PullPrepOut po{};
  po.hdr = reinterpret_cast<uint32_t*>(base + w.hdr);
  po.bperm = reinterpret_cast<int32_t*>(base + w.bperm);
  po.boff = reinterpret_cast<int32_t*>(base + w.boff);
  po.bwin = reinterpret_cast<int4*>(base + w.bwin);
  po.bgeo = reinterpret_cast<float4*>(base + w.bgeo);
  po.taps = reinterpret_cast<PullTap*>(base + w.taps);
  po.fp = fp;
  return po;
}

size_t roi_align_fpn_workspace_bytes(int K, int L, int out_h, int out_w, int sampling_ratio,
                                     int flags) {
  (void)L; (void)flags;
  if (out_h < 1) out_h = 1;
  if (out_w < 1) out_w = 1;
  return ws_layout(K, out_h, out_w, sampling_ratio).total;
}

int roi_fpn_assign_levels(const float* rois, int K, int L, float finest_scale, int32_t* levels,
                          int32_t* counts, int32_t* perm, void* ws, size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  if (K < 0 || L < 1 || L > kMaxLevels) return RAF_ERR_SHAPE;
  if (K > 0 && !rois) return RAF_ERR_NULL;
  if (!(finest_scale > 0.0f)) return RAF_ERR_SHAPE;
  if (K == 0 && !counts) return RAF_OK;
  return launch_assign_levels(rois, K, L, finest_scale, levels, counts, perm, (cudaStream_t)stream);
}

size_t roi_align_fpn_repack_bytes(const raf_level* levels, int L, raf_dtype dtype, int K, int out_h, int out_w) {
  (void)dtype;   // sized for fp32 copies: the backward's gradient pyramid is fp32 whatever the feature dtype
  if (!levels || L < 1 || L > kMaxLevels || K < 0 || out_h < 1 || out_w < 1) return 0;
  size_t total = 256;
  for (int l = 0; l < L; ++l) total += align256((size_t)levels[l].n * levels[l].c * levels[l].h * levels[l].w * 4);
  total += align256((size_t)K * levels[0].c * out_h * out_w * 4);
  return total;
}

// RAF_REPACK: channels-last descriptors of the scratch copies of dense NCHW levels, carved from `scratch`.
static char* repack_levels(const raf_level* src, int L, size_t esz, char* scratch, raf_level* dst) {
  for (int l = 0; l < L; ++l) {
    dst[l] = src[l];
    dst[l].data = scratch;
    dst[l].sc = 1;
    dst[l].sw = src[l].c;
    dst[l].sh = (int64_t)src[l].w * src[l].c;
    dst[l].sn = (int64_t)src[l].h * src[l].w * src[l].c;
    scratch += align256((size_t)src[l].n * src[l].c * src[l].h * src[l].w * esz);
  }
  return scratch;
}

int roi_align_fpn_forward(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                          int out_h, int out_w, int sampling_ratio, int aligned, float finest_scale,
                          void* out, const int64_t* out_strides, void* ws, size_t ws_bytes,
                          void* stream) {
  return roi_align_fpn_forward_ex(feats, L, dtype, rois, K, out_h, out_w, sampling_ratio, aligned, finest_scale,
                                  out, out_strides, 0, ws, ws_bytes, stream);
}

int roi_align_fpn_forward_ex(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                             int out_h, int out_w, int sampling_ratio, int aligned, float finest_scale,
                             void* out, const int64_t* out_strides, int flags, void* ws, size_t ws_bytes,
                             void* stream) {
  int rc = check_levels(feats, L);
  if (rc) return rc;
  rc = check_common(rois, K, out_h, out_w, sampling_ratio);
  if (rc) return rc;
  if (dtype != RAF_F32 && dtype != RAF_F16 && dtype != RAF_BF16) return RAF_ERR_DTYPE;
  if (!(finest_scale > 0.0f)) return RAF_ERR_SHAPE;
  if (!out_strides) return RAF_ERR_NULL;
  if (K == 0) return RAF_OK;  // nothing to do; strides of an empty tensor are not meaningful
  for (int i = 0; i < 4; ++i) if (out_strides[i] <= 0) return RAF_ERR_STRIDE;
  if (!out) return RAF_ERR_NULL;
  if (flags & ~(RAF_NO_PREP | RAF_REPACK)) return RAF_ERR_UNSUPPORTED;
  if (flags & RAF_REPACK) {
    const int vec0 = (int)(16 / esize(dtype));
    const bool cl0 = levels_vectorizable(feats, L, vec0, esize(dtype)) &&
                     tensor_vectorizable(out, out_strides, vec0, esize(dtype), K, out_h, out_w);
    if (!cl0) {   // repack NCHW -> channels-last inside the workspace, run the fast path, repack the result back
      for (int l = 0; l < L; ++l) if (!level_nchw(feats[l])) return RAF_ERR_STRIDE;
      if (!tensor_nchw(K, feats[0].c, out_h, out_w, out_strides) || feats[0].c % vec0) return RAF_ERR_STRIDE;
      const size_t base = roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, 0);
      if (!ws) return RAF_ERR_NULL;
      if ((uintptr_t)ws % 256) return RAF_ERR_WORKSPACE;
      if (ws_bytes < base + roi_align_fpn_repack_bytes(feats, L, dtype, K, out_h, out_w)) return RAF_ERR_WORKSPACE;
      cudaStream_t st = (cudaStream_t)stream;
      raf_level cl_lv[kMaxLevels];
      char* cur = repack_levels(feats, L, esize(dtype), (char*)ws + base, cl_lv);
      void* cl_out = cur;
      for (int l = 0; l < L; ++l) {
        rc = launch_transpose(feats[l].data, cl_lv[l].data, feats[l].n, feats[l].c, feats[l].h * feats[l].w, esize(dtype), st);
        if (rc) return rc;
      }
      const int C = feats[0].c;
      const int64_t cl_strides[4] = {(int64_t)out_h * out_w * C, 1, (int64_t)out_w * C, C};
      rc = roi_align_fpn_forward_ex(cl_lv, L, dtype, rois, K, out_h, out_w, sampling_ratio, aligned, finest_scale, cl_out,
                                    cl_strides, flags & ~RAF_REPACK, ws, base, stream);
      if (rc) return rc;
      return launch_transpose(cl_out, out, K, out_h * out_w, C, esize(dtype), st);
    }
  }
  const bool want_prep = !(flags & RAF_NO_PREP);
  if (want_prep) {
    if (!ws) return RAF_ERR_NULL;
    if ((uintptr_t)ws % 256) return RAF_ERR_WORKSPACE;
    if (ws_bytes < roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, 0)) return RAF_ERR_WORKSPACE;
  }

  LevelsParam p;
  fill_param(feats, L, &p);
  const RoiArgs a{rois, K, out_h, out_w, sampling_ratio, aligned ? 1 : 0, finest_scale};
  const int vec = (int)(16 / esize(dtype));
  const bool cl = levels_vectorizable(feats, L, vec, esize(dtype)) &&
                  tensor_vectorizable(out, out_strides, vec, esize(dtype), K, out_h, out_w);
  // the workspace receives the pull backward's prep tables (consumed by RAF_REUSE_PREP)
  PullPrepOut po{};
  const bool with_prep = want_prep && prep_possible(feats, L, sampling_ratio);
  if (with_prep)
    po = prep_out(ws, K, out_h, out_w, sampling_ratio, prep_fingerprint(feats, L, rois, K, out_h, out_w, sampling_ratio, aligned, finest_scale));
  return launch_forward(p, dtype, a, out, out_strides, cl, with_prep ? &po : nullptr, (cudaStream_t)stream);
}

int roi_align_fpn_backward(const raf_level* grad_feats, int L, raf_dtype gout_dtype,
                           const void* grad_out, const int64_t* gout_strides, const float* rois,
                           int K, int out_h, int out_w, int sampling_ratio, int aligned,
                           float finest_scale, int flags, void* ws, size_t ws_bytes, void* stream) {
  return roi_align_fpn_backward_ex(grad_feats, L, gout_dtype, RAF_F32, grad_out, gout_strides, rois, K, out_h, out_w,
                                   sampling_ratio, aligned, finest_scale, flags, ws, ws_bytes, stream);
}

int roi_align_fpn_backward_ex(const raf_level* grad_feats, int L, raf_dtype gout_dtype, raf_dtype grad_dtype,
                              const void* grad_out, const int64_t* gout_strides, const float* rois,
                              int K, int out_h, int out_w, int sampling_ratio, int aligned,
                              float finest_scale, int flags, void* ws, size_t ws_bytes, void* stream) {
  int rc = check_levels(grad_feats, L);
  if (rc) return rc;
  rc = check_common(rois, K, out_h, out_w, sampling_ratio);
  if (rc) return rc;
  if (gout_dtype != RAF_F32 && gout_dtype != RAF_F16 && gout_dtype != RAF_BF16) return RAF_ERR_DTYPE;
  if (grad_dtype != RAF_F32 && grad_dtype != RAF_F16 && grad_dtype != RAF_BF16) return RAF_ERR_DTYPE;
  // 16-bit gradient pyramid: only as the type of grad_out, only through the pull kernels (fp32 sums, one rounding)
  const bool g16 = grad_dtype != RAF_F32;
  if (g16 && (grad_dtype != gout_dtype || (flags & (RAF_ATOMIC | RAF_REPACK)))) return RAF_ERR_UNSUPPORTED;
  if (!(finest_scale > 0.0f)) return RAF_ERR_SHAPE;
  if (flags & ~(RAF_ACCUMULATE | RAF_DETERMINISTIC | RAF_ATOMIC | RAF_REUSE_PREP | RAF_PULL_STRIP | RAF_PULL_TILE | RAF_REPACK)) return RAF_ERR_UNSUPPORTED;
  if ((flags & RAF_DETERMINISTIC) && (flags & RAF_ATOMIC)) return RAF_ERR_UNSUPPORTED;
  if ((flags & RAF_PULL_STRIP) && (flags & (RAF_PULL_TILE | RAF_ATOMIC))) return RAF_ERR_UNSUPPORTED;
  if ((flags & RAF_PULL_TILE) && (flags & RAF_ATOMIC)) return RAF_ERR_UNSUPPORTED;
  if (!gout_strides) return RAF_ERR_NULL;
  for (int i = 0; i < 4; ++i) if (K > 0 && gout_strides[i] <= 0) return RAF_ERR_STRIDE;
  if (K > 0 && !grad_out) return RAF_ERR_NULL;
  if (!ws) return RAF_ERR_NULL;
  if ((uintptr_t)ws % 256) return RAF_ERR_WORKSPACE;
  if (ws_bytes < roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, flags))
    return RAF_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  if ((flags & RAF_REPACK) && K > 0) {
    const bool cl0 = levels_vectorizable(grad_feats, L, 4, esize(grad_dtype)) &&
                     tensor_vectorizable(grad_out, gout_strides, 4, esize(gout_dtype), K, out_h, out_w);
    if (!cl0) {   // grad_out -> channels-last copy, fast backward into a channels-last gradient copy, repack back
      for (int l = 0; l < L; ++l) if (!level_nchw(grad_feats[l])) return RAF_ERR_STRIDE;
      const int C = grad_feats[0].c;
      if (!tensor_nchw(K, C, out_h, out_w, gout_strides) || C % 4 || (esize(gout_dtype) == 2 && C % 8)) return RAF_ERR_STRIDE;
      const size_t base = roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, flags);
      if (ws_bytes < base + roi_align_fpn_repack_bytes(grad_feats, L, gout_dtype, K, out_h, out_w)) return RAF_ERR_WORKSPACE;
      raf_level cl_lv[kMaxLevels];
      char* cur = repack_levels(grad_feats, L, 4, (char*)ws + base, cl_lv);
      void* cl_gout = cur;
      rc = launch_transpose(grad_out, cl_gout, K, C, out_h * out_w, esize(gout_dtype), st);
      if (rc) return rc;
      if (flags & RAF_ACCUMULATE)
        for (int l = 0; l < L; ++l) {
          rc = launch_transpose(grad_feats[l].data, cl_lv[l].data, grad_feats[l].n, C, grad_feats[l].h * grad_feats[l].w, 4, st);
          if (rc) return rc;
        }
      const int64_t cl_strides[4] = {(int64_t)out_h * out_w * C, 1, (int64_t)out_w * C, C};
      rc = roi_align_fpn_backward(cl_lv, L, gout_dtype, cl_gout, cl_strides, rois, K, out_h, out_w, sampling_ratio, aligned,
                                  finest_scale, flags & ~RAF_REPACK, ws, base, stream);
      if (rc) return rc;
      for (int l = 0; l < L; ++l) {
        rc = launch_transpose(cl_lv[l].data, grad_feats[l].data, grad_feats[l].n, grad_feats[l].h * grad_feats[l].w, C, 4, st);
        if (rc) return rc;
      }
      return RAF_OK;
    }
  }
  LevelsParam p;
  fill_param(grad_feats, L, &p);
  const RoiArgs a{rois, K, out_h, out_w, sampling_ratio, aligned ? 1 : 0, finest_scale};
  const bool cl = levels_vectorizable(grad_feats, L, 4, esize(grad_dtype)) &&
                  (K == 0 || tensor_vectorizable(grad_out, gout_strides, 4, esize(gout_dtype), K, out_h, out_w));

  // ---- pull variant (K3d): deterministic, no zero-fill, every element written once -------------
  const bool pull_ok = cl && prep_possible(grad_feats, L, sampling_ratio);
  if (pull_ok && !(flags & RAF_ATOMIC)) {
    const PullPrepOut po = prep_out(ws, K, out_h, out_w, sampling_ratio, prep_fingerprint(grad_feats, L, rois, K, out_h, out_w, sampling_ratio, aligned,
                                                           finest_scale));
    // Two pull kernels (both deterministic, same prep tables): the strip kernel (raf_backward_strip.cu) wins
    // when there are many warp tiles to overlap and a grad_out vector feeds several pixels (bins at least
    // about a pixel wide: the usual 7 x 7 box head); the tile-owned kernel (raf_backward_pull.cu) wins on
    // small batches and on outputs finer than the pixel grid.  The strip kernel also takes what the
    // first one cannot (more than 128 taps per axis).
    const bool strip_ok = strip_eligible(p, gout_dtype, a, gout_strides) == RAF_OK;
    const bool pull_first_ok = pull_eligible(p, gout_dtype, a, grad_out, gout_strides) == RAF_OK;
    int64_t pixels = 0;
    for (int l = 0; l < L; ++l) pixels += (int64_t)grad_feats[l].h * grad_feats[l].w;
    pixels *= grad_feats[0].n;
    bool use_strip = strip_ok && (!pull_first_ok || (out_h <= 8 && out_w <= 8 && pixels >= 512 * 1024));
    if (flags & RAF_PULL_STRIP) { if (!strip_ok) return RAF_ERR_UNSUPPORTED; use_strip = true; }
    if (flags & RAF_PULL_TILE) { if (!pull_first_ok) return RAF_ERR_UNSUPPORTED; use_strip = false; }
    if (use_strip) {
      if (!(flags & RAF_REUSE_PREP) || K == 0) {
        rc = launch_pull_prep(p, a, po, st);
        if (rc) return rc;
      }
      return launch_backward_strip(p, gout_dtype, grad_dtype, a, grad_out, gout_strides, po, (flags & RAF_ACCUMULATE) ? 1 : 0, st);
    }
    rc = pull_eligible(p, gout_dtype, a, grad_out, gout_strides);
    if (rc == RAF_OK) {
      if (!(flags & RAF_REUSE_PREP) || K == 0) {   // else: written by roi_align_fpn_forward on the same arguments
                                                   // (the forward writes nothing when K == 0); the kernel checks
        rc = launch_pull_prep(p, a, po, st);
        if (rc) return rc;
      }
      return launch_backward_pull(p, gout_dtype, grad_dtype, a, grad_out, gout_strides, po, (flags & RAF_ACCUMULATE) ? 1 : 0, st);
    }
    if (rc != RAF_ERR_UNSUPPORTED) return rc;
  }
  if ((flags & (RAF_DETERMINISTIC | RAF_PULL_STRIP | RAF_PULL_TILE)) || g16) return RAF_ERR_UNSUPPORTED;

  // ---- atomic variant (K3) -----------------------------------------------------------------------
  if (!(flags & RAF_ACCUMULATE)) {
    for (int l = 0; l < L; ++l) {
      const raf_level& v = grad_feats[l];
      if (level_dense(v)) {
        if (cudaMemsetAsync(v.data, 0, sizeof(float) * (size_t)v.n * v.c * v.h * v.w, st) != cudaSuccess)
          return RAF_ERR_CUDA;
        count_launch();
      } else {
        rc = launch_zero_level((float*)v.data, v.n, v.c, v.h, v.w, v.sn, v.sc, v.sh, v.sw, st);
        if (rc) return rc;
      }
    }
  }
  if (K == 0) return RAF_OK;
  return launch_backward_atomic(p, gout_dtype, a, grad_out, gout_strides, cl, st);
}

// ---- RoIPool-max -------------------------------------------------------------------------------------
static bool unit_channel_stride(const raf_level* lv, int L) {
  for (int l = 0; l < L; ++l)
    if (lv[l].sc != 1) return false;
  return true;
}

static int zero_fill(const raf_level* grad_feats, int L, cudaStream_t st) {
  for (int l = 0; l < L; ++l) {
    const raf_level& v = grad_feats[l];
    if (level_dense(v)) {
      if (cudaMemsetAsync(v.data, 0, sizeof(float) * (size_t)v.n * v.c * v.h * v.w, st) != cudaSuccess) return RAF_ERR_CUDA;
      count_launch();
    } else {
      const int rc = launch_zero_level((float*)v.data, v.n, v.c, v.h, v.w, v.sn, v.sc, v.sh, v.sw, st);
      if (rc) return rc;
    }
  }
  return RAF_OK;
}

int roi_pool_fpn_forward(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                         int out_h, int out_w, float finest_scale, void* out, int32_t* argmax,
                         const int64_t* out_strides, void* stream) {
  int rc = check_levels(feats, L);
  if (rc) return rc;
  rc = check_common(rois, K, out_h, out_w, 1);
  if (rc) return rc;
  if (dtype != RAF_F32 && dtype != RAF_F16 && dtype != RAF_BF16) return RAF_ERR_DTYPE;
  if (!(finest_scale > 0.0f)) return RAF_ERR_SHAPE;
  if (!out_strides) return RAF_ERR_NULL;
  if (K == 0) return RAF_OK;
  for (int i = 0; i < 4; ++i) if (out_strides[i] <= 0) return RAF_ERR_STRIDE;
  if (!out) return RAF_ERR_NULL;
  for (int l = 0; l < L; ++l)
    if ((int64_t)feats[l].h * feats[l].w >= ((int64_t)1 << 31)) return RAF_ERR_UNSUPPORTED;   // argmax is int32
  LevelsParam p;
  fill_param(feats, L, &p);
  return launch_pool_forward(p, dtype, rois, K, out_h, out_w, finest_scale, out, argmax, out_strides,
                             unit_channel_stride(feats, L), (cudaStream_t)stream);
}

int roi_pool_fpn_backward(const raf_level* grad_feats, int L, raf_dtype gout_dtype, const void* grad_out,
                          const int32_t* argmax, const int64_t* gout_strides, const float* rois, int K,
                          int out_h, int out_w, float finest_scale, int flags, void* stream) {
  int rc = check_levels(grad_feats, L);
  if (rc) return rc;
  rc = check_common(rois, K, out_h, out_w, 1);
  if (rc) return rc;
  if (gout_dtype != RAF_F32 && gout_dtype != RAF_F16 && gout_dtype != RAF_BF16) return RAF_ERR_DTYPE;
  if (!(finest_scale > 0.0f)) return RAF_ERR_SHAPE;
  if (flags & ~RAF_ACCUMULATE) return RAF_ERR_UNSUPPORTED;
  if (!gout_strides) return RAF_ERR_NULL;
  for (int i = 0; i < 4; ++i) if (K > 0 && gout_strides[i] <= 0) return RAF_ERR_STRIDE;
  if (K > 0 && (!grad_out || !argmax)) return RAF_ERR_NULL;
  cudaStream_t st = (cudaStream_t)stream;
  if (!(flags & RAF_ACCUMULATE)) {
    rc = zero_fill(grad_feats, L, st);
    if (rc) return rc;
  }
  if (K == 0) return RAF_OK;
  LevelsParam p;
  fill_param(grad_feats, L, &p);
  return launch_pool_backward(p, gout_dtype, rois, K, out_h, out_w, finest_scale, grad_out, argmax, gout_strides,
                              unit_channel_stride(grad_feats, L), st);
}

// ---- RoIAlign gather fused into the first FC ------------------------------------------------------------
int roi_align_fc_fpn_forward(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                             int out_h, int out_w, int sampling_ratio, int aligned, float finest_scale,
                             const void* weight, const float* bias, int n_out, float* out, void* stream) {
  int rc = check_levels(feats, L);
  if (rc) return rc;
  rc = check_common(rois, K, out_h, out_w, sampling_ratio);
  if (rc) return rc;
  if (dtype != RAF_F32 && dtype != RAF_F16 && dtype != RAF_BF16) return RAF_ERR_DTYPE;
  if (!(finest_scale > 0.0f) || n_out < 1) return RAF_ERR_SHAPE;
  if (K == 0) return RAF_OK;
  if (!weight || !out) return RAF_ERR_NULL;
  if (dtype == RAF_F32 || sampling_ratio < 1 || sampling_ratio > 2 || n_out % 512 || feats[0].c % 64) return RAF_ERR_UNSUPPORTED;
  if (!levels_vectorizable(feats, L, 8, 2) || ((uintptr_t)weight) % 16 || ((uintptr_t)out) % 16) return RAF_ERR_UNSUPPORTED;
  if ((int64_t)K * n_out >= ((int64_t)1 << 40)) return RAF_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  if (cudaMemsetAsync(out, 0, sizeof(float) * (size_t)K * n_out, st) != cudaSuccess) return RAF_ERR_CUDA;
  count_launch();
  LevelsParam p;
  fill_param(feats, L, &p);
  const RoiArgs a{rois, K, out_h, out_w, sampling_ratio, aligned ? 1 : 0, finest_scale};
  return launch_fc_fused(p, dtype, a, weight, bias, n_out, out, st);
}

// ---- deformable RoI pooling ---------------------------------------------------------------------------
int roi_deform_pool_fpn_forward(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                                const float* offset, float gamma, int out_h, int out_w, int sampling_ratio,
                                float finest_scale, void* out, const int64_t* out_strides, void* stream) {
  int rc = check_levels(feats, L);
  if (rc) return rc;
  rc = check_common(rois, K, out_h, out_w, sampling_ratio);
  if (rc) return rc;
  if (dtype != RAF_F32 && dtype != RAF_F16 && dtype != RAF_BF16) return RAF_ERR_DTYPE;
  if (!(finest_scale > 0.0f) || !(gamma == gamma)) return RAF_ERR_SHAPE;
  if (!out_strides) return RAF_ERR_NULL;
  if (K == 0) return RAF_OK;
  for (int i = 0; i < 4; ++i) if (out_strides[i] <= 0) return RAF_ERR_STRIDE;
  if (!out) return RAF_ERR_NULL;
  LevelsParam p;
  fill_param(feats, L, &p);
  return launch_deform_forward(p, dtype, rois, K, offset, gamma, out_h, out_w, sampling_ratio, finest_scale, out, out_strides,
                               unit_channel_stride(feats, L), (cudaStream_t)stream);
}

int roi_deform_pool_fpn_backward(const raf_level* feats, const raf_level* grad_feats, int L, raf_dtype dtype,
                                 const void* grad_out, const int64_t* gout_strides, const float* rois, int K,
                                 const float* offset, float gamma, int out_h, int out_w, int sampling_ratio,
                                 float finest_scale, float* grad_offset, int flags, void* stream) {
  int rc = check_levels(feats, L);
  if (rc) return rc;
  if (grad_feats) {
    rc = check_levels(grad_feats, L);
    if (rc) return rc;
    for (int l = 0; l < L; ++l)
      if (grad_feats[l].n != feats[l].n || grad_feats[l].c != feats[l].c || grad_feats[l].h != feats[l].h ||
          grad_feats[l].w != feats[l].w)
        return RAF_ERR_SHAPE;
  }
  rc = check_common(rois, K, out_h, out_w, sampling_ratio);
  if (rc) return rc;
  if (dtype != RAF_F32 && dtype != RAF_F16 && dtype != RAF_BF16) return RAF_ERR_DTYPE;
  if (!(finest_scale > 0.0f) || !(gamma == gamma)) return RAF_ERR_SHAPE;
  if (flags & ~RAF_ACCUMULATE) return RAF_ERR_UNSUPPORTED;
  if (!gout_strides) return RAF_ERR_NULL;
  for (int i = 0; i < 4; ++i) if (K > 0 && gout_strides[i] <= 0) return RAF_ERR_STRIDE;
  if (K > 0 && !grad_out) return RAF_ERR_NULL;
  cudaStream_t st = (cudaStream_t)stream;
  if (grad_feats && !(flags & RAF_ACCUMULATE)) {
    rc = zero_fill(grad_feats, L, st);
    if (rc) return rc;
  }
  if (K == 0) return RAF_OK;
  if (grad_offset) {
    if (cudaMemsetAsync(grad_offset, 0, sizeof(float) * (size_t)K * 2 * out_h * out_w, st) != cudaSuccess) return RAF_ERR_CUDA;
    count_launch();
  }
  if (!grad_feats && !grad_offset) return RAF_OK;
  LevelsParam p, gp;
  fill_param(feats, L, &p);
  fill_param(grad_feats ? grad_feats : feats, L, &gp);
  return launch_deform_backward(p, gp, grad_feats != nullptr, dtype, rois, K, offset, gamma, out_h, out_w, sampling_ratio,
                                finest_scale, grad_out, gout_strides, grad_offset,
                                unit_channel_stride(feats, L) && (!grad_feats || unit_channel_stride(grad_feats, L)), st);
}

// ---- NMS / Soft-NMS ------------------------------------------------------------------------------------
size_t roi_nms_workspace_bytes(int n) { return nms_workspace_bytes(n > 0 ? n : 0); }

int roi_nms(const float* boxes, const float* scores, int n, float iou_threshold, int32_t* keep,
            int32_t* num_keep, void* ws, size_t ws_bytes, void* stream) {
  if (n < 0 || n > 65536) return RAF_ERR_SHAPE;
  if (!num_keep || (n > 0 && (!boxes || !scores || !keep))) return RAF_ERR_NULL;
  if (n > 0 && !ws) return RAF_ERR_NULL;
  if (n > 0 && (((uintptr_t)ws % 256) || ws_bytes < nms_workspace_bytes(n))) return RAF_ERR_WORKSPACE;
  return launch_nms(boxes, scores, n, iou_threshold, keep, num_keep, ws, (cudaStream_t)stream);
}

int roi_soft_nms(const float* boxes, const float* scores, int n, float iou_threshold, float sigma,
                 float min_score, int method, int32_t* keep, float* new_scores, int32_t* num_keep,
                 void* ws, size_t ws_bytes, void* stream) {
  (void)ws; (void)ws_bytes;
  if (n < 0 || n > 8192) return RAF_ERR_SHAPE;
  if (method != RAF_SOFT_LINEAR && method != RAF_SOFT_GAUSSIAN) return RAF_ERR_UNSUPPORTED;
  if (method == RAF_SOFT_GAUSSIAN && !(sigma > 0.0f)) return RAF_ERR_SHAPE;
  if (!num_keep || (n > 0 && (!boxes || !scores || !keep || !new_scores))) return RAF_ERR_NULL;
  return launch_soft_nms(boxes, scores, n, iou_threshold, sigma, min_score, method, keep, new_scores, num_keep, ws,
                         (cudaStream_t)stream);
}

// ---- end-to-end variants with HOST buffers -----------------------------------------------------
static bool tensor_dense(int K, int C, int PH, int PW, const int64_t* s) {
  raf_level v;
  v.n = K; v.c = C; v.h = PH; v.w = PW; v.sn = s[0]; v.sc = s[1]; v.sh = s[2]; v.sw = s[3];
  return level_dense(v);
}

size_t roi_align_fpn_host_arena_bytes(const raf_level* levels, int L, raf_dtype dtype, int K,
                                      int out_h, int out_w, int sampling_ratio, int flags) {
  if (!levels || L < 1 || L > kMaxLevels || K < 0) return 0;
  size_t total = 256;
  for (int l = 0; l < L; ++l)   // features (dtype) or gradients (fp32): size for the larger
    total += align256((size_t)levels[l].n * levels[l].c * levels[l].h * levels[l].w * 4);
  total += align256((size_t)K * 20);
  total += align256((size_t)K * levels[0].c * out_h * out_w * esize(dtype));
  total += roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, flags);
  return total;
}

int roi_align_fpn_forward_host(const raf_level* feats_host, int L, raf_dtype dtype,
                               const float* rois_host, int K, int out_h, int out_w,
                               int sampling_ratio, int aligned, float finest_scale, void* out_host,
                               const int64_t* out_strides, void* arena, size_t arena_bytes,
                               void* stream) {
  int rc = check_levels(feats_host, L);
  if (rc) return rc;
  if (dtype != RAF_F32 && dtype != RAF_F16 && dtype != RAF_BF16) return RAF_ERR_DTYPE;
  rc = check_common(rois_host, K, out_h, out_w, sampling_ratio);   // everything host-detectable before the first copy
  if (rc) return rc;
  if (!(finest_scale > 0.0f)) return RAF_ERR_SHAPE;
  if (!out_strides || !arena || (K > 0 && (!rois_host || !out_host))) return RAF_ERR_NULL;
  if (arena_bytes < roi_align_fpn_host_arena_bytes(feats_host, L, dtype, K, out_h, out_w, sampling_ratio, 0))
    return RAF_ERR_WORKSPACE;
  if (!tensor_dense(K, feats_host[0].c, out_h, out_w, out_strides)) return RAF_ERR_STRIDE;
  cudaStream_t st = (cudaStream_t)stream;
  char* cur = (char*)arena;
  raf_level dev[kMaxLevels];
  for (int l = 0; l < L; ++l) {
    if (!level_dense(feats_host[l])) return RAF_ERR_STRIDE;
    const size_t bytes = (size_t)feats_host[l].n * feats_host[l].c * feats_host[l].h * feats_host[l].w * esize(dtype);
    dev[l] = feats_host[l];
    dev[l].data = cur;
    if (cudaMemcpyAsync(cur, feats_host[l].data, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return RAF_ERR_CUDA;
    cur += align256(bytes);
  }
  float* d_rois = (float*)cur;
  if (K > 0 && cudaMemcpyAsync(d_rois, rois_host, (size_t)K * 20, cudaMemcpyHostToDevice, st) != cudaSuccess) return RAF_ERR_CUDA;
  cur += align256((size_t)K * 20);
  void* d_out = cur;
  const size_t out_bytes = (size_t)K * feats_host[0].c * out_h * out_w * esize(dtype);
  cur += align256(out_bytes);
  const size_t ws_bytes = roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, 0);
  rc = roi_align_fpn_forward(dev, L, dtype, d_rois, K, out_h, out_w, sampling_ratio, aligned,
                             finest_scale, d_out, out_strides, cur, ws_bytes, stream);
  if (rc) return rc;
  if (K > 0 && cudaMemcpyAsync(out_host, d_out, out_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) return RAF_ERR_CUDA;
  return RAF_OK;
}

int roi_align_fpn_backward_host(const raf_level* grad_feats_host, int L, raf_dtype gout_dtype,
                                const void* grad_out_host, const int64_t* gout_strides,
                                const float* rois_host, int K, int out_h, int out_w,
                                int sampling_ratio, int aligned, float finest_scale, int flags,
                                void* arena, size_t arena_bytes, void* stream) {
  int rc = check_levels(grad_feats_host, L);
  if (rc) return rc;
  if (gout_dtype != RAF_F32 && gout_dtype != RAF_F16 && gout_dtype != RAF_BF16) return RAF_ERR_DTYPE;
  rc = check_common(rois_host, K, out_h, out_w, sampling_ratio);   // everything host-detectable before the first copy
  if (rc) return rc;
  if (!(finest_scale > 0.0f)) return RAF_ERR_SHAPE;
  if (flags & ~(RAF_ACCUMULATE | RAF_DETERMINISTIC | RAF_ATOMIC | RAF_REUSE_PREP | RAF_PULL_STRIP | RAF_PULL_TILE)) return RAF_ERR_UNSUPPORTED;
  if ((flags & RAF_DETERMINISTIC) && (flags & RAF_ATOMIC)) return RAF_ERR_UNSUPPORTED;
  if ((flags & RAF_PULL_STRIP) && (flags & (RAF_PULL_TILE | RAF_ATOMIC))) return RAF_ERR_UNSUPPORTED;
  if ((flags & RAF_PULL_TILE) && (flags & RAF_ATOMIC)) return RAF_ERR_UNSUPPORTED;
  if (!gout_strides || !arena || (K > 0 && (!rois_host || !grad_out_host))) return RAF_ERR_NULL;
  if (arena_bytes < roi_align_fpn_host_arena_bytes(grad_feats_host, L, gout_dtype, K, out_h, out_w, sampling_ratio, flags))
    return RAF_ERR_WORKSPACE;
  if (!tensor_dense(K, grad_feats_host[0].c, out_h, out_w, gout_strides)) return RAF_ERR_STRIDE;
  cudaStream_t st = (cudaStream_t)stream;
  char* cur = (char*)arena;
  raf_level dev[kMaxLevels];
  size_t lbytes[kMaxLevels];
  for (int l = 0; l < L; ++l) {
    if (!level_dense(grad_feats_host[l])) return RAF_ERR_STRIDE;
    lbytes[l] = (size_t)grad_feats_host[l].n * grad_feats_host[l].c * grad_feats_host[l].h * grad_feats_host[l].w * 4;
    dev[l] = grad_feats_host[l];
    dev[l].data = cur;
    if ((flags & RAF_ACCUMULATE) &&
        cudaMemcpyAsync(cur, grad_feats_host[l].data, lbytes[l], cudaMemcpyHostToDevice, st) != cudaSuccess) return RAF_ERR_CUDA;
    cur += align256(lbytes[l]);
  }
  float* d_rois = (float*)cur;
  if (K > 0 && cudaMemcpyAsync(d_rois, rois_host, (size_t)K * 20, cudaMemcpyHostToDevice, st) != cudaSuccess) return RAF_ERR_CUDA;
  cur += align256((size_t)K * 20);
  void* d_gout = cur;
  const size_t gout_bytes = (size_t)K * grad_feats_host[0].c * out_h * out_w * esize(gout_dtype);
  if (K > 0 && cudaMemcpyAsync(d_gout, grad_out_host, gout_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return RAF_ERR_CUDA;
  cur += align256(gout_bytes);
  const size_t ws_bytes = roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, flags);
  rc = roi_align_fpn_backward(dev, L, gout_dtype, d_gout, gout_strides, d_rois, K, out_h, out_w,
                              sampling_ratio, aligned, finest_scale, flags, cur, ws_bytes, stream);
  if (rc) return rc;
  for (int l = 0; l < L; ++l)
    if (cudaMemcpyAsync(grad_feats_host[l].data, dev[l].data, lbytes[l], cudaMemcpyDeviceToHost, st) != cudaSuccess) return RAF_ERR_CUDA;
  return RAF_OK;
}

const char* roi_align_fpn_strerror(int status) {
  switch (status) {
    case RAF_OK: return "ok";
    case RAF_ERR_NULL: return "a required pointer is NULL";
    case RAF_ERR_SHAPE: return "invalid shape / size / count argument";
    case RAF_ERR_DTYPE: return "unknown dtype";
    case RAF_ERR_STRIDE: return "invalid stride";
    case RAF_ERR_UNSUPPORTED: return "valid request not supported by this build";
    case RAF_ERR_WORKSPACE: return "workspace too small";
    case RAF_ERR_CUDA: return "CUDA runtime error";
  }
  return "unknown status";
}

uint64_t roi_align_fpn_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

}  // extern "C"
