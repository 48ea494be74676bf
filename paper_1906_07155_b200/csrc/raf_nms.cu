// raf_nms.cu -- greedy NMS and Soft-NMS on the GPU ("Soft NMS [1]: an alternative to
// NMS"; "All basic bbox and mask operations run on GPUs"): the step that produces
// the RoIs the RoIAlign path consumes.  Readings N1-N6 in DESIGN.md 3b.
//
//   N1  order: descending score, ties by ascending index
//   N2  IoU = inter / ((area_a + area_b) - inter), continuous coordinates, fp32, each operation rounded
//   N3  greedy: a box is dropped when an earlier KEPT box has IoU > threshold (strict)
//   N4-N6  Soft-NMS: emit the best remaining box, decay the others (linear / Gaussian), prune by min_score
//
// Greedy NMS is three launches, everything stays on the device:
//   nms_rank_kernel   rank_i = #{j : s_j > s_i or (s_j == s_i and j < i)} (all-pairs, scores tiled through
//                     shared memory) -> sorted copy of the boxes + order[]; no general sort is needed at the
//                     sizes NMS runs on (n^2 comparisons are what the IoU mask costs anyway)
//   nms_mask_kernel   64 x 64 tiles of the upper triangle: one 64-bit word per (box, tile of later boxes)
//   nms_scan_kernel   one CTA walks the tiles in order: a single thread resolves the 64 boxes of a tile
//                     against each other from the diagonal words, then all threads OR the rows of the kept
//                     boxes into the `removed` bitmap of the later tiles (one (box, word) pair per thread)
// Soft-NMS is inherently sequential in the emitted box: one CTA keeps the current scores in shared memory
// and does an arg-max reduction + a decay sweep per emitted box.
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

constexpr int kNmsTile = 64;

__device__ __forceinline__ float box_iou(const float4 a, const float4 b) {
  float iw = __fsub_rn(fminf(a.z, b.z), fmaxf(a.x, b.x));
  float ih = __fsub_rn(fminf(a.w, b.w), fmaxf(a.y, b.y));
  if (!(iw > 0.0f)) iw = 0.0f;
  if (!(ih > 0.0f)) ih = 0.0f;
  const float inter = __fmul_rn(iw, ih);
  const float aa = __fmul_rn(__fsub_rn(a.z, a.x), __fsub_rn(a.w, a.y));
  const float ab = __fmul_rn(__fsub_rn(b.z, b.x), __fsub_rn(b.w, b.y));
  const float ua = __fsub_rn(__fadd_rn(aa, ab), inter);
  return __fdiv_rn(inter, ua);
}

// Workspace carve-up: [order n int32][sorted boxes n float4][mask n x nwords uint64]
struct NmsWs {
  int32_t* order;
  float4* sorted;
  unsigned long long* mask;
  int nwords;
};
static size_t a256(size_t v) { return (v + 255) & ~(size_t)255; }
size_t nms_workspace_bytes(int n) {
  const size_t nw = ((size_t)n + kNmsTile - 1) / kNmsTile;
  return a256(4 * (size_t)n) + a256(16 * (size_t)n) + a256(8 * (size_t)n * nw) + 256;
}
static NmsWs nms_ws(void* ws, int n) {
  NmsWs w;
  char* p = reinterpret_cast<char*>(ws);
  w.nwords = (n + kNmsTile - 1) / kNmsTile;
  w.order = reinterpret_cast<int32_t*>(p);
  p += a256(4 * (size_t)n);
  w.sorted = reinterpret_cast<float4*>(p);
  p += a256(16 * (size_t)n);
  w.mask = reinterpret_cast<unsigned long long*>(p);
  return w;
}

__global__ void __launch_bounds__(256)
nms_rank_kernel(const float* __restrict__ boxes, const float* __restrict__ scores, int n, int32_t* __restrict__ order,
                float4* __restrict__ sorted) {
  __shared__ float s_s[256];
  const int i = blockIdx.x * 256 + threadIdx.x;
  const float si = i < n ? scores[i] : 0.0f;
  int rank = 0;
  for (int j0 = 0; j0 < n; j0 += 256) {
    const int j = j0 + threadIdx.x;
    s_s[threadIdx.x] = j < n ? scores[j] : 0.0f;
    __syncthreads();
    const int m = min(256, n - j0);
    for (int t = 0; t < m; ++t) {
      const float sj = s_s[t];
      rank += (sj > si) || (sj == si && j0 + t < i);
    }
    __syncthreads();
  }
  if (i < n) {
    order[rank] = i;
    sorted[rank] = make_float4(boxes[4 * i], boxes[4 * i + 1], boxes[4 * i + 2], boxes[4 * i + 3]);
  }
}

// blockIdx = (tile of later boxes cb, tile of rows rb), cb >= rb; thread = row box.
__global__ void __launch_bounds__(kNmsTile)
nms_mask_kernel(const float4* __restrict__ sorted, int n, float thr, unsigned long long* __restrict__ mask, int nwords) {
  const int rb = blockIdx.y, cb = blockIdx.x;
  if (cb < rb) return;
  __shared__ float4 s_b[kNmsTile];
  const int cj = cb * kNmsTile + threadIdx.x;
  if (cj < n) s_b[threadIdx.x] = sorted[cj];
  __syncthreads();
  const int i = rb * kNmsTile + threadIdx.x;
  if (i >= n) return;
  const float4 a = sorted[i];
  const int m = min(kNmsTile, n - cb * kNmsTile);
  unsigned long long bits = 0;
  for (int t = (cb == rb ? threadIdx.x + 1 : 0); t < m; ++t)
    if (box_iou(a, s_b[t]) > thr) bits |= 1ull << t;
  mask[(size_t)i * nwords + cb] = bits;
}

__global__ void __launch_bounds__(256, 1)
nms_scan_kernel(const unsigned long long* __restrict__ mask, const int32_t* __restrict__ order, int n, int nwords,
                int32_t* __restrict__ keep, int32_t* __restrict__ num_keep) {
  extern __shared__ unsigned long long s_removed[];   // [nwords]
  __shared__ unsigned long long s_diag[kNmsTile];
  __shared__ int s_ord[kNmsTile], s_out[kNmsTile], s_bit[kNmsTile];
  __shared__ int s_nk, s_add;
  for (int w = threadIdx.x; w < nwords; w += blockDim.x) s_removed[w] = 0;
  if (threadIdx.x == 0) s_nk = 0;
  __syncthreads();
  for (int tb = 0; tb < nwords; ++tb) {
    const int m = min(kNmsTile, n - tb * kNmsTile);
    if (threadIdx.x < m) {
      s_diag[threadIdx.x] = mask[(size_t)(tb * kNmsTile + threadIdx.x) * nwords + tb];
      s_ord[threadIdx.x] = order[tb * kNmsTile + threadIdx.x];
    }
    __syncthreads();
    if (threadIdx.x == 0) {   // the 64 boxes of the tile against each other, in order (shared memory only)
      unsigned long long rem = s_removed[tb], kept = 0;
      int add = 0;
      for (int b = 0; b < m; ++b)
        if (!((rem >> b) & 1ull)) {
          kept |= 1ull << b;
          rem |= s_diag[b];
          s_bit[add] = b;
          s_out[add++] = s_ord[b];
        }
      s_add = add;
    }
    __syncthreads();
    if (threadIdx.x < s_add) keep[s_nk + threadIdx.x] = s_out[threadIdx.x];
    // rows of the kept boxes -> later tiles: one (kept box, word) pair per thread and step, so that all the
    // loads of a tile are independent (a per-word loop over the kept boxes is a chain of L2 round trips)
    const int nrem = nwords - tb - 1, npair = s_add * nrem;
    for (int e = threadIdx.x; e < npair; e += blockDim.x) {
      const int q = e / nrem, w = tb + 1 + (e - q * nrem);
      const unsigned long long v = mask[(size_t)(tb * kNmsTile + s_bit[q]) * nwords + w];
      if (v) atomicOr(&s_removed[w], v);
    }
    __syncthreads();
    if (threadIdx.x == 0) s_nk += s_add;
  }
  __syncthreads();
  if (threadIdx.x == 0) *num_keep = s_nk;
}

__global__ void nms_zero_count_kernel(int32_t* num_keep) { *num_keep = 0; }

int launch_nms(const float* boxes, const float* scores, int n, float iou_threshold, int32_t* keep, int32_t* num_keep,
               void* ws, cudaStream_t stream) {
  if (n == 0) {
    nms_zero_count_kernel<<<1, 1, 0, stream>>>(num_keep);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
  }
  const NmsWs w = nms_ws(ws, n);
  nms_rank_kernel<<<(n + 255) / 256, 256, 0, stream>>>(boxes, scores, n, w.order, w.sorted);
  count_launch();
  nms_mask_kernel<<<dim3(w.nwords, w.nwords), kNmsTile, 0, stream>>>(w.sorted, n, iou_threshold, w.mask, w.nwords);
  count_launch();
  nms_scan_kernel<<<1, 256, sizeof(unsigned long long) * w.nwords, stream>>>(w.mask, w.order, n, w.nwords, keep, num_keep);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

// ---- Soft-NMS: one CTA; scores and liveness in shared memory ------------------------------------------------
constexpr int kSoftThreads = 1024;

__global__ void __launch_bounds__(kSoftThreads, 1)
soft_nms_kernel(const float* __restrict__ boxes, const float* __restrict__ scores, int n, float thr, float sigma,
                float min_score, int method, int32_t* __restrict__ keep, float* __restrict__ new_scores,
                int32_t* __restrict__ num_keep) {
  extern __shared__ float s_score[];          // [n]; a dropped / emitted box holds -inf and gone = 1
  unsigned char* s_gone = reinterpret_cast<unsigned char*>(s_score + n);
  __shared__ float s_ws[kSoftThreads / 32];
  __shared__ int s_wi[kSoftThreads / 32];
  __shared__ int s_best;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int i = tid; i < n; i += kSoftThreads) {
    const float s = scores[i];
    s_score[i] = s;
    s_gone[i] = !(s >= min_score);
  }
  __syncthreads();
  int nk = 0;
  for (;;) {
    // arg-max of the live scores, ties to the lowest index
    float bs = 0.0f;
    int bi = -1;
    for (int i = tid; i < n; i += kSoftThreads)
      if (!s_gone[i] && (bi < 0 || s_score[i] > bs)) { bs = s_score[i]; bi = i; }
    for (int d = 16; d > 0; d >>= 1) {
      const float os = __shfl_down_sync(0xffffffffu, bs, d);
      const int oi = __shfl_down_sync(0xffffffffu, bi, d);
      if (oi >= 0 && (bi < 0 || os > bs || (os == bs && oi < bi))) { bs = os; bi = oi; }
    }
    if (lane == 0) { s_ws[warp] = bs; s_wi[warp] = bi; }
    __syncthreads();
    if (warp == 0) {
      bs = s_ws[lane];
      bi = s_wi[lane];
      for (int d = 16; d > 0; d >>= 1) {
        const float os = __shfl_down_sync(0xffffffffu, bs, d);
        const int oi = __shfl_down_sync(0xffffffffu, bi, d);
        if (oi >= 0 && (bi < 0 || os > bs || (os == bs && oi < bi))) { bs = os; bi = oi; }
      }
      if (lane == 0) {
        s_best = bi;
        if (bi >= 0) { keep[nk] = bi; new_scores[nk] = bs; s_gone[bi] = 1; }
      }
    }
    __syncthreads();
    const int m = s_best;
    if (m < 0) break;
    ++nk;
    const float4 bm = make_float4(boxes[4 * m], boxes[4 * m + 1], boxes[4 * m + 2], boxes[4 * m + 3]);
    for (int i = tid; i < n; i += kSoftThreads) {
      if (s_gone[i]) continue;
      const float iou = box_iou(bm, make_float4(boxes[4 * i], boxes[4 * i + 1], boxes[4 * i + 2], boxes[4 * i + 3]));
      float f = 1.0f;
      if (method == RAF_SOFT_LINEAR) { if (iou > thr) f = __fsub_rn(1.0f, iou); }
      else if (iou == iou) f = expf(-__fdiv_rn(__fmul_rn(iou, iou), sigma));
      const float s = __fmul_rn(s_score[i], f);
      s_score[i] = s;
      if (!(s >= min_score)) s_gone[i] = 1;
    }
    __syncthreads();
  }
  if (tid == 0) *num_keep = nk;
}

int launch_soft_nms(const float* boxes, const float* scores, int n, float iou_threshold, float sigma, float min_score,
                    int method, int32_t* keep, float* new_scores, int32_t* num_keep, void* ws, cudaStream_t stream) {
  (void)ws;
  if (n == 0) {
    nms_zero_count_kernel<<<1, 1, 0, stream>>>(num_keep);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
  }
  const size_t smem = (size_t)n * 5 + 16;
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(soft_nms_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return RAF_ERR_CUDA;
  soft_nms_kernel<<<1, kSoftThreads, smem, stream>>>(boxes, scores, n, iou_threshold, sigma, min_score, method, keep,
                                                     new_scores, num_keep);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

}  // namespace raf
