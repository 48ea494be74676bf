/* raf.h -- C ABI of libraf.so: B200-native multi-level (FPN) RoIAlign forward + backward.
 *
 * The operation is the RoIExtractor of a two-stage detector ("extracts RoI-wise features from a
 * single or multiple feature maps with RoIPooling-like operators ... from the corresponding level
 * of feature pyramids ... SingleRoIExtractor", section 3.1), run on the GPU as
 * the paper claims for "all basic bbox and mask operations".  The paper gives no
 * formula; the arithmetic is BASELINE.json `north_star` + the public RoIAlign definition (Mask
 * R-CNN) as fixed in SURVEY.md section 8(c) C1-C5 and DESIGN.md section 3.
 *
 * General conventions
 *  - Every pointer is a DEVICE pointer unless the parameter comment says HOST.
 *  - The caller owns every buffer, including the workspace.  The library keeps no state between calls
 *    (the one process-wide variable is the monotonic launch counter behind roi_align_fpn_launch_count),
 *    never allocates, never synchronises, never copies device->host (the *_host entry points below
 *    are the stated exception: they copy between the caller's host buffers and the caller's
 *    device arena).  All work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = the
 *    legacy default stream).  Calls are CUDA-graph capturable.
 *  - Return value: RAF_OK or a negative raf_status, decided on the host before any launch; no
 *    exception crosses the ABI.  Launch failures are reported as RAF_ERR_CUDA.
 *  - rois: float32 [K,5] row-major, row = (batch_idx, x1, y1, x2, y2) in image pixels.  A RoI whose
 *    batch_idx is not an integer in [0,N) yields an all-zero output row and no gradient.
 *    Non-finite coordinates are memory-safe but unspecified in value.
 *  - K == 0 returns RAF_OK without launching (backward still zero-fills in overwrite mode).
 */
#ifndef RAF_H_
#define RAF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  RAF_OK = 0,
  RAF_ERR_NULL = -1,        /* a required pointer is NULL                                        */
  RAF_ERR_SHAPE = -2,       /* L not in [1,8], K < 0, out_h/out_w not in [1,32], sampling_ratio < 0
                               or > 16, n/c mismatch across levels, non-positive dimension        */
  RAF_ERR_DTYPE = -3,       /* unknown raf_dtype                                                  */
  RAF_ERR_STRIDE = -4,      /* zero / negative stride (overlapping strides are the caller's to avoid) */
  RAF_ERR_UNSUPPORTED = -5, /* valid request this version does not implement                      */
  RAF_ERR_WORKSPACE = -6,   /* ws_bytes smaller than the *_workspace_bytes() query, or ws not 256-aligned */
  RAF_ERR_CUDA = -7         /* a CUDA runtime call / launch failed                                */
} raf_status;

typedef enum { RAF_F32 = 0, RAF_F16 = 1, RAF_BF16 = 2 } raf_dtype;

/* One FPN level.  The array of L descriptors lives in HOST memory and is read at call time. */
typedef struct {
  void* data;             /* DEVICE pointer: features (read-only) or gradients (written)           */
  int32_t n, c, h, w;     /* logical shape [N,C,H,W]; n and c identical across levels              */
  int64_t sn, sc, sh, sw; /* strides in ELEMENTS: NCHW and channels-last are both expressible      */
  float spatial_scale;    /* 1/stride of the level (0.25, 0.125, ...)                              */
} raf_level;

/* Backward flags (bitmask). */
enum {
  RAF_ACCUMULATE = 1,     /* add into the existing gradient pyramid instead of overwriting it      */
  RAF_DETERMINISTIC = 2,  /* REQUIRE a bit-reproducible pull kernel (K3d); RAF_ERR_UNSUPPORTED if the
                             layout is not eligible (needs channels-last operands, C % 4 == 0,
                             L*N <= 2047; any out_h, out_w <= 32 and any sampling grid incl. 0)     */
  RAF_ATOMIC = 4,         /* force the atomic scatter variant (zero-fill + red.global.add.v4.f32)  */
  RAF_REUSE_PREP = 8      /* the workspace still holds what roi_align_fpn_forward wrote into it when
                             called with the SAME rois pointer and K, level shapes and scales, out_h/out_w,
                             sampling_ratio, aligned, finest_scale: the backward then skips its own RoI
                             bucketing / tap-table launch.  The forward leaves the workspace in that state
                             when it returns RAF_OK (unless RAF_NO_PREP).  The tables carry a fingerprint
                             of those arguments; on a mismatch (other RoI tensor, other geometry, a
                             workspace never written) the pull kernel computes nothing from them and fills
                             the WHOLE gradient pyramid with NaN.  Changing the contents of the rois
                             buffer in place between the two calls is not detected.                     */
};
/* Backward with a 16-bit gradient pyramid ("optional bf16 grad output"): grad_dtype = RAF_F32 is
 * roi_align_fpn_backward; grad_dtype = gout_dtype (RAF_F16 / RAF_BF16) writes the pyramid in that type -- sums are
 * formed in fp32 registers and rounded once per element (tiles that meet more RoIs than one pass takes park their
 * partial sums in the pyramid, i.e. round once per pass).  Pull kernels only: RAF_ATOMIC, RAF_REPACK and layouts the
 * pull kernels do not take return RAF_ERR_UNSUPPORTED; so does any other combination of the two dtypes. */
int roi_align_fpn_backward_ex(const raf_level* grad_feats, int L, raf_dtype gout_dtype, raf_dtype grad_dtype,
                              const void* grad_out, const int64_t* gout_strides, const float* rois,
                              int K, int out_h, int out_w, int sampling_ratio, int aligned,
                              float finest_scale, int flags, void* ws, size_t ws_bytes, void* stream);

/* The deterministic pull backward has two kernels with the same contract and the same prep tables: the
 * TILE kernel (a CTA owns 8 x 8 pixels, one pixel per warp at a time) and the STRIP kernel (a warp owns
 * a tile and walks it in 8-pixel row strips, loading every grad_out vector once per strip; no limit on
 * out_h, out_w <= 32 or on the sampling grid).  The library picks per call (strip for large batches of
 * 7 x 7-like outputs, tile otherwise); these two flags force one of them (RAF_ERR_UNSUPPORTED if that
 * kernel does not take the arguments; both together are refused). */
enum {
  RAF_PULL_STRIP = 32,
  RAF_PULL_TILE = 64
};
/* Forward flags (roi_align_fpn_forward_ex). */
enum {
  RAF_NO_PREP = 16        /* forward only (inference): do not write the backward's prep tables; the
                             workspace is not touched and `ws` may be NULL                           */
};
/* Forward and backward flag: NCHW-contiguous operands (every level dense [N,C,H,W], out / grad_out dense
 * [K,C,out_h,out_w]) are REPACKED to channels-last inside the workspace, the channels-last kernels run on the
 * copies, and the result is repacked back -- all on `stream`, all inside the call ("any NCHW -> channel-last
 * repack counted in the timing", north_star).  `ws` must then hold roi_align_fpn_workspace_bytes(...) +
 * roi_align_fpn_repack_bytes(...) bytes (else RAF_ERR_WORKSPACE).  Ignored when the operands already are
 * channels-last; RAF_ERR_STRIDE when they are neither.  Without the flag NCHW runs on the strided
 * thread-per-element kernels (no extra memory, about 2.5x slower). */
enum { RAF_REPACK = 128 };
/* Bytes of channels-last scratch RAF_REPACK needs for these levels and this RoI tensor (the larger of the
 * forward's and the backward's need; 256-aligned).  `levels`: HOST array, only the shapes are read. */
size_t roi_align_fpn_repack_bytes(const raf_level* levels, int L, raf_dtype dtype, int K, int out_h, int out_w);
/* With neither RAF_DETERMINISTIC nor RAF_ATOMIC the library picks the pull variant when eligible
 * and the atomic variant otherwise. */

/* Bytes of device workspace the calls below need for these arguments (never 0; 256-aligned). */
size_t roi_align_fpn_workspace_bytes(int K, int L, int out_h, int out_w, int sampling_ratio,
                                     int flags);

/* Level assignment + per-level histogram + stable bucketing (north_star).
 *   level_k = #{ j in [1,L-1] : t_k >= 2^j },  t_k = sqrt((x2-x1)*(y2-y1)) / finest_scale + 1e-6f,
 *   every operation an individually rounded fp32 IEEE operation (== clamp(floor(log2 t),0,L-1)).
 *   counts[l] = #{k : level_k = l};  perm = RoI indices grouped by level, ascending k inside a
 *   level (stable).  levels[K], counts[L], perm[K] are int32 DEVICE buffers; any of the three may
 *   be NULL if not wanted. */
int roi_fpn_assign_levels(const float* rois, int K, int L, float finest_scale, int32_t* levels,
                          int32_t* counts, int32_t* perm, void* ws, size_t ws_bytes, void* stream);

/* Forward:
 *   out[k,c,ph,pw] = (1/count) * sum_{iy<gh, ix<gw} bilinear(F_{level_k}[b_k,c], y(ph,iy), x(pw,ix))
 * with fp32 sample coordinates in the canonical operation order, fp32 accumulation.
 *   feats        HOST array of L descriptors (device data pointers), dtype = `dtype`
 *   out          DEVICE, dtype = `dtype`, logical [K,C,out_h,out_w] addressed through
 *                out_strides (HOST array of 4 element strides); row k = RoI k (original order)
 *   sampling_ratio  > 0: fixed grid; 0: adaptive gh = ceil(roi_h/out_h), gw = ceil(roi_w/out_w) (per RoI; the
 *                channels-last kernels tabulate grids up to 8 x 8 and sample larger ones directly)
 *   aligned      != 0: half-pixel shift, no minimum box size; 0: legacy (no shift, size >= 1)
 *   ws           written: RoI buckets, windows, geometry and tap tables that a following
 *                roi_align_fpn_backward on the same arguments may reuse (RAF_REUSE_PREP); 256-byte aligned */
int roi_align_fpn_forward(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                          int out_h, int out_w, int sampling_ratio, int aligned, float finest_scale,
                          void* out, const int64_t* out_strides, void* ws, size_t ws_bytes,
                          void* stream);

/* Forward with flags: 0 = roi_align_fpn_forward; RAF_NO_PREP = gather only. */
int roi_align_fpn_forward_ex(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                             int out_h, int out_w, int sampling_ratio, int aligned, float finest_scale,
                             void* out, const int64_t* out_strides, int flags, void* ws, size_t ws_bytes,
                             void* stream);

/* Backward: exact transpose of the forward.
 *   grad_feats   HOST array of L descriptors; data = fp32 DEVICE gradient pyramid, same logical
 *                shapes as the features.  Overwritten (every element written: zero or sum) unless
 *                RAF_ACCUMULATE.
 *   grad_out     DEVICE, dtype = gout_dtype, logical [K,C,out_h,out_w] through gout_strides (HOST)
 *   flags        RAF_ACCUMULATE | RAF_DETERMINISTIC | RAF_ATOMIC | RAF_REUSE_PREP | RAF_PULL_STRIP | RAF_PULL_TILE | RAF_REPACK */
int roi_align_fpn_backward(const raf_level* grad_feats, int L, raf_dtype gout_dtype,
                           const void* grad_out, const int64_t* gout_strides, const float* rois,
                           int K, int out_h, int out_w, int sampling_ratio, int aligned,
                           float finest_scale, int flags, void* ws, size_t ws_bytes, void* stream);

/* Backward WITHOUT a caller workspace and without any device allocation (for callers that cannot call cudaMalloc:
 * code under CUDA graph capture, tight serving loops, harnesses that forbid it).  Same operation, kernels and
 * results as roi_align_fpn_backward (fp32 gradient pyramid); the scratch it needs -- the prep tables:
 * RoI buckets, windows, geometry, tap tables -- lives in a static device array of RAF_STATIC_WS_BYTES inside the
 * library, which every GPU that loads the library holds until the process exits.
 *   limit    roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, flags) <= RAF_STATIC_WS_BYTES, else
 *            RAF_ERR_WORKSPACE, decided on the host before any CUDA call (4 MiB: K = 8192 RoIs at 7 x 7 bins,
 *            K = 4096 at 14 x 14, sampling_ratio 2)
 *   flags    RAF_ACCUMULATE | RAF_DETERMINISTIC | RAF_ATOMIC | RAF_PULL_STRIP | RAF_PULL_TILE; RAF_REUSE_PREP and
 *            RAF_REPACK return RAF_ERR_UNSUPPORTED (the array is shared by all calls and has no room for repack copies)
 *   sharing  all calls on a device use the same array and it keeps the last call's contents: each call first clears
 *            the fingerprint header (a 256-byte cudaMemsetAsync on `stream`, enqueued before the remaining argument
 *            checks) and its prep launch rewrites everything the backward then reads.  Calls that OVERLAP on the GPU
 *            (different streams without ordering between them) race on the array: order them.
 * Calls no cudaMalloc, cudaFree or allocating library routine; the array's device address is looked up once per
 * device (cudaGetSymbolAddress, with the caller's current device). */
#define RAF_STATIC_WS_BYTES (4u << 20)
int roi_align_fpn_backward_static(const raf_level* grad_feats, int L, raf_dtype gout_dtype,
                                  const void* grad_out, const int64_t* gout_strides, const float* rois,
                                  int K, int out_h, int out_w, int sampling_ratio, int aligned,
                                  float finest_scale, int flags, void* stream);

/* ---- the max variant of the "RoIPooling-like operators" (the RoI pooling
 * layer of Fast R-CNN), on the same FPN level map (C1) -------------------------------------------
 * Window of bin (ph,pw) on the RoI's level (fp32, each operation rounded; readings P1-P4):
 *   sw = roundf(x1*scale), ew = roundf(x2*scale), rw = max(ew - sw + 1, 1), bw = rw / out_w,
 *   ws = clamp(floorf(pw*bw) + sw, 0, W), we = clamp(ceilf((pw+1)*bw) + sw, 0, W); rows likewise.
 * out = max of the features over the window (0 for an empty window or an invalid batch index);
 * argmax (int32 DEVICE, same logical shape and strides as `out`; may be NULL) = y*W + x of the FIRST maximum
 * in row-major order, -1 when there is none.  NaN never wins.  Values are copies of inputs: exact. */
int roi_pool_fpn_forward(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                         int out_h, int out_w, float finest_scale, void* out, int32_t* argmax,
                         const int64_t* out_strides, void* stream);

/* Backward of RoIPool-max: grad_feats[level_k][b_k][c][argmax] += grad_out[k,c,ph,pw] (fp32 atomics: the
 * summation order is not fixed).  grad_feats is zero-filled first unless RAF_ACCUMULATE (the only flag
 * accepted).  argmax: what roi_pool_fpn_forward wrote for the same rois, addressed through gout_strides;
 * entries that are not a pixel index of the RoI's level are ignored. */
int roi_pool_fpn_backward(const raf_level* grad_feats, int L, raf_dtype gout_dtype, const void* grad_out,
                          const int32_t* argmax, const int64_t* gout_strides, const float* rois, int K,
                          int out_h, int out_w, float finest_scale, int flags, void* stream);

/* ---- the RoIAlign gather fused into the box head's first fully connected layer (RoIHead /
 * BBoxHead; "2fc" heads PAPER.md:269-271).  Readings F1-F3:
 *   out[k, n] = sum_{ph,pw,c} A[k, (ph*out_w + pw)*C + c] * weight[n, (ph*out_w + pw)*C + c]  (+ bias[n])
 * with A = the RoIAlign forward of RoI k (same definition as roi_align_fpn_forward) ROUNDED to `dtype`, i.e. exactly
 * the RoI feature tensor the head would read -- but it is never written: tiles of it are produced straight into the
 * A operand of a tcgen05 GEMM (bf16 / fp16 inputs, fp32 accumulation in tensor memory).
 *   feats    channels-last (sc == 1), dtype RAF_F16 or RAF_BF16, C % 64 == 0
 *   weight   DEVICE, dtype, [n_out, out_h*out_w*C] row-major, columns in (ph, pw, c) order; n_out % 512 == 0
 *   bias     DEVICE fp32 [n_out] or NULL
 *   out      DEVICE fp32 [K, n_out] row-major, overwritten (zero-filled, then fp32 reductions: the summation order
 *            over the out_h split-K slices is not fixed)
 *   sampling_ratio 1 or 2.  Anything else: RAF_ERR_UNSUPPORTED. */
int roi_align_fc_fpn_forward(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                             int out_h, int out_w, int sampling_ratio, int aligned, float finest_scale,
                             const void* weight, const float* bias, int n_out, float* out, void* stream);

/* ---- deformable RoI pooling ("DCN [8]: deformable convolution and deformable RoI pooling",
 * PAPER.md:57-58), on the same FPN level map (C1).  Readings D1-D5: RoIAlign with the half-pixel
 * shift and no minimum size whose bin (ph,pw) is moved by (gamma*rw*offset[k,0,ph,pw], gamma*rh*offset[k,1,ph,pw])
 * feature pixels (rw, rh = RoI size on its level): sample coordinate = the C3 coordinate + that shift (one more fp32
 * addition), then the C3 tap rule; out = sum / count.
 *   offset   float32 DEVICE [K,2,out_h,out_w] contiguous (plane 0 = x, 1 = y); NULL = all zero (= RoIAlign)
 *   sampling_ratio  > 0 fixed grid, 0 adaptive (ceil of the bin size)
 * fp32 coordinates bit-identical to the oracle's, fp32 accumulation. */
int roi_deform_pool_fpn_forward(const raf_level* feats, int L, raf_dtype dtype, const float* rois, int K,
                                const float* offset, float gamma, int out_h, int out_w, int sampling_ratio,
                                float finest_scale, void* out, const int64_t* out_strides, void* stream);

/* Backward of deformable RoI pooling.  grad_feats (HOST array of L fp32 descriptors, or NULL): += the exact
 * transpose (fp32 atomics; zero-filled first unless RAF_ACCUMULATE).  grad_offset (float32 DEVICE [K,2,out_h,out_w],
 * or NULL): overwritten with d loss / d offset -- the derivative of the forward where it exists (a sample whose
 * coordinate is clamped at a border does not move with the offset).  feats: the forward's features (read for the
 * offset gradient), dtype = grad_out's dtype.  flags: RAF_ACCUMULATE only (applies to grad_feats). */
int roi_deform_pool_fpn_backward(const raf_level* feats, const raf_level* grad_feats, int L, raf_dtype dtype,
                                 const void* grad_out, const int64_t* gout_strides, const float* rois, int K,
                                 const float* offset, float gamma, int out_h, int out_w, int sampling_ratio,
                                 float finest_scale, float* grad_offset, int flags, void* stream);

/* ---- NMS and Soft-NMS on the GPU ("Soft NMS [1]: an alternative to NMS", PAPER.md:55;
 * "All basic bbox and mask operations run on GPUs") ---------------------------------------------
 * boxes: float32 DEVICE [n,4] = (x1,y1,x2,y2), continuous coordinates (no "+1"); scores: float32 DEVICE [n],
 * no NaN.  IoU = inter / ((area_a + area_b) - inter), fp32, each operation rounded (readings N1-N6).
 * Greedy NMS: boxes in descending score (ties: lower index first); a box is dropped when an earlier KEPT box
 * has IoU > iou_threshold (strict).  keep[n] int32 DEVICE receives the kept indices in that order,
 * num_keep[1] int32 DEVICE their number.  n <= 65536.  ws: roi_nms_workspace_bytes(n) bytes, 256-aligned. */
size_t roi_nms_workspace_bytes(int n);
int roi_nms(const float* boxes, const float* scores, int n, float iou_threshold, int32_t* keep,
            int32_t* num_keep, void* ws, size_t ws_bytes, void* stream);

/* Soft-NMS: repeatedly emit the remaining box of highest current score (ties: lowest index) and decay every
 * other remaining score by  method RAF_SOFT_LINEAR: (iou > iou_threshold ? 1 - iou : 1),
 * RAF_SOFT_GAUSSIAN: exp(-iou*iou / sigma);  boxes whose score falls below min_score are dropped.
 * keep[n] / new_scores[n] in emission order, num_keep[1] their number.  n <= 8192 (one CTA, scores in
 * shared memory).  The Gaussian method uses expf: scores agree with a host evaluation to a few ulp. */
enum { RAF_SOFT_LINEAR = 1, RAF_SOFT_GAUSSIAN = 2 };
int roi_soft_nms(const float* boxes, const float* scores, int n, float iou_threshold, float sigma,
                 float min_score, int method, int32_t* keep, float* new_scores, int32_t* num_keep,
                 void* ws, size_t ws_bytes, void* stream);

/* End-to-end variants with HOST buffers (used for the e2e benchmark line): every `data` pointer in
 * the descriptors, `rois`, `out` / `grad_out` are HOST pointers (pinned for full copy speed) and
 * must be contiguous in the order the strides describe (each level / tensor occupies exactly
 * n*c*h*w resp. K*C*out_h*out_w elements).  The call copies the inputs into `arena` (DEVICE,
 * caller-owned, at least roi_align_fpn_host_arena_bytes()), runs the device path, and copies the
 * result back, all on `stream`; it does not synchronise. */
size_t roi_align_fpn_host_arena_bytes(const raf_level* levels, int L, raf_dtype dtype, int K,
                                      int out_h, int out_w, int sampling_ratio, int flags);
int roi_align_fpn_forward_host(const raf_level* feats_host, int L, raf_dtype dtype,
                               const float* rois_host, int K, int out_h, int out_w,
                               int sampling_ratio, int aligned, float finest_scale, void* out_host,
                               const int64_t* out_strides, void* arena, size_t arena_bytes,
                               void* stream);
int roi_align_fpn_backward_host(const raf_level* grad_feats_host, int L, raf_dtype gout_dtype,
                                const void* grad_out_host, const int64_t* gout_strides,
                                const float* rois_host, int K, int out_h, int out_w,
                                int sampling_ratio, int aligned, float finest_scale, int flags,
                                void* arena, size_t arena_bytes, void* stream);

/* Static description of a status code. */
const char* roi_align_fpn_strerror(int status);

/* Number of kernels the library has launched in this process (monotonic; for bench accounting). */
uint64_t roi_align_fpn_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* RAF_H_ */
