// raf_host.h -- internal host-side declarations shared by the raf translation units.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/raf.h"

namespace raf {

struct LevelsParam;

// Common per-call arguments of the RoIAlign kernels.
struct RoiArgs {
  const float* rois;
  int K;
  int PH, PW;
  int sampling_ratio;
  int aligned;
  float finest_scale;
};

void count_launch();

int launch_assign_levels(const float* rois, int K, int L, float finest_scale, int32_t* levels,
                         int32_t* counts, int32_t* perm, cudaStream_t stream);

// Forward.  `channels_last` = every level has sc == 1 and the output has stride 1 along C, with
// 16-byte aligned pixel vectors (checked by the caller).
struct PullPrepOut;
// `prep` (may be null): also write the pull backward's prep tables (see launch_pull_prep) -- in the
// channels-last path they ride in the leading blocks of the forward launch.
int launch_forward(const LevelsParam& lv, raf_dtype dtype, const RoiArgs& a, void* out,
                   const int64_t* out_strides, bool channels_last, const PullPrepOut* prep, cudaStream_t stream);

// Backward (atomic scatter).  The gradient pyramid must already hold its starting values.
int launch_backward_atomic(const LevelsParam& glv, raf_dtype gout_dtype, const RoiArgs& a,
                           const void* grad_out, const int64_t* gout_strides, bool channels_last,
                           cudaStream_t stream);

// One merged bilinear tap of an output bin along one axis (pull backward tap tables).
struct PullTap {
  uint32_t pb;  // pixel | bin << 24; pixel == 0xffffff marks an empty slot
  float w;      // weight (y taps carry 1/count)
};

// Prep launch of the pull backward (sampling_ratio > 0): block 0 buckets the RoIs by (level, image)
// -- bperm[K], boff[L*N + 1], bwin[K] = conservative touched-pixel window of every kept RoI in
// bperm order -- and writes the argument fingerprint; the other blocks write the tap tables
// taps[K][PH + PW][2 * sampling_ratio] (raf_pull_prep.cuh).
size_t bucket_smem_bytes(int L, int N);
int launch_pull_prep(const LevelsParam& lv, const RoiArgs& a, const PullPrepOut& prep, cudaStream_t stream);

// RAF_OK when launch_backward_pull takes these arguments, RAF_ERR_UNSUPPORTED otherwise (host-side test).
int pull_eligible(const LevelsParam& glv, raf_dtype gout_dtype, const RoiArgs& a, const void* grad_out,
                  const int64_t* gout_strides);
// Backward, deterministic pull formulation (channels-last, sampling_ratio > 0).  Writes every
// gradient element exactly once (or adds into it when `accumulate`).  `prep` = the tables
// launch_pull_prep (or the forward) left in the workspace for the same arguments, with the
// fingerprint the kernel checks them against.
int launch_backward_pull(const LevelsParam& glv, raf_dtype gout_dtype, raf_dtype grad_dtype, const RoiArgs& a, const void* grad_out,
                         const int64_t* gout_strides, const PullPrepOut& prep, int accumulate, cudaStream_t stream);

// Second-generation pull backward (raf_backward_strip.cu): row-strip register accumulators, each grad_out
// vector loaded once per strip.  Same prep tables (bperm / boff / bwin / bgeo), same fingerprint check.
int strip_eligible(const LevelsParam& glv, raf_dtype gout_dtype, const RoiArgs& a, const int64_t* gout_strides);
int launch_backward_strip(const LevelsParam& glv, raf_dtype gout_dtype, raf_dtype grad_dtype, const RoiArgs& a, const void* grad_out,
                          const int64_t* gout_strides, const PullPrepOut& prep, int accumulate, cudaStream_t stream);

// RoIPool-max (raf_pool.cu).  `chan_fastest`: enumerate outputs with the channel fastest (channels-last
// features: coalesced window loads).  The gradient pyramid must already hold its starting values.
int launch_pool_forward(const LevelsParam& lv, raf_dtype dtype, const float* rois, int K, int PH, int PW, float fs,
                        void* out, int32_t* argmax, const int64_t* os, bool chan_fastest, cudaStream_t stream);
int launch_pool_backward(const LevelsParam& glv, raf_dtype dtype, const float* rois, int K, int PH, int PW, float fs,
                         const void* gout, const int32_t* argmax, const int64_t* gs, bool chan_fastest, cudaStream_t stream);

// Deformable RoI pooling (raf_deform.cu).  The gradient pyramid / grad_offset must already hold their starting values.
int launch_deform_forward(const LevelsParam& lv, raf_dtype dtype, const float* rois, int K, const float* offset, float gamma,
                          int PH, int PW, int g, float fs, void* out, const int64_t* os, bool chan_fastest, cudaStream_t stream);
int launch_deform_backward(const LevelsParam& lv, const LevelsParam& glv, bool want_feats, raf_dtype dtype, const float* rois,
                           int K, const float* offset, float gamma, int PH, int PW, int g, float fs, const void* gout,
                           const int64_t* gs, float* grad_offset, bool chan_fastest, cudaStream_t stream);

// RoIAlign gather fused into the box head's first FC (raf_fc.cu; tcgen05).  `out` must already be zero.
int launch_fc_fused(const LevelsParam& lv, raf_dtype dtype, const RoiArgs& a, const void* W, const float* bias, int n_out,
                    float* out, cudaStream_t stream);

// NMS / Soft-NMS (raf_nms.cu).
size_t nms_workspace_bytes(int n);
int launch_nms(const float* boxes, const float* scores, int n, float iou_threshold, int32_t* keep, int32_t* num_keep,
               void* ws, cudaStream_t stream);
int launch_soft_nms(const float* boxes, const float* scores, int n, float iou_threshold, float sigma, float min_score,
                    int method, int32_t* keep, float* new_scores, int32_t* num_keep, void* ws, cudaStream_t stream);

// Batched transpose src[batch][R][S] -> dst[batch][S][R] (raf_repack.cu): the NCHW <-> channels-last repack.
int launch_transpose(const void* src, void* dst, int64_t batch, int R, int S, size_t esz, cudaStream_t stream);

// Zero-fill of one strided level (used when the level is not one dense block).
int launch_zero_level(float* data, int n, int c, int h, int w, int64_t sn, int64_t sc, int64_t sh,
                      int64_t sw, cudaStream_t stream);

}  // namespace raf
