// raf_static.cu -- roi_align_fpn_backward_static: the RoIAlign backward for callers
// that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  The backward's scratch -- the prep tables of raf_pull_prep.cuh: fingerprint header, stable
// (level, image) buckets, pixel windows, RoI geometry, tap tables -- lives in a file-scope device array of
// RAF_STATIC_WS_BYTES instead of a caller-supplied workspace.  Every GPU that loads the library holds that array
// until the process exits.  The kernels are the ones roi_align_fpn_backward launches, given the array's address.
//
// In HOST code the name of a __device__ array is a host-side stand-in, not a device address: the address the
// kernels need comes from cudaGetSymbolAddress, asked once per device with that device current, return code checked.
//
// No cudaMalloc / cudaFree / allocating library call on this path.  All calls share the one array, which keeps the
// previous call's contents: the fingerprint header is cleared first (tables of an earlier call can then never pass
// the kernels' fingerprint check), and everything else the backward reads is rewritten by this call's prep launch
// before it is read (same stream).  Calls that overlap on the GPU (different streams, no ordering) race on the array.
#include "../../include/raf.h"
#include <cuda_runtime.h>
#include <cstdint>
#include <mutex>

namespace {

__device__ __align__(256) unsigned char g_static_ws[RAF_STATIC_WS_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_ws_ptr[kMaxDevices] = {};

// Device address of g_static_ws on the CURRENT device (looked up once per device).
int static_ws_address(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return RAF_ERR_CUDA;
  if (dev < 0 || dev >= kMaxDevices) return RAF_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_ws_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_static_ws) != cudaSuccess || !p) return RAF_ERR_CUDA;
    g_ws_ptr[dev] = p;
  }
  *out = g_ws_ptr[dev];
  return RAF_OK;
}

}  // namespace

extern "C" int roi_align_fpn_backward_static(const raf_level* grad_feats, int L, raf_dtype gout_dtype,
                                             const void* grad_out, const int64_t* gout_strides, const float* rois,
                                             int K, int out_h, int out_w, int sampling_ratio, int aligned,
                                             float finest_scale, int flags, void* stream) {
  // The shared array cannot stand in for a workspace another call filled, nor hold the repack copies.
  if (flags & (RAF_REUSE_PREP | RAF_REPACK)) return RAF_ERR_UNSUPPORTED;
  // Size limit, decided on the host before any CUDA call.
  if (roi_align_fpn_workspace_bytes(K, L, out_h, out_w, sampling_ratio, flags) > (size_t)RAF_STATIC_WS_BYTES)
    return RAF_ERR_WORKSPACE;
  void* ws = nullptr;
  int rc = static_ws_address(&ws);
  if (rc) return rc;
  if (cudaMemsetAsync(ws, 0, 256, (cudaStream_t)stream) != cudaSuccess) return RAF_ERR_CUDA;   // fingerprint header
  return roi_align_fpn_backward_ex(grad_feats, L, gout_dtype, RAF_F32, grad_out, gout_strides, rois, K, out_h, out_w,
                                   sampling_ratio, aligned, finest_scale, flags, ws, (size_t)RAF_STATIC_WS_BYTES, stream);
}
