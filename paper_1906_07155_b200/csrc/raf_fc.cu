// raf_fc.cu -- the RoIAlign gather fused into the box head's first fully connected layer (
// RoIHead / BBoxHead "2fc"): out[k, n] = sum_{ph,pw,c} A[k,(ph,pw,c)] * W[n,(ph,pw,c)] (+ bias),
// A = the RoIAlign features of RoI k rounded to the feature dtype (readings F1-F3).  The [K, PH*PW*C]
// feature tensor never goes to HBM: it is produced tile by tile straight into the A operand of a tcgen05 GEMM.
//
// CTA = (128 RoIs) x (512 outputs) x (one bin row ph: split-K, fp32 `red` into out), 1024 threads.  Per k-step = (bin pw, 64 channels):
//   * the threads gather the A tile: thread (RoI r, 16-byte chunk j) evaluates the bin's merged separable taps (same
//     tables and FMA order as raf_forward.cu, so the value is bit-identical to the stand-alone forward), rounds to the
//     feature dtype and stores 16 bytes into shared memory in the K-major 128-byte-swizzled UMMA layout
//     (row r at r * 128 B, chunk j at (j ^ (r & 7)) * 16 B: eight lanes write one row, conflict-free);
//   * the same threads copy the W tile [512 x 64] (K-major in memory: W is [N_out, PH*PW*C] row-major) the same way;
//   * fence.proxy.async + barrier, then ONE thread issues eight tcgen05.mma (M 128, N 256, K 16; two N halves; bf16/fp16 in,
//     fp32 accumulate in all 512 columns of tensor memory) and commits them to an mbarrier; shared memory is double-buffered,
//     so the gather of step i+1 overlaps the MMAs of step i;
//   * epilogue: tcgen05.ld (32 lanes x 8 columns per warp and step), bias added by the ph == 0 split, red.global.add.
// Cost model: the 512-column accumulator means every RoI window is gathered N_out / 512 times; this
// kernel exists to be correct and measured, not yet to beat forward + library GEMM.
#include "raf_device.cuh"
#include "raf_host.h"
#include "raf_taps.cuh"

namespace raf {

constexpr int kFcM = 128, kFcN = 512, kFcK = 64;   // CTA tile: 128 RoIs x 512 outputs (all 512 tensor-memory columns)
constexpr int kFcUmmaN = 256;                      // N of one tcgen05.mma (two per k-slice)
constexpr int kFcThreads = 1024;                   // one (RoI, 16-byte chunk) gather unit per thread and k-step

__device__ __forceinline__ uint32_t fc_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// K-major, SWIZZLE_128B shared-memory matrix descriptor (sm_100 UMMA): start address >> 4 in bits [0,14), leading
// byte offset >> 4 in [16,30) (unused for swizzled K-major: 1), stride byte offset >> 4 in [32,46) (8 rows x 128 B),
// descriptor version 1 in [46,48), layout type 2 (128-byte swizzle) in [61,64).
__device__ __forceinline__ uint64_t fc_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(1024 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}

__device__ __forceinline__ void fc_mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(fc_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fc_mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "FC_WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra FC_WAIT_DONE;\n\t"
      "bra FC_WAIT_LOOP;\n\t"
      "FC_WAIT_DONE:\n\t}" ::"r"(fc_smem_u32(bar)), "r"(parity) : "memory");
}

template <typename T> struct FcFmt;
template <> struct FcFmt<__half> { static constexpr uint32_t kFmt = 0; };          // UMMA F16
template <> struct FcFmt<__nv_bfloat16> { static constexpr uint32_t kFmt = 1; };   // UMMA BF16

template <typename T>
__global__ void __launch_bounds__(kFcThreads, 1)
fc_fused_kernel(const LevelsParam lv, const RoiArgs a, const T* __restrict__ W, const float* __restrict__ bias, int n_out,
                float* __restrict__ out) {
  using V = Vec16<T>;   // 8 elements per 16 bytes
  extern __shared__ __align__(1024) unsigned char fc_smem[];
  unsigned char* sA = fc_smem;                              // 2 stages x 128 rows x 128 B
  unsigned char* sB = fc_smem + 2 * kFcM * 128;             // 2 stages x 256 rows x 128 B
  __shared__ uint64_t mma_done[2];
  __shared__ uint32_t tmem_base_s;
  __shared__ const T* s_base[kFcM];                         // feature pointer of the RoI's (level, image)
  __shared__ FwdTap s_ty[kFcM][4], s_tx[kFcM][4];           // merged taps of the current bin (row taps: once per CTA)
  __shared__ unsigned char s_ny[kFcM], s_nx[kFcM];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int m0 = blockIdx.x * kFcM, n0 = blockIdx.y * kFcN, ph = blockIdx.z;
  const int PH = a.PH, PW = a.PW, C = lv.c, g = a.sampling_ratio;
  const int64_t Kd = (int64_t)PH * PW * C;

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(fc_smem_u32(&tmem_base_s)), "n"(kFcN));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 32) {
    fc_mbar_init(&mma_done[0], 1);
    fc_mbar_init(&mma_done[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;");
  }
  // per-RoI set-up: level, image, row taps of bin row ph (1 / count folded in, as the forward does)
  RoiGeom geo{};
  int level = 0;
  bool live = false;
  if (tid < kFcM) {
    const int k = m0 + tid;
    int ny = 0;
    const T* base = nullptr;
    if (k < a.K) {
      const float* r = a.rois + 5 * (int64_t)k;
      const float r0 = __ldg(r), x1 = __ldg(r + 1), y1 = __ldg(r + 2), x2 = __ldg(r + 3), y2 = __ldg(r + 4);
      level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);
      const int b = batch_index_of(r0, lv.n);
      if (b >= 0) {
        live = true;
        geo = roi_geom(x1, y1, x2, y2, lv.scale[level], PH, PW, g, a.aligned);
        base = reinterpret_cast<const T*>(lv.data[level]) + (int64_t)b * lv.sn[level];
        ny = fwd_bin_taps(geo.sy, geo.bh, ph, g, lv.h[level], (int)lv.sh[level], geo.inv_count, s_ty[tid]);
      }
    }
    s_base[tid] = base;
    s_ny[tid] = (unsigned char)ny;
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tmem = tmem_base_s;
  const uint32_t idesc = (1u << 4) | (FcFmt<T>::kFmt << 7) | (FcFmt<T>::kFmt << 10) | ((uint32_t)(kFcUmmaN >> 3) << 17) |
                         ((uint32_t)(kFcM >> 4) << 24);

  const int cchunks = C / kFcK;
  uint32_t phase[2] = {0, 0};
  int step = 0;
  for (int pw = 0; pw < PW; ++pw) {
    // column taps of bin pw for every RoI of the tile (previous readers are past the barrier of their k-step)
    if (tid < kFcM) {
      int nx = 0;
      if (live) nx = fwd_bin_taps(geo.sx, geo.bw, pw, g, lv.w[level], (int)lv.sw[level], 1.0f, s_tx[tid]);
      s_nx[tid] = (unsigned char)nx;
    }
    __syncthreads();
    for (int cc = 0; cc < cchunks; ++cc, ++step) {
      const int st = step & 1;
      if (step >= 2) { fc_mbar_wait(&mma_done[st], phase[st]); phase[st] ^= 1; }   // the MMAs that read this stage are done
      unsigned char* At = sA + st * kFcM * 128;
      unsigned char* Bt = sB + st * kFcN * 128;
      // ---- W tile first (its loads fly while the A tile is gathered): W[n0 + n][(ph * PW + pw) * C + cc * 64 + j * 8 ...] ---
      const int j = tid & 7;
      const int64_t kidx = ((int64_t)ph * PW + pw) * C + cc * kFcK + j * 8;
      uint4 wv[kFcN * 8 / kFcThreads];
#pragma unroll
      for (int i = 0; i < kFcN * 8 / kFcThreads; ++i) {
        const int n = (tid >> 3) + (kFcThreads / 8) * i;
        wv[i] = __ldg(reinterpret_cast<const uint4*>(W + (int64_t)(n0 + n) * Kd + kidx));
      }
      // ---- A tile: thread = (RoI row r, 16-byte chunk j); eight lanes cover the 64 channels of one RoI -----------
#pragma unroll 1
      for (int i = 0; i < kFcM * 8 / kFcThreads; ++i) {
        const int r = (tid >> 3) + (kFcThreads / 8) * i;
        float acc[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[q] = 0.0f;
        const T* base = s_base[r];
        const int ny = s_ny[r], nx = s_nx[r];
        if (base != nullptr) {
          const T* p0 = base + cc * kFcK + j * 8;
          const FwdTap* ty = s_ty[r];
          const FwdTap* tx = s_tx[r];
          // the loads of two tap rows (<= 8) are issued before their FMAs: memory-level parallelism is what bounds the
          // gather (1024 threads x 8 loads x 16 B = 128 KB in flight per SM at 64 registers per thread)
#pragma unroll
          for (int y0 = 0; y0 < 4; y0 += 2) {
            if (y0 < ny) {
              uint4 raw[2][4];
#pragma unroll
              for (int ya = 0; ya < 2; ++ya)
#pragma unroll
                for (int xb = 0; xb < 4; ++xb)
                  if (y0 + ya < ny && xb < nx) raw[ya][xb] = V::load_raw(p0 + ty[y0 + ya].off + tx[xb].off);
#pragma unroll
              for (int ya = 0; ya < 2; ++ya)
#pragma unroll
                for (int xb = 0; xb < 4; ++xb)
                  if (y0 + ya < ny && xb < nx) {
                    float v[8];
                    V::widen(raw[ya][xb], v);
                    const float w = ty[y0 + ya].w * tx[xb].w;
#pragma unroll
                    for (int q = 0; q < 8; ++q) acc[q] = fmaf(w, v[q], acc[q]);
                  }
            }
          }
        }
        uint4 packed;
        {
          T tmp[8];
#pragma unroll
          for (int q = 0; q < 8; ++q) tmp[q] = Elem<T>::from_f32(acc[q]);
          packed = *reinterpret_cast<const uint4*>(tmp);
        }
        *reinterpret_cast<uint4*>(At + r * 128 + ((j ^ (r & 7)) << 4)) = packed;
      }
#pragma unroll
      for (int i = 0; i < kFcN * 8 / kFcThreads; ++i) {
        const int n = (tid >> 3) + (kFcThreads / 8) * i;
        *reinterpret_cast<uint4*>(Bt + n * 128 + ((j ^ (n & 7)) << 4)) = wv[i];
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the tensor core
      __syncthreads();
      if (tid == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;");
#pragma unroll
        for (int s = 0; s < kFcK / 16; ++s) {
          const uint64_t ad = fc_desc(fc_smem_u32(At) + s * 32);
          const uint32_t accf = (step > 0 || s > 0) ? 1u : 0u;
#pragma unroll
          for (int h = 0; h < kFcN / kFcUmmaN; ++h) {   // N halves: rows h*256.. of the W tile -> columns h*256.. of the accumulator
            const uint64_t bd = fc_desc(fc_smem_u32(Bt) + h * kFcUmmaN * 128 + s * 32);
            asm volatile(
                "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem + h * kFcUmmaN), "l"(ad), "l"(bd), "r"(idesc),
                "r"(accf));
          }
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.b64 [%0];" ::"l"(
            (uint64_t)__cvta_generic_to_shared(&mma_done[st])));
      }
    }
    __syncthreads();   // the column taps are rewritten for the next bin
  }
  // ---- epilogue: wait for the last MMAs (the commit of step-1 also covers every earlier one) -------------------
  {
    const int st = (step - 1) & 1;
    fc_mbar_wait(&mma_done[st], phase[st]);
  }
  asm volatile("tcgen05.fence::after_thread_sync;");
  const int row = (warp & 3) * 32 + lane;          // tensor-memory lane = row of the tile (a warp reaches lanes 32 * (warp % 4) ..)
  constexpr int kColsPerWarp = kFcN / (kFcThreads / 128);
  const int col0 = (warp >> 2) * kColsPerWarp;
  const int kroi = m0 + row;
  for (int c = 0; c < kColsPerWarp; c += 8) {
    uint32_t v[8];
    const uint32_t taddr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(col0 + c);
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;");
    if (kroi < a.K) {
      float* o = out + (int64_t)kroi * n_out + n0 + col0 + c;
      float val[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        val[q] = __uint_as_float(v[q]);
        if (ph == 0 && bias != nullptr) val[q] += __ldg(bias + n0 + col0 + c + q);
      }
      red_add_v4(o, val[0], val[1], val[2], val[3]);
      red_add_v4(o + 4, val[4], val[5], val[6], val[7]);
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kFcN));
}

template <typename T>
static int fc_typed(const LevelsParam& lv, const RoiArgs& a, const void* W, const float* bias, int n_out, float* out,
                    cudaStream_t stream) {
  const size_t smem = 2 * (size_t)kFcM * 128 + 2 * (size_t)kFcN * 128 + 1024;
  if (cudaFuncSetAttribute(fc_fused_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return RAF_ERR_CUDA;
  const dim3 grid((unsigned)((a.K + kFcM - 1) / kFcM), (unsigned)(n_out / kFcN), (unsigned)a.PH);
  fc_fused_kernel<T><<<grid, kFcThreads, smem, stream>>>(lv, a, reinterpret_cast<const T*>(W), bias, n_out, out);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

int launch_fc_fused(const LevelsParam& lv, raf_dtype dtype, const RoiArgs& a, const void* W, const float* bias, int n_out,
                    float* out, cudaStream_t stream) {
  switch (dtype) {
    case RAF_F16: return fc_typed<__half>(lv, a, W, bias, n_out, out, stream);
    case RAF_BF16: return fc_typed<__nv_bfloat16>(lv, a, W, bias, n_out, out, stream);
    default: return RAF_ERR_UNSUPPORTED;
  }
}

}  // namespace raf
