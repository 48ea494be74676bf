// raf_forward.cu -- K2: multi-level RoIAlign forward gather.
//
//   out[k,c,ph,pw] = (1/count) * sum_{iy,ix} bilinear(F_{level_k}[b_k,c], y(ph,iy), x(pw,ix))
//
// Two kernels:
//  * fwd_cl_kernel   channels-last fast path: one CTA per (RoI, 32 channel-vectors).  The RoI's
//                    level, image and its per-axis TAP tables are staged in shared memory: the g
//                    samples of a bin give up to 2g (pixel, weight) taps per axis, equal pixels
//                    merged, computed ONCE per RoI and reused by every channel (north_star).  The
//                    operator is separable, so a bin is sum_{y taps} sum_{x taps} wy*wx*F[y][x]:
//                    typically 3x3 loads instead of 4 samples x 4 taps.  A warp owns an output bin
//                    row (its y taps and row pointers stay in registers) and walks the bins of the
//                    row; lanes = channel vectors: each 128-bit load covers 4 fp32 / 8 half
//                    channels of one tap, a warp reads 512 contiguous bytes.
//  * fwd_generic_kernel  any strides / any C / adaptive sampling: one thread per output element.
#include "raf_device.cuh"
#include "raf_host.h"
#include "raf_pull_prep.cuh"
#include "raf_taps.cuh"
#include <cstdlib>

namespace raf {

#ifndef RAF_FWD_MINB
#define RAF_FWD_MINB 3
#endif
constexpr int kFwdWarps = 8;   // max warps per CTA (one output bin row each, strided)
constexpr int kFwdAdaptGrid = 8;   // adaptive sampling: grids up to 8 per axis are tabulated (16 tap slots per bin)

// acc += sum_{a < NY, b < NX} (yw[a] * xw[b]) * F[rp[a] + xo[b]]: all NY*NX loads are issued before
// the first use (memory-level parallelism is what bounds this kernel).
template <typename T, int NY, int NX>
__device__ __forceinline__ void fwd_accumulate(const T* rp0, const T* rp1, const T* rp2, const T* rp3,
                                               const float (&yw)[4], const int (&xo)[4],
                                               const float (&xw)[4], float (&acc)[Vec16<T>::N]) {
  constexpr int VN = Vec16<T>::N;
  const T* rp[4] = {rp0, rp1, rp2, rp3};
  float v[NY][NX][VN];
#pragma unroll
  for (int a = 0; a < NY; ++a)
#pragma unroll
    for (int b = 0; b < NX; ++b) Vec16<T>::load(rp[a] + xo[b], v[a][b]);
#pragma unroll
  for (int a = 0; a < NY; ++a)
#pragma unroll
    for (int b = 0; b < NX; ++b) {
      const float w = yw[a] * xw[b];
#ifndef RAF_NO_FFMA2
      const float2 ww = make_float2(w, w);   // packed fp32x2 FMAs (sm_100): one issue slot per two channels
#pragma unroll
      for (int j = 0; j < VN; j += 2) {
        const float2 r = __ffma2_rn(ww, make_float2(v[a][b][j], v[a][b][j + 1]), make_float2(acc[j], acc[j + 1]));
        acc[j] = r.x; acc[j + 1] = r.y;
      }
#else
#pragma unroll
      for (int j = 0; j < VN; ++j) acc[j] = fmaf(w, v[a][b][j], acc[j]);
#endif
    }
}

template <typename T, int NY>
__device__ __forceinline__ void fwd_dispatch_x(int nx, const T* rp0, const T* rp1, const T* rp2, const T* rp3,
                                               const float (&yw)[4], const int (&xo)[4], const float (&xw)[4],
                                               float (&acc)[Vec16<T>::N]) {
  switch (nx) {
    case 1: fwd_accumulate<T, NY, 1>(rp0, rp1, rp2, rp3, yw, xo, xw, acc); break;
    case 2: fwd_accumulate<T, NY, 2>(rp0, rp1, rp2, rp3, yw, xo, xw, acc); break;
    case 3: fwd_accumulate<T, NY, 3>(rp0, rp1, rp2, rp3, yw, xo, xw, acc); break;
    default: fwd_accumulate<T, NY, 4>(rp0, rp1, rp2, rp3, yw, xo, xw, acc); break;
  }
}

// Adaptive grids beyond the tables: one warp per bin row, lanes = channel vectors, every sample evaluated as C3
// writes it (rare: bins wider than kFwdAdaptGrid pixels).
template <typename T>
__device__ __noinline__ void fwd_direct_rows(const RoiGeom geo, const T* base, T* out_k, int b, int H, int W, int sh, int sw,
                                             int PW, int ph0, int rend, int nwarps, int64_t os_h, int64_t os_w) {
  using V = Vec16<T>;
  constexpr int VN = V::N;
  for (int ph = ph0; ph < rend; ph += nwarps) {
    for (int pw = 0; pw < PW; ++pw) {
      float acc[VN];
#pragma unroll
      for (int j = 0; j < VN; ++j) acc[j] = 0.0f;
      if (b >= 0) {
        for (int iy = 0; iy < geo.gh; ++iy) {
          const AxisTap ty = axis_tap(sample_coord(geo.sy, geo.bh, ph, iy, geo.gh), H);
          if (!ty.valid) continue;
          for (int ix = 0; ix < geo.gw; ++ix) {
            const AxisTap tx = axis_tap(sample_coord(geo.sx, geo.bw, pw, ix, geo.gw), W);
            if (!tx.valid) continue;
            const float w4[4] = {ty.wh * tx.wh, ty.wh * tx.wl, ty.wl * tx.wh, ty.wl * tx.wl};
            const int o4[4] = {ty.lo * sh + tx.lo * sw, ty.lo * sh + tx.hi * sw, ty.hi * sh + tx.lo * sw, ty.hi * sh + tx.hi * sw};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              float v[VN];
              V::load(base + o4[q], v);
#pragma unroll
              for (int j = 0; j < VN; ++j) acc[j] = fmaf(w4[q], v[j], acc[j]);
            }
          }
        }
#pragma unroll
        for (int j = 0; j < VN; ++j) acc[j] *= geo.inv_count;
      }
      V::store(out_k + ph * os_h + pw * os_w, acc);
    }
  }
}

// Channels-last forward.  CTA = (RoI, chunk of 32 channel-vectors); warp = output bin row(s);
// lanes = channel vectors (16 bytes each: a warp-wide load covers 512 contiguous bytes).
#ifndef RAF_FWD_MINB7
#define RAF_FWD_MINB7 4
#endif
// kThreads = 224 (7 warps: 7-row outputs, the common case) or 256: the register budget follows the real block size.
// A RoI's bin rows are split over `rsplit` CTAs (rows_per rows each) when there are more rows than warps.
// The struct parameters are __grid_constant__: `lv` is indexed by the RoI's level, and without the qualifier every
// thread first copies the arrays to its local memory (96-112 bytes of stack, 12 STL.64 in the prologue, LDL in the body);
// with it the indexed reads come straight from the constant bank (config 2 forward 62.4 -> 55.8 us, config 3 37.3 -> 36.0 us,
// config 5 198.2 -> 193.8 us).  The tile backward does NOT take the same change: its fp32 instantiation gets slower
// (85.8 -> 90.3 us), profiles/r2_experiments.md.
template <typename T, int kThreads>
__global__ void __launch_bounds__(kThreads, kThreads == 224 ? RAF_FWD_MINB7 : (kThreads == 128 ? 7 : RAF_FWD_MINB))
fwd_cl_kernel(const __grid_constant__ LevelsParam lv, const __grid_constant__ RoiArgs a, T* __restrict__ out, int64_t os_k, int64_t os_h,
              int64_t os_w, int chunks, int rsplit, int rows_per, const __grid_constant__ PullPrepOut prep) {
  using V = Vec16<T>;
  constexpr int VN = V::N;
  extern __shared__ __align__(16) unsigned char fwd_smem[];
  // sampling_ratio == 0 (adaptive grid, reading S7): the grid is per RoI, gh = ceil(bin height), gw likewise;
  // the tables take grids up to kFwdAdaptGrid per axis, larger ones (bins wider than 8 pixels: boxes far
  // beyond what the level map assigns) are sampled directly
  const int g = a.sampling_ratio, slots = g > 0 ? 2 * g : 2 * kFwdAdaptGrid;
  const int PH = a.PH, PW = a.PW, nb = PH + PW;
  FwdTap* s_tab = reinterpret_cast<FwdTap*>(fwd_smem);          // [PH + PW][slots]; y bins first
  int* s_cnt = reinterpret_cast<int*>(s_tab + nb * slots);     // [PH + PW]
  __shared__ int s_b;

  // The backward's prep rides in this launch (same RoIs, same geometry): block 0 buckets the RoIs (a
  // serial chain, so it starts first), the blocks after the forward's own write the tap tables
  // (independent items: they fill the tail of the grid).
  const int nfwd = a.K * chunks * rsplit;
  if (prep.nblocks > 0 && ((int)blockIdx.x == 0 || (int)blockIdx.x > nfwd)) {
    pull_prep_block(lv, a, prep, (int)blockIdx.x == 0 ? 0 : (int)blockIdx.x - nfwd, reinterpret_cast<int*>(fwd_smem));
    return;
  }
  const int bid = (int)blockIdx.x - (prep.nblocks > 0 ? 1 : 0);
  const int part = bid % rsplit, kc = bid / rsplit;
  const int k = kc / chunks, chunk = kc - k * chunks;
  const int rbeg = part * rows_per, rend = min(PH, rbeg + rows_per);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  const float* r = a.rois + 5 * (int64_t)k;
  const float r0 = __ldg(r), x1 = __ldg(r + 1), y1 = __ldg(r + 2), x2 = __ldg(r + 3), y2 = __ldg(r + 4);
  const int level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);

  RoiGeom geo{};
  if (g == 0 || (int)threadIdx.x < nb) geo = roi_geom(x1, y1, x2, y2, lv.scale[level], PH, PW, g, a.aligned);
  const bool direct = g == 0 && (geo.gh > kFwdAdaptGrid || geo.gw > kFwdAdaptGrid);   // (uniform over the CTA)
  if ((int)threadIdx.x < nb) {
    const int t = threadIdx.x;
    const bool isy = t < PH;
    if (!direct)
      s_cnt[t] = isy ? fwd_bin_taps(geo.sy, geo.bh, t, geo.gh, lv.h[level], (int)lv.sh[level], geo.inv_count, s_tab + t * slots)
                     : fwd_bin_taps(geo.sx, geo.bw, t - PH, geo.gw, lv.w[level], (int)lv.sw[level], 1.0f, s_tab + t * slots);
    if (t == 0) s_b = batch_index_of(r0, lv.n);
  }
  __syncthreads();

  const int b = s_b;
  const int cv = chunk * 32 + lane;
  if (cv * VN >= lv.c) return;
  T* out_k = out + (int64_t)k * os_k + cv * VN;
  const T* base = reinterpret_cast<const T*>(lv.data[level]) + (int64_t)(b >= 0 ? b : 0) * lv.sn[level] + cv * VN;

  if (direct) {   // rare: sample by sample (C3 as written); kept out of line so that it costs the hot path no registers
    fwd_direct_rows<T>(geo, base, out_k, b, lv.h[level], lv.w[level], (int)lv.sh[level], (int)lv.sw[level], PW, rbeg + warp,
                       rend, nwarps, os_h, os_w);
    return;
  }

  for (int ph = rbeg + warp; ph < rend; ph += nwarps) {
    const int ny = (b >= 0) ? s_cnt[ph] : 0;
    const FwdTap* ty = s_tab + ph * slots;
    float yw[4];
    int yo[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const FwdTap e = (q < slots) ? ty[q] : FwdTap{0, 0.f};
      yo[q] = e.off;
      yw[q] = e.w;
    }
    const T* rp0 = base + yo[0];
    const T* rp1 = base + yo[1];
    const T* rp2 = base + yo[2];
    const T* rp3 = base + yo[3];
    for (int pw = 0; pw < PW; ++pw) {
      const int nx = s_cnt[PH + pw];
      const FwdTap* tx = s_tab + (PH + pw) * slots;
      float acc[VN];
#pragma unroll
      for (int j = 0; j < VN; ++j) acc[j] = 0.0f;
      if (ny > 0 && nx > 0) {
        if (ny <= 4 && nx <= 4) {
          int xo[4];
          float xw[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const FwdTap e = (q < slots) ? tx[q] : FwdTap{0, 0.f};
            xo[q] = e.off;
            xw[q] = e.w;
          }
          switch (ny) {
            case 1: fwd_dispatch_x<T, 1>(nx, rp0, rp1, rp2, rp3, yw, xo, xw, acc); break;
            case 2: fwd_dispatch_x<T, 2>(nx, rp0, rp1, rp2, rp3, yw, xo, xw, acc); break;
            case 3: fwd_dispatch_x<T, 3>(nx, rp0, rp1, rp2, rp3, yw, xo, xw, acc); break;
            default: fwd_dispatch_x<T, 4>(nx, rp0, rp1, rp2, rp3, yw, xo, xw, acc); break;
          }
        } else {   // sampling_ratio > 2: walk the tap lists
          for (int qa = 0; qa < ny; ++qa) {
            const FwdTap ey = ty[qa];
            for (int qb = 0; qb < nx; ++qb) {
              const FwdTap ex = tx[qb];
              float v[VN];
              V::load(base + ey.off + ex.off, v);
              const float w = ey.w * ex.w;
#pragma unroll
              for (int j = 0; j < VN; ++j) acc[j] = fmaf(w, v[j], acc[j]);
            }
          }
        }
      }
      V::store(out_k + ph * os_h + pw * os_w, acc);
    }
  }
}

template <typename T>
__global__ void __launch_bounds__(256)
fwd_generic_kernel(const LevelsParam lv, const RoiArgs a, T* __restrict__ out, int64_t os_k,
                   int64_t os_c, int64_t os_h, int64_t os_w, int64_t total) {
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int pw = (int)(idx % a.PW);
    const int ph = (int)((idx / a.PW) % a.PH);
    const int c = (int)((idx / ((int64_t)a.PW * a.PH)) % lv.c);
    const int k = (int)(idx / ((int64_t)a.PW * a.PH * lv.c));
    const float* r = a.rois + 5 * (int64_t)k;
    const float x1 = r[1], y1 = r[2], x2 = r[3], y2 = r[4];
    const int level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);
    const int b = batch_index_of(r[0], lv.n);
    float acc = 0.0f;
    if (b >= 0) {
      const RoiGeom geo = roi_geom(x1, y1, x2, y2, lv.scale[level], a.PH, a.PW, a.sampling_ratio, a.aligned);
      const int H = lv.h[level], W = lv.w[level];
      const int64_t sh = lv.sh[level], sw = lv.sw[level];
      const T* F = reinterpret_cast<const T*>(lv.data[level]) + b * lv.sn[level] + c * lv.sc[level];
      for (int iy = 0; iy < geo.gh; ++iy) {
        const AxisTap ty = axis_tap(sample_coord(geo.sy, geo.bh, ph, iy, geo.gh), H);
        if (!ty.valid) continue;
        for (int ix = 0; ix < geo.gw; ++ix) {
          const AxisTap tx = axis_tap(sample_coord(geo.sx, geo.bw, pw, ix, geo.gw), W);
          if (!tx.valid) continue;
          const float w1 = __fmul_rn(ty.wh, tx.wh), w2 = __fmul_rn(ty.wh, tx.wl);
          const float w3 = __fmul_rn(ty.wl, tx.wh), w4 = __fmul_rn(ty.wl, tx.wl);
          acc += w1 * Elem<T>::to_f32(F[ty.lo * sh + tx.lo * sw]) + w2 * Elem<T>::to_f32(F[ty.lo * sh + tx.hi * sw]) +
                 w3 * Elem<T>::to_f32(F[ty.hi * sh + tx.lo * sw]) + w4 * Elem<T>::to_f32(F[ty.hi * sh + tx.hi * sw]);
        }
      }
      acc *= geo.inv_count;
    }
    out[k * os_k + c * os_c + ph * os_h + pw * os_w] = Elem<T>::from_f32(acc);
  }
}

template <typename T>
static int forward_typed(const LevelsParam& lv, const RoiArgs& a, void* out, const int64_t* os,
                         bool channels_last, const PullPrepOut* prep, cudaStream_t stream) {
  T* o = reinterpret_cast<T*>(out);
  const int g = a.sampling_ratio;
  if (channels_last) {
    const int CV = lv.c / Vec16<T>::N;
    const int chunks = (CV + 31) / 32;
    size_t smem = (size_t)(a.PH + a.PW) * (2 * (g > 0 ? g : kFwdAdaptGrid) * sizeof(FwdTap) + sizeof(int));
    // one warp per bin row: outputs taller than 8 rows are split over several CTAs of equal height
    // (14 rows: 2 x 7 warps -- measured 33.7 us vs 43.4 us for one CTA of 8 warps on config 4; splitting
    // 7-row outputs into 4 + 3 rows is slower: 43.4 us vs 39.6 us on config 3)
    int rsplit = (a.PH + kFwdWarps - 1) / kFwdWarps;
#ifdef RAF_EXPERIMENT
    if (const char* e = getenv("RAF_TUNE_RSPLIT")) rsplit = atoi(e);
#endif
    const int rows_per = (a.PH + rsplit - 1) / rsplit;
    int nw = rows_per < kFwdWarps ? rows_per : kFwdWarps;   // one warp per output bin row
    while (32 * nw < a.PH + a.PW) ++nw;                     // the table set-up needs PH + PW threads
    PullPrepOut po{};
    if (prep) {                                             // carry the backward's prep in extra blocks
      po = *prep;
      po.nblocks = pull_prep_blocks(a, 32 * nw);
      const size_t psmem = (size_t)(nw + 1) * ((size_t)lv.L * lv.n + 1) * sizeof(int);
      if (psmem > smem) smem = psmem;
    }
    const unsigned grid = (unsigned)((int64_t)a.K * chunks * rsplit + po.nblocks);
    if (nw == 7) {
      if (smem > 48 * 1024 &&
          cudaFuncSetAttribute(fwd_cl_kernel<T, 224>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return RAF_ERR_CUDA;
      fwd_cl_kernel<T, 224><<<grid, 224, smem, stream>>>(lv, a, o, os[0], os[2], os[3], chunks, rsplit, rows_per, po);
    } else if (nw <= 4) {
      if (smem > 48 * 1024 &&
          cudaFuncSetAttribute(fwd_cl_kernel<T, 128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return RAF_ERR_CUDA;
      fwd_cl_kernel<T, 128><<<grid, 32 * nw, smem, stream>>>(lv, a, o, os[0], os[2], os[3], chunks, rsplit, rows_per, po);
    } else {
      if (smem > 48 * 1024 &&
          cudaFuncSetAttribute(fwd_cl_kernel<T, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return RAF_ERR_CUDA;
      fwd_cl_kernel<T, 256><<<grid, 32 * nw, smem, stream>>>(lv, a, o, os[0], os[2], os[3], chunks, rsplit, rows_per, po);
    }
  } else {
    if (prep) {   // generic path: the prep tables still get written, by their own launch
      const int rc = launch_pull_prep(lv, a, *prep, stream);
      if (rc) return rc;
    }
    const int64_t total = (int64_t)a.K * lv.c * a.PH * a.PW;
    const int64_t blocks = (total + 255) / 256;
    const int grid = (int)(blocks < (int64_t)148 * 64 ? blocks : (int64_t)148 * 64);
    fwd_generic_kernel<T><<<grid, 256, 0, stream>>>(lv, a, o, os[0], os[1], os[2], os[3], total);
  }
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

int launch_forward(const LevelsParam& lv, raf_dtype dtype, const RoiArgs& a, void* out,
                   const int64_t* out_strides, bool channels_last, const PullPrepOut* prep, cudaStream_t stream) {
  switch (dtype) {
    case RAF_F32: return forward_typed<float>(lv, a, out, out_strides, channels_last, prep, stream);
    case RAF_F16: return forward_typed<__half>(lv, a, out, out_strides, channels_last, prep, stream);
    case RAF_BF16: return forward_typed<__nv_bfloat16>(lv, a, out, out_strides, channels_last, prep, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
