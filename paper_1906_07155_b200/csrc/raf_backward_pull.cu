// raf_backward_pull.cu -- K3d: deterministic PULL formulation of the RoIAlign backward
// (reading S12; H5: the backward's bytes are the gradient pyramid).
//
// Instead of scattering every tap with atomics into a zero-filled pyramid, every CTA OWNS a tile of
// the gradient pyramid -- (image n, level l, rows y0..y0+RY-1, columns x0..x0+15, all channels) --
// sums everything that lands in it in registers, and writes each element exactly once (zero where
// nothing lands).  No memset, no atomics, every fp32 gradient element written once = the
// algorithmic byte count; the summation order is fixed (RoIs of the tile's (level, image) bucket in
// ascending k, bins in ascending order), so two runs give identical bits.
//
// The operator is separable.  For RoI k, row y, column x:
//   g[y][x] += sum_ph sum_pw  Wy[y][ph] * Cw[x][pw] * gout[k][ph][pw] / count
//   Wy[y][ph] = sum_iy [lo(ph,iy)==y]*wh + [hi(ph,iy)==y]*wl      (same taps / weights as forward)
// so a thread (row, 4 channels) first forms T[pw] = sum_ph Wy*gout (gout read once per needed bin),
// parks T in a thread-private shared-memory column, and then accumulates its 16 columns
// acc[j] += sum_pw Cw[x0+j][pw] * T[pw] in registers (static indices).
//
// Per tile: (A) scan the bucket, keep the RoIs whose window meets the tile (ballot compaction, order
// preserved); (B) for batches of 8 candidates build the sample tables and the tile-local Wy / Cw
// weights cooperatively in shared memory; (C) consume.  Tiles of the coarsest level are scheduled
// first (most RoIs per pixel).
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

constexpr int kPullThreads = 256;
constexpr int kTW = 16;   // tile columns (register accumulators per thread)
constexpr int kNB = 8;    // RoIs per batch

struct PullTiles {
  int32_t order[kMaxLevels];      // level processed at position i (coarsest first)
  int32_t start[kMaxLevels + 1];  // first block of position i
  int32_t tiles_y[kMaxLevels], tiles_x[kMaxLevels];
  int32_t RY, TPR, chunks;        // rows per tile, threads per row, channel chunks
};

struct PullEntry {  // one bilinear sample along one axis
  int lo, hi;
  float wl, wh;
};

template <typename T> __device__ __forceinline__ float4 load_gout4(const T* p);
template <> __device__ __forceinline__ float4 load_gout4<float>(const float* p) {
  return __ldg(reinterpret_cast<const float4*>(p));
}
template <> __device__ __forceinline__ float4 load_gout4<__half>(const __half* p) {
  const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
  const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
  return make_float4(a.x, a.y, b.x, b.y);
}
template <> __device__ __forceinline__ float4 load_gout4<__nv_bfloat16>(const __nv_bfloat16* p) {
  const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
  return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u),
                     __uint_as_float(r.y << 16), __uint_as_float(r.y & 0xffff0000u));
}

// Shared-memory carve-up (dynamic): sizes depend on PH, PW, g, RY.
struct PullSmem {
  int* cand;          // [kPullThreads] candidate RoI indices of the current scan chunk
  int* wcount;        // [8] per-warp candidate counts
  PullEntry* tab;     // [kNB][ny + nx]
  int* meta_k;        // [kNB] RoI index
  float* meta_ic;     // [kNB] 1 / count
  int* nph;           // [kNB][RY] number of (ph, w) pairs of the row
  unsigned char* ph_idx;  // [kNB][RY][PH]
  float* ph_w;        // [kNB][RY][PH]  (already divided by count)
  float* cw;          // [kNB][kTW][PW]
  signed char* cpa;   // [kNB][kTW] first / last pw with a non-zero weight (pa > pb: none)
  signed char* cpb;
  int* pwlo;          // [kNB] pw range the tile's columns need
  int* pwhi;
  float4* T;          // [PW][kPullThreads]
};

__host__ __device__ inline size_t pull_align16(size_t v) { return (v + 15) & ~(size_t)15; }

__host__ __device__ inline size_t pull_smem_layout(int PH, int PW, int g, int RY, PullSmem* s, char* base) {
  size_t o = 0;
  auto take = [&](size_t bytes) { const size_t at = o; o = pull_align16(o + bytes); return base + at; };
  const int ns = (PH + PW) * g;
  char* p;
  p = take(sizeof(int) * kPullThreads); if (s) s->cand = (int*)p;
  p = take(sizeof(int) * 8); if (s) s->wcount = (int*)p;
  p = take(sizeof(PullEntry) * kNB * ns); if (s) s->tab = (PullEntry*)p;
  p = take(sizeof(int) * kNB); if (s) s->meta_k = (int*)p;
  p = take(sizeof(float) * kNB); if (s) s->meta_ic = (float*)p;
  p = take(sizeof(int) * kNB * RY); if (s) s->nph = (int*)p;
  p = take((size_t)kNB * RY * PH); if (s) s->ph_idx = (unsigned char*)p;
  p = take(sizeof(float) * kNB * RY * PH); if (s) s->ph_w = (float*)p;
  p = take(sizeof(float) * kNB * kTW * PW); if (s) s->cw = (float*)p;
  p = take((size_t)kNB * kTW); if (s) s->cpa = (signed char*)p;
  p = take((size_t)kNB * kTW); if (s) s->cpb = (signed char*)p;
  p = take(sizeof(int) * kNB); if (s) s->pwlo = (int*)p;
  p = take(sizeof(int) * kNB); if (s) s->pwhi = (int*)p;
  p = take(sizeof(float4) * (size_t)PW * kPullThreads); if (s) s->T = (float4*)p;
  return o;
}

template <typename T>
__global__ void __launch_bounds__(kPullThreads, 2)
bwd_pull_kernel(const LevelsParam lv, const RoiArgs a, const T* __restrict__ gout, int64_t gs_k,
                int64_t gs_h, int64_t gs_w, const int32_t* __restrict__ bperm,
                const int32_t* __restrict__ boff, const PullTiles tiles, int accumulate) {
  extern __shared__ __align__(16) char smem_raw[];
  PullSmem S;
  pull_smem_layout(a.PH, a.PW, a.sampling_ratio, tiles.RY, &S, smem_raw);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int PH = a.PH, PW = a.PW, g = a.sampling_ratio;
  const int ny = PH * g, nx = PW * g, ns = ny + nx;
  const int RY = tiles.RY, TPR = tiles.TPR;

  // ---- decode the tile --------------------------------------------------------------------------
  int pos = 0;
  while (pos + 1 < lv.L && (int)blockIdx.x >= tiles.start[pos + 1]) ++pos;
  const int level = tiles.order[pos];
  int rem = blockIdx.x - tiles.start[pos];
  const int chunk = rem % tiles.chunks; rem /= tiles.chunks;
  const int txi = rem % tiles.tiles_x[level]; rem /= tiles.tiles_x[level];
  const int tyi = rem % tiles.tiles_y[level];
  const int n = rem / tiles.tiles_y[level];
  const int H = lv.h[level], W = lv.w[level];
  const int y0 = tyi * RY, x0 = txi * kTW;
  const int y1 = min(y0 + RY, H) - 1, x1 = min(x0 + kTW, W) - 1;  // inclusive
  const float scale = lv.scale[level];

  const int ty = tid / TPR, tc = tid - ty * TPR;
  const int c4 = (chunk * TPR + tc) * 4;
  const bool live = (c4 < lv.c) && (y0 + ty <= y1);
  float* grow = reinterpret_cast<float*>(const_cast<void*>(lv.data[level])) + (int64_t)n * lv.sn[level] +
                (int64_t)(y0 + ty) * lv.sh[level] + c4;
  const int64_t sw = lv.sw[level];

  float4 acc[kTW];
#pragma unroll
  for (int j = 0; j < kTW; ++j) acc[j] = make_float4(0.f, 0.f, 0.f, 0.f);
  if (accumulate && live) {
#pragma unroll
    for (int j = 0; j < kTW; ++j)
      if (x0 + j <= x1) acc[j] = *reinterpret_cast<const float4*>(grow + (int64_t)(x0 + j) * sw);
  }

  const int key = level * lv.n + n;
  const int bbeg = boff[key], bend = boff[key + 1];

  for (int s0 = bbeg; s0 < bend; s0 += kPullThreads) {
    // ---- (A) candidates of this scan chunk, order preserved ------------------------------------
    bool hit = false;
    int k = -1;
    if (s0 + tid < bend) {
      k = bperm[s0 + tid];
      const float* r = a.rois + 5 * (int64_t)k;
      const RoiGeom geo = roi_geom(__ldg(r + 1), __ldg(r + 2), __ldg(r + 3), __ldg(r + 4), scale, PH, PW, g, a.aligned);
      // conservative window from the first and last sample of each axis (samples are monotone)
      const float ya = sample_coord(geo.sy, geo.bh, 0, 0, g), yb = sample_coord(geo.sy, geo.bh, PH - 1, g - 1, g);
      const float xa = sample_coord(geo.sx, geo.bw, 0, 0, g), xb = sample_coord(geo.sx, geo.bw, PW - 1, g - 1, g);
      // (+-0.01 px slack: interior samples may exceed the end samples by an ulp; a superset is harmless)
      const float ylo = fminf(ya, yb) - 0.01f, yhi = fmaxf(ya, yb) + 0.01f;
      const float xlo = fminf(xa, xb) - 0.01f, xhi = fmaxf(xa, xb) + 0.01f;
      // a sample at v touches pixels floor(v) and floor(v)+1 (after clamping to [0, n-1])
      hit = (ylo <= yhi) && (xlo <= xhi) &&                       // false for NaN
            (yhi >= -1.0f) && (ylo <= (float)H) && (xhi >= -1.0f) && (xlo <= (float)W) &&   // some sample may be valid
            (yhi >= (float)y0 - 1.0f) && (ylo < (float)y1 + 1.0f || y1 == H - 1) &&
            (xhi >= (float)x0 - 1.0f) && (xlo < (float)x1 + 1.0f || x1 == W - 1);
    }
    const unsigned m = __ballot_sync(0xffffffffu, hit);
    if (lane == 0) S.wcount[warp] = __popc(m);
    __syncthreads();
    int before = 0, ncand = 0;
    for (int w = 0; w < kPullThreads / 32; ++w) {
      const int cnt = S.wcount[w];
      if (w < warp) before += cnt;
      ncand += cnt;
    }
    if (hit) S.cand[before + __popc(m & ((1u << lane) - 1u))] = k;
    __syncthreads();

    for (int b0 = 0; b0 < ncand; b0 += kNB) {
      const int nb = min(kNB, ncand - b0);
      // ---- (B1) sample tables of the batch ------------------------------------------------------
      for (int it = tid; it < nb * ns; it += kPullThreads) {
        const int r_ = it / ns, s = it - r_ * ns;
        const int kk = S.cand[b0 + r_];
        const float* r = a.rois + 5 * (int64_t)kk;
        const RoiGeom geo = roi_geom(__ldg(r + 1), __ldg(r + 2), __ldg(r + 3), __ldg(r + 4), scale, PH, PW, g, a.aligned);
        const bool isy = s < ny;
        const int si = isy ? s : s - ny;
        const int p = si / g, i = si - p * g;
        const float v = isy ? sample_coord(geo.sy, geo.bh, p, i, g) : sample_coord(geo.sx, geo.bw, p, i, g);
        const AxisTap t = axis_tap(v, isy ? H : W);
        PullEntry e;
        e.lo = t.valid ? t.lo : -0x40000000;
        e.hi = t.valid ? t.hi : -0x40000000;
        e.wl = t.valid ? t.wl : 0.0f;
        e.wh = t.valid ? t.wh : 0.0f;
        S.tab[r_ * ns + s] = e;
        if (s == 0) { S.meta_k[r_] = kk; S.meta_ic[r_] = geo.inv_count; }
      }
      __syncthreads();
      // ---- (B2) tile-local weights --------------------------------------------------------------
      const int items = nb * (RY + kTW + 1);
      for (int it = tid; it < items; it += kPullThreads) {
        const int r_ = it / (RY + kTW + 1), q = it - r_ * (RY + kTW + 1);
        const PullEntry* ty_tab = S.tab + r_ * ns;
        const PullEntry* tx_tab = ty_tab + ny;
        if (q < RY) {                       // row q: compact list of (ph, Wy/count)
          const int y = y0 + q;
          const float ic = S.meta_ic[r_];
          int cnt = 0;
          for (int ph = 0; ph < PH; ++ph) {
            float w = 0.0f;
            for (int i = 0; i < g; ++i) {
              const PullEntry e = ty_tab[ph * g + i];
              w += (e.lo == y ? e.wh : 0.0f) + (e.hi == y ? e.wl : 0.0f);
            }
            if (w != 0.0f) {
              S.ph_idx[(r_ * RY + q) * PH + cnt] = (unsigned char)ph;
              S.ph_w[(r_ * RY + q) * PH + cnt] = w * ic;
              ++cnt;
            }
          }
          S.nph[r_ * RY + q] = (y <= y1) ? cnt : 0;
        } else if (q < RY + kTW) {          // column j: dense Cw[pw] + its non-zero range
          const int j = q - RY, x = x0 + j;
          int pa = 127, pb = -1;
          for (int pw = 0; pw < PW; ++pw) {
            float w = 0.0f;
            for (int i = 0; i < g; ++i) {
              const PullEntry e = tx_tab[pw * g + i];
              w += (e.lo == x ? e.wh : 0.0f) + (e.hi == x ? e.wl : 0.0f);
            }
            S.cw[(r_ * kTW + j) * PW + pw] = w;
            if (w != 0.0f) { pa = min(pa, pw); pb = pw; }
          }
          if (x > x1) { pa = 127; pb = -1; }
          S.cpa[r_ * kTW + j] = (signed char)pa;
          S.cpb[r_ * kTW + j] = (signed char)pb;
        } else {                            // pw range any tile column needs
          int lo_ = 127, hi_ = -1;
          for (int pw = 0; pw < PW; ++pw)
            for (int i = 0; i < g; ++i) {
              const PullEntry e = tx_tab[pw * g + i];
              const bool in = (e.lo >= x0 && e.lo <= x1 && e.wh != 0.0f) || (e.hi >= x0 && e.hi <= x1 && e.wl != 0.0f);
              if (in) { lo_ = min(lo_, pw); hi_ = pw; }
            }
          S.pwlo[r_] = lo_;
          S.pwhi[r_] = hi_;
        }
      }
      __syncthreads();
      // ---- (C) consume --------------------------------------------------------------------------
      if (live) {
        for (int r_ = 0; r_ < nb; ++r_) {
          const int np = S.nph[r_ * RY + ty];
          const int pl = S.pwlo[r_], phh = S.pwhi[r_];
          if (np == 0 || pl > phh) continue;
          const T* gk = gout + (int64_t)S.meta_k[r_] * gs_k + c4;
          const unsigned char* pidx = S.ph_idx + (r_ * RY + ty) * PH;
          const float* pwt = S.ph_w + (r_ * RY + ty) * PH;
          for (int pw = pl; pw <= phh; ++pw) {
            float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int i = 0; i < np; ++i) {
              const float w = pwt[i];
              const float4 v = load_gout4<T>(gk + (int64_t)pidx[i] * gs_h + (int64_t)pw * gs_w);
              t.x += w * v.x; t.y += w * v.y; t.z += w * v.z; t.w += w * v.w;
            }
            S.T[pw * kPullThreads + tid] = t;
          }
          const float* cwr = S.cw + r_ * kTW * PW;
#pragma unroll
          for (int j = 0; j < kTW; ++j) {
            const int pa = S.cpa[r_ * kTW + j], pb = S.cpb[r_ * kTW + j];
            for (int pw = pa; pw <= pb; ++pw) {
              const float w = cwr[j * PW + pw];
              const float4 t = S.T[pw * kPullThreads + tid];
              acc[j].x += w * t.x; acc[j].y += w * t.y; acc[j].z += w * t.z; acc[j].w += w * t.w;
            }
          }
        }
      }
      __syncthreads();
    }
  }

  if (live) {
#pragma unroll
    for (int j = 0; j < kTW; ++j)
      if (x0 + j <= x1) *reinterpret_cast<float4*>(grow + (int64_t)(x0 + j) * sw) = acc[j];
  }
}

template <typename T>
static int pull_typed(const LevelsParam& lv, const RoiArgs& a, const void* gout, const int64_t* gs,
                      const int32_t* bperm, const int32_t* boff, int accumulate, cudaStream_t stream) {
  PullTiles t;
  const int CG = lv.c / 4;
  int tpr = 16;
  while (tpr < CG && tpr < kPullThreads) tpr <<= 1;
  t.TPR = tpr;
  t.RY = kPullThreads / tpr;
  t.chunks = (CG + tpr - 1) / tpr;
  int total = 0;
  for (int i = 0; i < lv.L; ++i) {
    const int l = lv.L - 1 - i;  // coarsest level first
    t.order[i] = l;
    t.tiles_y[l] = (lv.h[l] + t.RY - 1) / t.RY;
    t.tiles_x[l] = (lv.w[l] + kTW - 1) / kTW;
    t.start[i] = total;
    total += lv.n * t.tiles_y[l] * t.tiles_x[l] * t.chunks;
  }
  t.start[lv.L] = total;
  const size_t smem = pull_smem_layout(a.PH, a.PW, a.sampling_ratio, t.RY, nullptr, nullptr);
  if (smem > 200 * 1024) return RAF_ERR_UNSUPPORTED;
  if (cudaFuncSetAttribute(bwd_pull_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return RAF_ERR_CUDA;
  bwd_pull_kernel<T><<<total, kPullThreads, smem, stream>>>(lv, a, reinterpret_cast<const T*>(gout), gs[0], gs[2],
                                                            gs[3], bperm, boff, t, accumulate);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

int launch_backward_pull(const LevelsParam& glv, raf_dtype gout_dtype, const RoiArgs& a, const void* grad_out,
                         const int64_t* gout_strides, const int32_t* bperm, const int32_t* boff, int accumulate,
                         cudaStream_t stream) {
  switch (gout_dtype) {
    case RAF_F32: return pull_typed<float>(glv, a, grad_out, gout_strides, bperm, boff, accumulate, stream);
    case RAF_F16: return pull_typed<__half>(glv, a, grad_out, gout_strides, bperm, boff, accumulate, stream);
    case RAF_BF16: return pull_typed<__nv_bfloat16>(glv, a, grad_out, gout_strides, bperm, boff, accumulate, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
