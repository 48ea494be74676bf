// raf_pull_prep.cuh -- device code of the pull backward's PREP work, shared by pull_prep_kernel
// (raf_backward_pull.cu) and by the leading blocks of the forward launch (raf_forward.cu: the
// forward has the same RoIs and geometry, so it can produce the backward's tables for free while it
// gathers; roi_align_fpn_backward(RAF_REUSE_PREP) then skips its own prep launch).
#pragma once
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

constexpr uint32_t kPixMask = 0x00ffffffu;   // tap.pb = pixel | bin << 24; pixel == kPixMask: empty slot
constexpr int kPrepThreads = 256;            // block size of the stand-alone prep launch

// Arguments the tables depend on, hashed on the host (raf_api.cu); the prep writes it, the pull
// kernel compares it before it trusts a workspace it did not just fill (RAF_REUSE_PREP).
struct PrepFingerprint {
  uint32_t v[8];
};

struct PullPrepOut {
  uint32_t* hdr;    // [8] fingerprint of the arguments the tables were built for
  int32_t* bperm;   // [K]
  int32_t* boff;    // [L*N + 1]
  int4* bwin;       // [K]
  float4* bgeo;     // [K] {sy, bh, sx, bw} of every kept RoI on its level, bperm order (strip backward)
  PullTap* taps;    // [K][PH + PW][2g]
  int nblocks;      // 1 + ceil(K * (PH + PW) / block size); 0: no prep work in this launch
  PrepFingerprint fp;
};

__host__ __device__ inline int pull_prep_blocks(const RoiArgs& a, int nthreads) {
  if (a.sampling_ratio <= 0) return 1;   // adaptive grid: no tap tables (only the strip backward takes it), buckets only
  const int64_t items = (int64_t)a.K * (a.PH + a.PW);
  return 1 + (int)((items + nthreads - 1) / nthreads);
}

// ---------------------------------------------------------------------------------------------
// Tap tables.  One thread per (RoI, axis, bin): the bin's g samples give up to 2g (pixel, weight)
// taps; equal pixels are merged (weights summed in sample order); unused slots are marked empty.
// Layout: taps[k][PH + PW bins][2g slots]; y bins first.  Invalid samples (outside [-1, n], reading
// S6) produce no tap, so the product Y x X enumerates exactly the valid samples of the forward.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void pull_taps_item(const LevelsParam& lv, const RoiArgs& a, int64_t idx,
                                               PullTap* __restrict__ taps) {
  const int nb = a.PH + a.PW;
  const int k = (int)(idx / nb), b = (int)(idx - (int64_t)k * nb);
  const bool isy = b < a.PH;
  const int bin = isy ? b : b - a.PH;
  const int g = a.sampling_ratio, slots = 2 * g;
  const float* r = a.rois + 5 * (int64_t)k;
  const float x1 = __ldg(r + 1), y1 = __ldg(r + 2), x2 = __ldg(r + 3), y2 = __ldg(r + 4);
  const int level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);
  const RoiGeom geo = roi_geom(x1, y1, x2, y2, lv.scale[level], a.PH, a.PW, g, a.aligned);
  const int n = isy ? lv.h[level] : lv.w[level];
  const float scale_w = isy ? geo.inv_count : 1.0f;
  const float start = isy ? geo.sy : geo.sx, bsz = isy ? geo.bh : geo.bw;
  PullTap* out = taps + idx * slots;
  const uint32_t tag = (uint32_t)bin << 24;
  if (g <= 2) {   // the usual case: merge in registers, one 8-byte store per slot
    uint32_t pix[4] = {kPixMask, kPixMask, kPixMask, kPixMask};
    float w[4] = {0.f, 0.f, 0.f, 0.f};
    int cnt = 0;
    auto add = [&](uint32_t p, float v) {
      bool found = false;
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (q < cnt && pix[q] == p) { w[q] += v; found = true; }
      if (!found) {
#pragma unroll
        for (int q = 0; q < 4; ++q)
          if (q == cnt) { pix[q] = p; w[q] = v; }
        ++cnt;
      }
    };
    for (int i = 0; i < g; ++i) {
      const AxisTap t = axis_tap(sample_coord(start, bsz, bin, i, g), n);
      if (!t.valid) continue;
      add((uint32_t)t.lo, t.wh * scale_w);
      add((uint32_t)t.hi, t.wl * scale_w);
    }
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if (q < slots) { PullTap e; e.pb = tag | pix[q]; e.w = w[q]; out[q] = e; }
    return;
  }
  int cnt = 0;
  auto add = [&](int pix, float w) {
    for (int q = 0; q < cnt; ++q)
      if ((out[q].pb & kPixMask) == (uint32_t)pix) { out[q].w += w; return; }
    out[cnt].pb = tag | (uint32_t)pix;
    out[cnt].w = w;
    ++cnt;
  };
  for (int i = 0; i < g; ++i) {
    const AxisTap t = axis_tap(sample_coord(start, bsz, bin, i, g), n);
    if (!t.valid) continue;
    add(t.lo, t.wh * scale_w);
    add(t.hi, t.wl * scale_w);
  }
  for (int q = cnt; q < slots; ++q) { out[q].pb = tag | kPixMask; out[q].w = 0.0f; }
}


// ---------------------------------------------------------------------------------------------
// Stable bucketing by (level, image): key = level * N + batch_idx.  Feeds the pull backward
// (raf_backward_pull.cu), whose tiles walk the RoIs of their own (level, image) in ascending k --
// a fixed order, hence bit-reproducible sums.  RoIs with an invalid batch index are dropped.
//   bperm[K]      RoI indices grouped by key, ascending k inside a key
//   boff[NK + 1]  start of every key's group (NK = L * N)
//   bwin[K]       (optional) in bperm order: conservative window {ymin, ymax, xmin, xmax} of the
//                 pixels the RoI's samples can touch on its level (empty: ymin > ymax)
// Block 0 of pull_prep_kernel (the other blocks write the tap tables, same launch): 8 warps; warp w owns the contiguous RoI range [w*q, (w+1)*q).  cnt[w][key] first
// counts, then (after a scan over keys, warps minor) holds the next free slot of (key, warp):
// warp-private rows, so neither atomics nor block barriers inside the walks.
// ---------------------------------------------------------------------------------------------

// Pixels an axis can touch: samples are monotone in (bin, i) up to rounding, so the first and the
// last sample (with slack for that rounding) bound all of them; a sample at v touches
// floor(max(v,0)) and the next pixel (clamped to n-1); samples outside [-1, n] touch nothing.
__device__ __forceinline__ void axis_window(float start, float bin, int P, int g, int n, int& lo, int& hi) {
  lo = 0x7fffffff; hi = -1;
  if (g <= 0) return;   // adaptive grid of a box with no extent: no samples
  const float va = sample_coord(start, bin, 0, 0, g), vb = sample_coord(start, bin, P - 1, g - 1, g);
  const float slack = 0.01f + 1e-6f * fmaxf(fabsf(va), fabsf(vb));
  const float vlo = fminf(va, vb) - slack, vhi = fmaxf(va, vb) + slack;
  if (!(vlo <= vhi) || vhi < -1.0f || vlo > (float)n) return;   // NaN or entirely outside
  lo = (int)fminf(fmaxf(vlo, 0.0f), (float)(n - 1));
  hi = min(n - 1, (int)fminf(fmaxf(vhi, 0.0f), (float)(n - 1)) + 1);
}

// The prep work of one block of `blockDim.x` threads (a multiple of 32): block 0 buckets, blocks
// 1.. write tap tables.  s_cnt: (blockDim.x / 32 + 1) * (L * N + 1) ints of shared memory.
__device__ __forceinline__ void pull_prep_block(const LevelsParam& lv, const RoiArgs& a, const PullPrepOut& o,
                                                int block, int* s_cnt) {
  const int nthreads = blockDim.x, nwarps = nthreads >> 5;
  int32_t* __restrict__ bperm = o.bperm;
  int32_t* __restrict__ boff = o.boff;
  int4* __restrict__ bwin = o.bwin;
  if (block > 0) {           // blocks 1.. : tap tables (independent of the bucketing; fixed grids only)
    if (a.sampling_ratio <= 0) return;
    const int64_t idx = (int64_t)(block - 1) * nthreads + threadIdx.x;
    if (idx < (int64_t)a.K * (a.PH + a.PW)) pull_taps_item(lv, a, idx, o.taps);
    return;
  }
  const int K = a.K, L = lv.L, N = lv.n;
  const int NK = L * N, NK1 = NK + 1;
  int* s_tot = s_cnt + nwarps * NK1;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int q = ((K + nwarps - 1) / nwarps + 31) & ~31;  // per-warp range, multiple of 32
  const int lo = warp * q, hi = min(K, lo + q);
  if (tid < 8) o.hdr[tid] = o.fp.v[tid];
  for (int i = tid; i < nwarps * NK1 + NK1; i += nthreads) s_cnt[i] = 0;
  __syncthreads();

  auto key_of = [&](int k) -> int {
    if (k >= hi) return -1;
    const float* r = a.rois + 5 * (int64_t)k;
    const int b = batch_index_of(r[0], N);
    if (b < 0) return NK;  // dropped
    return level_of(r[1], r[2], r[3], r[4], L, a.finest_scale) * N + b;
  };

  int* mine = s_cnt + warp * NK1;
  for (int k0 = lo; k0 < hi; k0 += 32) {
    const int key = key_of(k0 + lane);
    const unsigned peers = __match_any_sync(0xffffffffu, key);
    if (key >= 0 && lane == __ffs(peers) - 1) mine[key] += __popc(peers);
    __syncwarp();
  }
  __syncthreads();

  // totals per key
  for (int key = tid; key < NK1; key += nthreads) {
    int t = 0;
    for (int w = 0; w < nwarps; ++w) t += s_cnt[w * NK1 + key];
    s_tot[key] = t;
  }
  __syncthreads();
  if (warp == 0) {  // exclusive scan of the totals over keys, 32 at a time
    int carry = 0;
    for (int base = 0; base < NK1; base += 32) {
      const int key = base + lane;
      const int v = key < NK1 ? s_tot[key] : 0;
      int incl = v;
      for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
      }
      if (key < NK1) s_tot[key] = carry + incl - v;
      carry += __shfl_sync(0xffffffffu, incl, 31);
    }
  }
  __syncthreads();
  for (int key = tid; key < NK1; key += nthreads) {
    if (key <= NK) boff[key] = s_tot[key];  // boff[NK] = number of kept RoIs
    int run = s_tot[key];
    for (int w = 0; w < nwarps; ++w) {
      const int c = s_cnt[w * NK1 + key];
      s_cnt[w * NK1 + key] = run;
      run += c;
    }
  }
  __syncthreads();

  for (int k0 = lo; k0 < hi; k0 += 32) {
    const int k = k0 + lane;
    const int key = key_of(k);
    const unsigned peers = __match_any_sync(0xffffffffu, key);
    const int base = (key >= 0) ? mine[key] : 0;
    __syncwarp();
    if (key >= 0 && key < NK) {
      const int p = base + __popc(peers & ((1u << lane) - 1u));
      bperm[p] = k;
      if (bwin) {
        const float* r = a.rois + 5 * (int64_t)k;
        const int level = key / N;
        const RoiGeom geo = roi_geom(r[1], r[2], r[3], r[4], lv.scale[level], a.PH, a.PW, a.sampling_ratio, a.aligned);
        int4 w;
        axis_window(geo.sy, geo.bh, a.PH, geo.gh, lv.h[level], w.x, w.y);
        axis_window(geo.sx, geo.bw, a.PW, geo.gw, lv.w[level], w.z, w.w);
        if (w.x > w.y || w.z > w.w) w = make_int4(0x7fffffff, -1, 0x7fffffff, -1);
        bwin[p] = w;
        if (o.bgeo) o.bgeo[p] = make_float4(geo.sy, geo.bh, geo.sx, geo.bw);
      }
    }
    if (key >= 0 && lane == __ffs(peers) - 1) mine[key] = base + __popc(peers);
    __syncwarp();
  }
}


}  // namespace raf
