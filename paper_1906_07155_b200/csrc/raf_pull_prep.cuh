// raf_pull_prep.cuh -- device code of the pull backward's PREP work, shared by pull_prep_kernel
// (raf_backward_pull.cu) and by the extra blocks of the forward launch (raf_forward.cu: the
// forward has the same RoIs and geometry, so it can produce the backward's tables for free while it
// gathers; roi_align_fpn_backward(RAF_REUSE_PREP) then skips its own prep launch).
//
// What the prep leaves in the workspace:
//   hdr[0..7]     fingerprint of the arguments the tables were built for (checked by the pull kernel)
//   hdr[8], hdr[9]  work-item counter and finished-CTA counter of the persistent pull kernel, zeroed here
//   bperm[K]      RoI indices grouped by (level, image), ascending k inside a group (stable)
//   boff[L*N+1]   start of every group
//   bwin[K]       in bperm order: conservative window {ymin, ymax, xmin, xmax} of the pixels the RoI's
//                 samples can touch on its level (empty: ymin > ymax)
//   inv[K][2][kInvCap]  INVERSE tap tables, indexed by original k, axis (0 = y, 1 = x) and pixel offset
//                 j = pixel - window_min: which output bins have a sample tap on that pixel row /
//                 column, and with which (merged) weight.  The bins that touch one pixel are
//                 consecutive, so an entry is {first bin, count, weights[count]}; y weights carry
//                 1/count of the sampling grid.  This is the transpose of the forward's per-bin tap
//                 lists: row y of the backward gets  sum_ph wy[ph] * sum_pw wx[pw] * gout[ph][pw].
#pragma once
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

constexpr int kPrepThreads = 256;   // block size of the stand-alone prep launch
constexpr int kInvCap = 64;         // pixels per axis covered by a RoI's inverse table; wider windows
                                    // are evaluated on the fly by the pull kernel (same function)
constexpr int kInvW = 7;            // weights stored per entry; longer runs (bins narrower than 2/7 px)
                                    // are evaluated on the fly

struct __align__(16) InvEntry {
  uint32_t meta;      // first bin | count << 8   (count == 0: nothing lands on this pixel)
  float w[kInvW];     // weights of bins first .. first + count - 1 (the first kInvW of them)
};
static_assert(sizeof(InvEntry) == 32, "InvEntry is two 16-byte words");

// Arguments the tables depend on, hashed on the host (raf_api.cu); the prep writes it, the pull
// kernel compares it before it trusts a workspace it did not just fill (RAF_REUSE_PREP).
struct PrepFingerprint {
  uint32_t v[8];
};

struct PullPrepOut {
  uint32_t* hdr;    // [10]
  int32_t* bperm;   // [K]
  int32_t* boff;    // [L*N + 1]
  int4* bwin;       // [K]
  InvEntry* inv;    // [K][2][kInvCap]
  int nblocks;      // 1 + ceil(K * 2 * kInvCap / block size); 0: no prep work in this launch
  PrepFingerprint fp;
};

__host__ __device__ inline int pull_prep_blocks(const RoiArgs& a, int nthreads) {
  const int64_t items = (int64_t)a.K * 2 * kInvCap;
  return 1 + (int)((items + nthreads - 1) / nthreads);
}

// Pixels an axis can touch: samples are monotone in (bin, i) up to rounding, so the first and the
// last sample (with slack for that rounding) bound all of them; a sample at v touches
// floor(max(v,0)) and the next pixel (clamped to n-1); samples outside [-1, n] touch nothing.
__device__ __forceinline__ void axis_window(float start, float bin, int P, int g, int n, int& lo, int& hi) {
  lo = 0x7fffffff; hi = -1;
  if (g <= 0) return;   // adaptive grid of a box with non-positive extent: no samples (reading S7)
  const float va = sample_coord(start, bin, 0, 0, g), vb = sample_coord(start, bin, P - 1, g - 1, g);
  const float slack = 0.01f + 1e-6f * fmaxf(fabsf(va), fabsf(vb));
  const float vlo = fminf(va, vb) - slack, vhi = fmaxf(va, vb) + slack;
  if (!(vlo <= vhi) || vhi < -1.0f || vlo > (float)n) return;   // NaN or entirely outside
  lo = (int)fminf(fmaxf(vlo, 0.0f), (float)(n - 1));
  hi = min(n - 1, (int)fminf(fmaxf(vhi, 0.0f), (float)(n - 1)) + 1);
}

// Geometry of RoI k on its level, as every kernel of the path evaluates it (C1, C3).
struct RoiOnLevel {
  int level, b;     // b < 0: invalid batch index (reading S17)
  RoiGeom geo;
};
__device__ __forceinline__ RoiOnLevel roi_on_level(const LevelsParam& lv, const RoiArgs& a, int k) {
  const float* r = a.rois + 5 * (int64_t)k;
  const float r0 = __ldg(r), x1 = __ldg(r + 1), y1 = __ldg(r + 2), x2 = __ldg(r + 3), y2 = __ldg(r + 4);
  RoiOnLevel o;
  o.b = batch_index_of(r0, lv.n);
  o.level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);
  o.geo = roi_geom(x1, y1, x2, y2, lv.scale[o.level], a.PH, a.PW, a.sampling_ratio, a.aligned);
  return o;
}

// Weight with which output bin `bin` of an axis lands on pixel `pix`: the taps of the bin's g samples
// that fall on the pixel, summed in sample order (lo tap before hi tap) -- the same floats, in the
// same order, as the forward's merged tap of that bin and pixel.  `hit` tells whether any tap did.
__device__ __forceinline__ float inv_bin_weight(float start, float bsz, int bin, int g, int n, float scale_w,
                                                int pix, bool& hit) {
  float acc = 0.0f;
  hit = false;
  for (int i = 0; i < g; ++i) {
    const AxisTap t = axis_tap(sample_coord(start, bsz, bin, i, g), n);
    if (!t.valid) continue;
    if (t.lo == pix) { acc += t.wh * scale_w; hit = true; }
    if (t.hi == pix) { acc += t.wl * scale_w; hit = true; }
  }
  return acc;
}

// Inverse table entry of one pixel row (axis 0) or column (axis 1) of a RoI.  Bins between the first
// and the last one that hit get their weight (0 for a bin without a tap, which monotone sample
// coordinates exclude up to rounding flukes of degenerate boxes).
__device__ __forceinline__ InvEntry inv_entry_compute(const LevelsParam& lv, const RoiArgs& a,
                                                      const RoiOnLevel& r, int axis, int pix) {
  const int n = axis ? lv.w[r.level] : lv.h[r.level];
  const int P = axis ? a.PW : a.PH, g = axis ? r.geo.gw : r.geo.gh;
  const float start = axis ? r.geo.sx : r.geo.sy, bsz = axis ? r.geo.bw : r.geo.bh;
  const float scale_w = axis ? 1.0f : r.geo.inv_count;
  InvEntry e;
  e.meta = 0;
#pragma unroll
  for (int q = 0; q < kInvW; ++q) e.w[q] = 0.0f;
  int first = -1, last = -1;
  for (int bin = 0; bin < P; ++bin) {
    bool hit;
    const float w = inv_bin_weight(start, bsz, bin, g, n, scale_w, pix, hit);
    if (!hit) continue;
    if (first < 0) first = bin;
    last = bin;
    const int idx = bin - first;
#pragma unroll
    for (int q = 0; q < kInvW; ++q)
      if (q == idx) e.w[q] = w;
  }
  if (first >= 0) e.meta = (uint32_t)first | ((uint32_t)(last - first + 1) << 8);
  return e;
}

// One inverse-table item: idx = (k * 2 + axis) * kInvCap + j.
__device__ __forceinline__ void pull_inv_item(const LevelsParam& lv, const RoiArgs& a, int64_t idx,
                                              InvEntry* __restrict__ inv) {
  const int j = (int)(idx % kInvCap);
  const int axis = (int)((idx / kInvCap) & 1);
  const int k = (int)(idx / (2 * kInvCap));
  const RoiOnLevel r = roi_on_level(lv, a, k);
  if (r.b < 0) return;
  int lo, hi;
  if (axis) axis_window(r.geo.sx, r.geo.bw, a.PW, r.geo.gw, lv.w[r.level], lo, hi);
  else axis_window(r.geo.sy, r.geo.bh, a.PH, r.geo.gh, lv.h[r.level], lo, hi);
  if (lo > hi || lo + j > hi) return;   // outside the window: never read
  const InvEntry e = inv_entry_compute(lv, a, r, axis, lo + j);
  uint4* dst = reinterpret_cast<uint4*>(inv + idx);
  dst[0] = make_uint4(e.meta, __float_as_uint(e.w[0]), __float_as_uint(e.w[1]), __float_as_uint(e.w[2]));
  dst[1] = make_uint4(__float_as_uint(e.w[3]), __float_as_uint(e.w[4]), __float_as_uint(e.w[5]), __float_as_uint(e.w[6]));
}

// ---------------------------------------------------------------------------------------------
// Stable bucketing by (level, image): key = level * N + batch_idx.  Feeds the pull backward
// (raf_backward_pull.cu), whose tiles walk the RoIs of their own (level, image) in ascending k --
// a fixed order, hence bit-reproducible sums.  RoIs with an invalid batch index are dropped.
// Block 0 of the prep (the other blocks write the inverse tables, same launch): warp w owns the
// contiguous RoI range [w*q, (w+1)*q).  cnt[w][key] first counts, then (after a scan over keys,
// warps minor) holds the next free slot of (key, warp): warp-private rows, so neither atomics nor
// block barriers inside the walks.
// ---------------------------------------------------------------------------------------------

// The prep work of one block of `blockDim.x` threads (a multiple of 32): block 0 buckets, blocks
// 1.. write inverse tables.  s_cnt: (blockDim.x / 32 + 1) * (L * N + 1) ints of shared memory.
__device__ __forceinline__ void pull_prep_block(const LevelsParam& lv, const RoiArgs& a, const PullPrepOut& o,
                                                int block, int* s_cnt) {
  const int nthreads = blockDim.x, nwarps = nthreads >> 5;
  int32_t* __restrict__ bperm = o.bperm;
  int32_t* __restrict__ boff = o.boff;
  int4* __restrict__ bwin = o.bwin;
  if (block > 0) {           // blocks 1.. : inverse tables (independent of the bucketing)
    const int64_t idx = (int64_t)(block - 1) * nthreads + threadIdx.x;
    if (idx < (int64_t)a.K * 2 * kInvCap) pull_inv_item(lv, a, idx, o.inv);
    return;
  }
  const int K = a.K, L = lv.L, N = lv.n;
  const int NK = L * N, NK1 = NK + 1;
  int* s_tot = s_cnt + nwarps * NK1;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int q = ((K + nwarps - 1) / nwarps + 31) & ~31;  // per-warp range, multiple of 32
  const int lo = warp * q, hi = min(K, lo + q);
  if (tid < 8) o.hdr[tid] = o.fp.v[tid];
  if (tid == 8 || tid == 9) o.hdr[tid] = 0u;   // work counter / finished-CTA counter of the pull kernel
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
        const int o2 = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o2;
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
        const RoiOnLevel r = roi_on_level(lv, a, k);
        int4 w;
        axis_window(r.geo.sy, r.geo.bh, a.PH, r.geo.gh, lv.h[r.level], w.x, w.y);
        axis_window(r.geo.sx, r.geo.bw, a.PW, r.geo.gw, lv.w[r.level], w.z, w.w);
        if (w.x > w.y || w.z > w.w) w = make_int4(0x7fffffff, -1, 0x7fffffff, -1);
        bwin[p] = w;
      }
    }
    if (key >= 0 && lane == __ffs(peers) - 1) mine[key] = base + __popc(peers);
    __syncwarp();
  }
}

}  // namespace raf
