// raf_backward_strip.cu -- K3d, second generation: deterministic PULL backward with row-strip
// register accumulators and warp-autonomous tiles (reading S12; H5: the
// backward's bytes are the gradient pyramid, so every element of it is owned by exactly one warp and
// written exactly once -- no memset, no atomics, fixed summation order).
//
// Work unit = one WARP TILE: (image n, level l, TH rows x 8 columns, a chunk of 256 channels), TH = 8
// on sparse levels, smaller on the dense coarse ones.  A warp processes its tile alone -- there is no
// block-wide barrier anywhere in the kernel, so the warps resident on an SM are always in different
// phases and cover each other's latencies.  Lanes = channels (two float4 per lane, 128 channels apart:
// every warp-wide access covers contiguous bytes); the warp walks the rows of the tile and holds one
// row STRIP of 8 pixels x 256 channels in 64 fp32 accumulator registers per lane.
//
// The transpose of the forward is separable: for RoI k and pixel (y, x)
//     g[y][x] += sum_{ph} sum_{pw} wy_k(y, ph) * wx_k(x, pw) * gout[k][ph][pw]
// and it is evaluated BINS-OUTER: each vector gout[k][ph][pw][256 channels] a strip needs is loaded
// ONCE per strip and FMA'd into every pixel of the strip it touches (the first generation,
// raf_backward_pull.cu, re-loaded it for every pixel: 508 MB through the L1 path against 51 MB of
// grad_out -- profiles/r1_v6.md).  Which accumulators a vector lands in is decided by warp-uniform
// branches on the item's column mask (all lanes of a warp work on the same item: no divergence).
//
// Per warp tile:
//  (A) scan: the lanes test the conservative pixel windows `bwin` of the tile's (level, image) bucket
//      against the tile, 288 records per round trip, and keep the next NC RoIs that meet it (bucket
//      order = ascending k: fixed summation order); their geometry `bgeo` and grad_out row offset
//      follow in one more round trip.  A tile that meets more than NC RoIs takes the bucket in several
//      batches; later batches add to what the earlier ones stored (one-row tiles keep their sums in
//      registers instead).
//  (B) tables: one lane per (candidate, axis, bin) evaluates the bin's g samples with the canonical
//      fp32 coordinate arithmetic (raf_device.cuh, bit-identical to the forward) and leaves DENSE
//      weights in the warp's shared memory: xw[c][pw][8 columns], yw[c][8 rows][ph], the ph bits with a
//      tap on every row and the list of bins with a tap inside the strip.  No tap tables in global memory.
//  (C) work list: lane c owns candidate c and emits its items -- one per (row, ph, pw) with a tap on the
//      row and inside the strip: grad_out offset, column mask, wy * xw[8 columns] -- at the positions a
//      warp prefix sum assigns (row-major, then c, ph, pw).  The warp consumes the list through a ring
//      of cp.async stages: the vectors of the next kRing - 1 items, across row boundaries, are in flight
//      while the current one is FMA'd with packed fp32x2 FMAs (memory-level parallelism at no register
//      cost; each lane copies and reads back its own 16 bytes, so no barrier is needed).
//  (D) a row is stored when its last item is done (zero where nothing lands; added to the old value
//      with RAF_ACCUMULATE or in a later batch).
// Any sampling grid (fixed g >= 1, or the adaptive per-RoI grid of sampling_ratio == 0) and any
// out_h / out_w <= 32 take this path (no tap-count limit).
//
// Measured (B200, cold-L2 rotation, profiles/r2_experiments.md): config 5 (16 images, 25.8 K warp tiles)
// 516 -> 455 us against the first generation; on config 2 (2 images, 3.2 K warp tiles = 1.8 waves of
// 12 resident warps per SM) the fixed ~8 us of dependent round trips per tile is not covered and the
// first generation stays ahead (89 vs 95 us), as it does for outputs finer than the pixel grid
// (14 x 14 bins: a vector then feeds only 1-2 pixels, so loading it once per strip buys nothing).
// raf_api.cu picks per call.
#include "raf_device.cuh"
#include "raf_host.h"
#include "raf_pull_prep.cuh"
#include <cstdlib>
#include <cstring>

namespace raf {

#ifndef RAF_STRIP_WARPS
#define RAF_STRIP_WARPS 2
#endif
constexpr int kStripWarps = RAF_STRIP_WARPS;   // warps per CTA (independent of one another)
constexpr int kStripCols = 8;                  // strip width (accumulator sets per lane)
constexpr int kStripMaxRows = 8;
#ifndef RAF_STRIP_RING
#define RAF_STRIP_RING 6
#endif
constexpr int kRing = RAF_STRIP_RING;          // cp.async stages per warp
#ifndef RAF_STRIP_WORK
#define RAF_STRIP_WORK 96
#endif
constexpr int kWorkCap = RAF_STRIP_WORK;       // work-list items per flush (>= 32)
constexpr int kScanRounds = 9;                 // bucket records per lane and round trip

struct StripLevels {
  void* data[kMaxLevels];
  int64_t sn[kMaxLevels];
  int32_t sh[kMaxLevels], sw[kMaxLevels];
  int32_t h[kMaxLevels], w[kMaxLevels];
  int32_t th[kMaxLevels];         // tile rows of the level (1, 2, 4 or 8)
  int32_t tiles_x[kMaxLevels];
  int32_t start[kMaxLevels + 1];  // first tile of the level at schedule position i (coarsest level first)
  int32_t order[kMaxLevels];      // level at schedule position i
  int32_t L, N, C, chunks;
  int32_t total;                  // warp tiles = tiles x N x chunks
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int kBytes>
__device__ __forceinline__ void cp_async_ca(uint32_t dst, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst), "l"(src), "n"(kBytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int kPending>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(kPending) : "memory"); }

// 4 channels of grad_out per lane and half: 16 bytes of fp32 or 8 bytes of fp16 / bf16.
template <typename T> struct StripVec;
template <> struct StripVec<float> {
  static constexpr int kBytes = 16;
  static __device__ __forceinline__ float4 read(const unsigned char* p) { return *reinterpret_cast<const float4*>(p); }
};
template <> struct StripVec<__half> {
  static constexpr int kBytes = 8;
  static __device__ __forceinline__ float4 read(const unsigned char* p) {
    const uint2 r = *reinterpret_cast<const uint2*>(p);
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
    return make_float4(a.x, a.y, b.x, b.y);
  }
};
template <> struct StripVec<__nv_bfloat16> {
  static constexpr int kBytes = 8;
  static __device__ __forceinline__ float4 read(const unsigned char* p) {
    const uint2 r = *reinterpret_cast<const uint2*>(p);
    return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u),
                       __uint_as_float(r.y << 16), __uint_as_float(r.y & 0xffff0000u));
  }
};

// acc += w * v on 4 channels with two packed fp32x2 FMAs (sm_100: one issue slot per two FMAs; each half
// rounds exactly like fmaf).
__device__ __forceinline__ void strip_fma(float4& acc, float w, const float4& v) {
  const float2 ww = make_float2(w, w);
  const float2 lo = __ffma2_rn(ww, make_float2(v.x, v.y), make_float2(acc.x, acc.y));
  const float2 hi = __ffma2_rn(ww, make_float2(v.z, v.w), make_float2(acc.z, acc.w));
  acc = make_float4(lo.x, lo.y, hi.x, hi.y);
}

// Dense weights of one output bin along one axis on the 8 pixels [origin, origin + 8): the bin's g
// samples (C3), weights of equal pixels summed in sample order, invalid samples (reading S6) skipped.
__device__ __forceinline__ uint32_t strip_bin_weights(float start, float bsz, int bin, int g, int n, float scale_w,
                                                      int origin, float (&w)[8]) {
  uint32_t mask = 0;
#pragma unroll
  for (int r = 0; r < 8; ++r) w[r] = 0.0f;
  for (int s = 0; s < g; ++s) {
    const AxisTap t = axis_tap(sample_coord(start, bsz, bin, s, g), n);
    if (!t.valid) continue;
    const int rlo = t.lo - origin, rhi = t.hi - origin;
    const float wlo = t.wh * scale_w, whi = t.wl * scale_w;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      if (rlo == r) { w[r] += wlo; mask |= 1u << r; }
      if (rhi == r) { w[r] += whi; mask |= 1u << r; }
    }
  }
  return mask;
}

// Per-warp shared memory (bytes), in this order: ring | work list | xw | yw | cgeo | xl | yph | cgoff | rowend | cnb.
__host__ __device__ inline size_t strip_warp_smem(int NC, int PH, int PW, size_t esz) {
  size_t s = (size_t)kRing * 256 * esz;
  s += 40 * (size_t)(kWorkCap + 2);
  s += sizeof(float) * NC * PW * 8;
  s += sizeof(float) * NC * 8 * PH;
  s += 16 * (size_t)NC + 8 * (size_t)NC * PW + 4 * (size_t)NC * 8 + 4 * (size_t)NC + 4 * (kStripMaxRows + 1);
  s += (size_t)NC;
  return (s + 127) & ~(size_t)127;
}

__device__ __forceinline__ int strip_pow2_lanes(int P) { return P <= 8 ? 8 : (P <= 16 ? 16 : 32); }


template <typename T, typename G, bool kFull>
__global__ void __launch_bounds__(32 * kStripWarps)
bwd_strip_kernel(const __grid_constant__ StripLevels sl, const RoiArgs a, const T* __restrict__ gout, int gs_k, int gs_h,
                 int gs_w, const uint32_t* __restrict__ hdr, const int32_t* __restrict__ bperm,
                 const int32_t* __restrict__ boff, const int4* __restrict__ bwin, const float4* __restrict__ bgeo, int NC,
                 int accumulate, const PrepFingerprint fp) {
  using SV = StripVec<T>;
  constexpr int kStage = 64 * SV::kBytes;   // bytes of one ring stage: 256 channels
  extern __shared__ __align__(128) unsigned char strip_smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int wt = blockIdx.x * kStripWarps + warp;
  if (wt >= sl.total) return;
  const int PH = a.PH, PW = a.PW, g = a.sampling_ratio;

  // ---- this warp's shared memory --------------------------------------------------------------------
  unsigned char* sp = strip_smem + (size_t)warp * strip_warp_smem(NC, PH, PW, sizeof(T));
  unsigned char* ring = sp;                            sp += (size_t)kRing * kStage;
  float4* work_wa = reinterpret_cast<float4*>(sp);     sp += 16 * (size_t)(kWorkCap + 2);   // wy * xw[columns 0..3] per item
  float4* work_wb = reinterpret_cast<float4*>(sp);     sp += 16 * (size_t)(kWorkCap + 2);   // wy * xw[columns 4..7]
  int2* work_hd = reinterpret_cast<int2*>(sp);         sp += 8 * (size_t)(kWorkCap + 2);    // {grad_out offset, column mask}
  float* s_xw = reinterpret_cast<float*>(sp);          sp += sizeof(float) * NC * PW * 8;   // [c][pw][column]
  float* s_yw = reinterpret_cast<float*>(sp);          sp += sizeof(float) * NC * 8 * PH;   // [c][row][ph]
  float4* s_cgeo = reinterpret_cast<float4*>(sp);      sp += 16 * (size_t)NC;               // {sy, bh, sx, bw}
  int2* s_xl = reinterpret_cast<int2*>(sp);            sp += 8 * (size_t)NC * PW;           // [c][e]: bins with a tap in the strip
  uint32_t* s_yph = reinterpret_cast<uint32_t*>(sp);   sp += 4 * (size_t)NC * 8;            // [c][row]: ph bits with a tap on the row
  int* s_cgoff = reinterpret_cast<int*>(sp);           sp += 4 * (size_t)NC;                // k * gs_k
  int* s_rowend = reinterpret_cast<int*>(sp);          sp += 4 * (kStripMaxRows + 1);
  unsigned char* s_cnb = sp;                                                                // entries of xl[c]

  // ---- decode the warp tile: tiles of the coarsest level first (most RoIs per pixel), image and
  //      channel chunk fastest --------------------------------------------------------------------------
  const int per_tile = sl.N * sl.chunks;
  const int tile = wt / per_tile, rem = wt - tile * per_tile;
  const int n = rem / sl.chunks, chunk = rem - n * sl.chunks;
  int pos = 0;
  while (pos + 1 < sl.L && tile >= sl.start[pos + 1]) ++pos;
  const int level = sl.order[pos];
  const int trem = tile - sl.start[pos];
  const int tiles_x = sl.tiles_x[level];
  const int tyi = trem / tiles_x, txi = trem - tyi * tiles_x;
  const int H = sl.h[level], W = sl.w[level], TH = sl.th[level];
  const int y0 = tyi * TH, x0 = txi * kStripCols;
  const int npy = min(TH, H - y0), npx = min(kStripCols, W - x0);
  const int x1 = x0 + npx - 1;
  const int chA = chunk * 256 + lane * 4, chB = chA + 128;
  const bool actA = kFull || chA < sl.C, actB = kFull || chB < sl.C;
  const T* goutA = gout + (actA ? chA : 0);
  const int sw = sl.sw[level], sh = sl.sh[level];
  G* gtile = reinterpret_cast<G*>(sl.data[level]) + (int64_t)n * sl.sn[level] + (int64_t)y0 * sh + (int64_t)x0 * sw + chA;

  const int key = level * sl.N + n;
  const int bbeg = __ldg(boff + key), bend = __ldg(boff + key + 1);
  // The workspace must hold the tables of exactly these arguments (RAF_REUSE_PREP contract): the warp
  // compares the fingerprint the prep left; on a mismatch the tile is poisoned with NaN.
  const bool bad = __any_sync(0xffffffffu, lane < 8 && __ldg(hdr + (lane & 7)) != fp.v[lane & 7]);

  float4 acc[kStripCols][2];
  const uint32_t ring_u32 = smem_u32(ring) + lane * SV::kBytes;
  const unsigned char* ring_rd = ring + lane * SV::kBytes;
  const unsigned lt_mask = (1u << lane) - 1u;

  auto zero_acc = [&]() {
#pragma unroll
    for (int j = 0; j < kStripCols; ++j) {
      acc[j][0] = make_float4(0.f, 0.f, 0.f, 0.f);
      acc[j][1] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  };
  auto store_row = [&](int r, bool add_old) {
    G* gp = gtile + r * sh;
#pragma unroll
    for (int j = 0; j < kStripCols; ++j) {
      if (j < npx) {
        float4 vA = acc[j][0], vB = acc[j][1];
        if (add_old) {
          if (actA) { const float4 o = Grad4<G>::load(gp); vA.x += o.x; vA.y += o.y; vA.z += o.z; vA.w += o.w; }
          if (actB) { const float4 o = Grad4<G>::load(gp + 128); vB.x += o.x; vB.y += o.y; vB.z += o.z; vB.w += o.w; }
        }
        if (actA) Grad4<G>::store(gp, vA);
        if (actB) Grad4<G>::store(gp + 128, vB);
      }
      gp += sw;
    }
  };
  auto prefetch = [&](int goff, int slot) {
    const T* src = goutA + goff;
    const uint32_t dst = ring_u32 + slot * kStage;
    if (actA) cp_async_ca<SV::kBytes>(dst, src);
    if (actB) cp_async_ca<SV::kBytes>(dst + 32 * SV::kBytes, src + 128);
  };

  if (bad) {
    const float qnan = __int_as_float(0x7fc00000);
#pragma unroll
    for (int j = 0; j < kStripCols; ++j) {
      acc[j][0] = make_float4(qnan, qnan, qnan, qnan);
      acc[j][1] = acc[j][0];
    }
    for (int r = 0; r < npy; ++r) store_row(r, false);
    return;
  }

  const int P2y = strip_pow2_lanes(PH), P2x = strip_pow2_lanes(PW);

  // The bucket is taken in batches of NC RoIs (usually one batch: one scan, one table build, one work list
  // across the rows of the tile).  Later batches add to what the earlier ones stored (tiles of one row
  // keep their sums in registers instead): the summation order stays fixed.
  {
    const int rb = 0, nr = npy;
    int spos = bbeg, batch = 0;
    zero_acc();
    while (true) {
      // ---- (A) the next <= NC RoIs of the bucket whose window meets the tile ---------------------------
      const int ya = y0, yb = y0 + npy - 1;
      int ncand = 0;
      while (spos < bend && ncand < NC) {
        int4 wv[kScanRounds];
#pragma unroll
        for (int u = 0; u < kScanRounds; ++u) {
          const int i = spos + u * 32 + lane;
          wv[u] = (i < bend) ? __ldg(bwin + i) : make_int4(0x7fffffff, -1, 0x7fffffff, -1);
        }
#pragma unroll
        for (int u = 0; u < kScanRounds; ++u) {
          if (ncand < NC && spos < bend) {   // (warp-uniform)
            const bool hit = (wv[u].x <= yb) && (wv[u].y >= ya) && (wv[u].z <= x1) && (wv[u].w >= x0);
            const unsigned mh = __ballot_sync(0xffffffffu, hit);
            const int nh = __popc(mh), room = NC - ncand;
            const int rank = __popc(mh & lt_mask);
            if (hit && rank < room) s_cgoff[ncand + rank] = spos + lane;   // bucket position, for now
            if (nh > room) {   // the batch is full: resume after the last record taken
              spos += __ffs(__ballot_sync(0xffffffffu, hit && rank == room - 1));
              ncand = NC;
            } else {
              spos += 32;
              ncand += nh;
            }
          }
        }
      }
      if (spos > bend) spos = bend;
      const bool last = spos >= bend;
      if (ncand == 0 && batch > 0 && npy > 1) break;   // (the bucket ended exactly at a batch boundary)
      __syncwarp();
      for (int c = lane; c < ncand; c += 32) {
        const int i = s_cgoff[c];
        s_cgeo[c] = __ldg(bgeo + i);
        s_cgoff[c] = __ldg(bperm + i) * gs_k;
      }
      __syncwarp();

      // ---- (B) dense weights.  Rows: one lane per (candidate, ph), 32 / P2y candidates per round -----
      for (int c0 = 0; c0 < ncand; c0 += 32 / P2y) {
        const int cl = lane / P2y, ph = lane - cl * P2y, c = c0 + cl;
        const bool cval = c < ncand, val = cval && ph < PH;
        float w[8];
        uint32_t m = 0;
        if (val) {
          const float4 geo = s_cgeo[c];
          const int gh = sampling_grid(g, geo.y), gw = sampling_grid(g, geo.w);   // (the fixed grid, or per RoI)
          const int cnt = gh * gw;
          m = strip_bin_weights(geo.x, geo.y, ph, gh, H, 1.0f / (float)(cnt > 1 ? cnt : 1), y0, w);
#pragma unroll
          for (int r = 0; r < 8; ++r) s_yw[(c * 8 + r) * PH + ph] = w[r];
        }
#pragma unroll
        for (int r = 0; r < 8; ++r) {
          const unsigned bal = __ballot_sync(0xffffffffu, (m >> r) & 1u);
          if (cval && ph == r) s_yph[c * 8 + r] = P2y == 32 ? bal : ((bal >> (cl * P2y)) & ((1u << P2y) - 1u));
        }
      }
      //      Columns: one lane per (candidate, pw); the bins with a tap inside the strip are also listed
      for (int c0 = 0; c0 < ncand; c0 += 32 / P2x) {
        const int cl = lane / P2x, pw = lane - cl * P2x, c = c0 + cl;
        const bool cval = c < ncand, val = cval && pw < PW;
        float w[8];
        uint32_t m = 0;
        if (val) {
          const float4 geo = s_cgeo[c];
          m = strip_bin_weights(geo.z, geo.w, pw, sampling_grid(g, geo.w), W, 1.0f, x0, w);
          float4* dst = reinterpret_cast<float4*>(s_xw + (c * PW + pw) * 8);
          dst[0] = make_float4(w[0], w[1], w[2], w[3]);
          dst[1] = make_float4(w[4], w[5], w[6], w[7]);
        }
        const unsigned bal = __ballot_sync(0xffffffffu, m != 0u);
        const unsigned seg = P2x == 32 ? bal : ((bal >> (cl * P2x)) & ((1u << P2x) - 1u));
        if (m) s_xl[c * PW + __popc(seg & ((1u << pw) - 1u))] = make_int2(pw * gs_w, (int)((((uint32_t)(c * PW + pw) * 8u) << 8) | m));
        if (cval && pw == 0) s_cnb[c] = (unsigned char)__popc(seg);
      }
      __syncwarp();

      // ---- (C) work list over the rows, consumed through the cp.async ring --------------------------
      // builder: lane c owns candidate c; cursor = (remaining ph bits of the row, next entry of xl[c])
      int r = rb;
      const int nbl = lane < ncand ? (int)s_cnb[lane] : 0;
      const int goffc = lane < ncand ? s_cgoff[lane] : 0;
      unsigned ym = (nbl && r < rb + nr) ? s_yph[lane * 8 + r] : 0u;
      int e = 0;
      int rdone = rb;             // rows below rdone are finished (stored, or kept for the next batch)
      while (rdone < rb + nr) {
        int nitems = 0;
        while (r < rb + nr) {
          const int remc = __popc(ym) * nbl - e;
          int incl = remc;
#pragma unroll
          for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += o;
          }
          const int total = __shfl_sync(0xffffffffu, incl, 31);
          const int space = kWorkCap - nitems;
          const int start = incl - remc;
          const int nem = min(remc, space - start);
          if (nem > 0) {
            const float* ywp = s_yw + (lane * 8 + r) * PH;
            const int2* xl = s_xl + lane * PW;
            const int at = nitems + start;
            for (int i = 0; i < nem; ++i) {
              const int ph = __ffs(ym) - 1;
              const int2 xe = xl[e];
              const float wy = ywp[ph];
              const float* xw = s_xw + ((uint32_t)xe.y >> 8);
              const float4 xa = *reinterpret_cast<const float4*>(xw), xb = *reinterpret_cast<const float4*>(xw + 4);
              work_hd[at + i] = make_int2(goffc + ph * gs_h + xe.x, xe.y & 0xff);
              work_wa[at + i] = make_float4(wy * xa.x, wy * xa.y, wy * xa.z, wy * xa.w);
              work_wb[at + i] = make_float4(wy * xb.x, wy * xb.y, wy * xb.z, wy * xb.w);
              if (++e == nbl) { e = 0; ym &= ym - 1; }
            }
          }
          if (total > space) { nitems = kWorkCap; break; }   // flush, then go on with this row
          nitems += total;
          s_rowend[r - rb] = nitems;                        // row complete
          ++r;
          ym = (nbl && r < rb + nr) ? s_yph[lane * 8 + r] : 0u;
          e = 0;
        }
        __syncwarp();
        // consume: item t is FMA'd while items t+1 .. t+kRing-1 are in flight; its header and weights
        // are read one item ahead
#pragma unroll 1
        for (int t = 0; t < kRing - 1; ++t) {
          if (t < nitems) prefetch(work_hd[t].x, t);
          cp_async_commit();
        }
        int t = 0, slot = 0, pslot = kRing - 1;
        int2 hd = work_hd[0];
        float4 wa = work_wa[0], wb = work_wb[0];
        for (int rr = rdone; rr <= r && rr < rb + nr; ++rr) {
          const int tend = rr < r ? s_rowend[rr - rb] : nitems;
#pragma unroll 1
          for (; t < tend; ++t) {
            if (t + kRing - 1 < nitems) prefetch(work_hd[t + kRing - 1].x, pslot);
            cp_async_commit();
            cp_async_wait<kRing - 1>();
            const unsigned char* stage = ring_rd + slot * kStage;
            const float4 vA = SV::read(stage), vB = SV::read(stage + 32 * SV::kBytes);
            const int2 hd_n = work_hd[t + 1];
            const float4 wa_n = work_wa[t + 1], wb_n = work_wb[t + 1];
            slot = slot + 1 == kRing ? 0 : slot + 1;
            pslot = pslot + 1 == kRing ? 0 : pslot + 1;
            if (hd.y & 0x0f) {
              strip_fma(acc[0][0], wa.x, vA); strip_fma(acc[0][1], wa.x, vB);
              strip_fma(acc[1][0], wa.y, vA); strip_fma(acc[1][1], wa.y, vB);
              strip_fma(acc[2][0], wa.z, vA); strip_fma(acc[2][1], wa.z, vB);
              strip_fma(acc[3][0], wa.w, vA); strip_fma(acc[3][1], wa.w, vB);
            }
            if (hd.y & 0xf0) {
              strip_fma(acc[4][0], wb.x, vA); strip_fma(acc[4][1], wb.x, vB);
              strip_fma(acc[5][0], wb.y, vA); strip_fma(acc[5][1], wb.y, vB);
              strip_fma(acc[6][0], wb.z, vA); strip_fma(acc[6][1], wb.z, vB);
              strip_fma(acc[7][0], wb.w, vA); strip_fma(acc[7][1], wb.w, vB);
            }
            hd = hd_n; wa = wa_n; wb = wb_n;
          }
          if (rr < r) {   // every item of row rr (of this batch) is in
            if (npy > 1) { store_row(rr, accumulate || batch > 0); zero_acc(); }
            else if (last) store_row(rr, accumulate != 0);
            rdone = rr + 1;
          }
        }
        cp_async_wait<0>();
        __syncwarp();   // the work list is rewritten by the next flush
      }
      if (last) break;
      ++batch;
    }
  }
}

// Launch plan; RAF_ERR_UNSUPPORTED when the arguments are outside the kernel's range (decided on the
// host before anything is launched).
struct StripPlan {
  StripLevels sl;
  unsigned grid;
  size_t smem;
  int NC;
};

#ifndef RAF_STRIP_MINTILES
#define RAF_STRIP_MINTILES 128
#endif

static int strip_plan(const LevelsParam& lv, const RoiArgs& a, const int64_t* gs, size_t esz, StripPlan* pl) {
  StripLevels& t = pl->sl;
  if (a.sampling_ratio < 0 || a.PH > 32 || a.PW > 32) return RAF_ERR_UNSUPPORTED;
  memset(&t, 0, sizeof(t));
  t.L = lv.L; t.N = lv.n; t.C = lv.c;
  t.chunks = (lv.c + 255) / 256;
  int mintiles = RAF_STRIP_MINTILES;
#ifdef RAF_EXPERIMENT
  if (const char* e = getenv("RAF_TUNE_MINTILES")) mintiles = atoi(e);
#endif
  int64_t total = 0;
  for (int i = 0; i < lv.L; ++i) {
    const int l = lv.L - 1 - i;  // coarsest level first
    t.order[i] = l;
    t.data[l] = const_cast<void*>(lv.data[l]);
    t.sn[l] = lv.sn[l];
    if (lv.sh[l] >= ((int64_t)1 << 31) || lv.sw[l] >= ((int64_t)1 << 31)) return RAF_ERR_UNSUPPORTED;
    t.sh[l] = (int32_t)lv.sh[l]; t.sw[l] = (int32_t)lv.sw[l];
    t.h[l] = lv.h[l]; t.w[l] = lv.w[l];
    t.tiles_x[l] = (lv.w[l] + kStripCols - 1) / kStripCols;
    int th = kStripMaxRows;   // dense coarse levels get short tiles: more, shorter warp tiles where the RoIs pile up
    while (th > 1 && (int64_t)((lv.h[l] + th - 1) / th) * t.tiles_x[l] < mintiles) th >>= 1;
#ifdef RAF_EXPERIMENT
    if (const char* e = getenv("RAF_TUNE_TH")) { if ((int)strlen(e) > 2 * l) th = e[2 * l] - '0'; }   // e.g. "8,4,2,1"
#endif
    t.th[l] = th;
    t.start[i] = (int32_t)total;
    total += (int64_t)((lv.h[l] + th - 1) / th) * t.tiles_x[l];
  }
  for (int i = lv.L; i <= kMaxLevels; ++i) t.start[i] = (int32_t)total;
  const int64_t wtiles = total * lv.n * t.chunks;
  // 32-bit offset arithmetic inside the kernel: grad_out and every image of a level must fit
  const int64_t span = (int64_t)a.K * gs[0] + (int64_t)a.PH * gs[2] + (int64_t)a.PW * gs[3] + lv.c;
  if (wtiles >= ((int64_t)1 << 31) - 64 || span >= ((int64_t)1 << 31)) return RAF_ERR_UNSUPPORTED;
  for (int l = 0; l < lv.L; ++l)
    if ((int64_t)lv.w[l] * lv.sw[l] + (int64_t)kStripMaxRows * lv.sh[l] >= ((int64_t)1 << 31)) return RAF_ERR_UNSUPPORTED;
  t.total = (int32_t)wtiles;
  // RoIs per batch: the dense weight tables of a batch live in the warp's shared memory
  const int P = a.PH > a.PW ? a.PH : a.PW;
  int NC = P <= 8 ? 16 : (P <= 16 ? 8 : 4);
#ifdef RAF_EXPERIMENT
  if (const char* e = getenv("RAF_TUNE_NC")) NC = atoi(e);
#endif
  pl->NC = NC;
  pl->smem = kStripWarps * strip_warp_smem(NC, a.PH, a.PW, esz);
  pl->grid = (unsigned)((wtiles + kStripWarps - 1) / kStripWarps);
  return RAF_OK;
}

int strip_eligible(const LevelsParam& glv, raf_dtype gout_dtype, const RoiArgs& a, const int64_t* gout_strides) {
  StripPlan pl;
  return strip_plan(glv, a, gout_strides, gout_dtype == RAF_F32 ? 4 : 2, &pl);
}

template <typename T, typename G>
static int strip_typed(const LevelsParam& lv, const RoiArgs& a, const void* gout, const int64_t* gs,
                       const PullPrepOut& prep, int accumulate, cudaStream_t stream) {
  StripPlan pl;
  const int rc = strip_plan(lv, a, gs, sizeof(T), &pl);
  if (rc) return rc;
  const T* g = reinterpret_cast<const T*>(gout);
#define RAF_LAUNCH_STRIP(FULL)                                                                                   \
  do {                                                                                                           \
    if (pl.smem > 48 * 1024 &&                                                                                   \
        cudaFuncSetAttribute(bwd_strip_kernel<T, G, FULL>, cudaFuncAttributeMaxDynamicSharedMemorySize,          \
                             (int)pl.smem) != cudaSuccess)                                                       \
      return RAF_ERR_CUDA;                                                                                       \
    bwd_strip_kernel<T, G, FULL><<<pl.grid, 32 * kStripWarps, pl.smem, stream>>>(                                \
        pl.sl, a, g, (int)gs[0], (int)gs[2], (int)gs[3], prep.hdr, prep.bperm, prep.boff, prep.bwin, prep.bgeo,  \
        pl.NC, accumulate, prep.fp);                                                                             \
  } while (0)
  if (lv.c % 256 == 0) RAF_LAUNCH_STRIP(true);
  else RAF_LAUNCH_STRIP(false);
#undef RAF_LAUNCH_STRIP
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

// grad_dtype: RAF_F32, or the 16-bit type of grad_out (checked by the caller).
int launch_backward_strip(const LevelsParam& glv, raf_dtype gout_dtype, raf_dtype grad_dtype, const RoiArgs& a, const void* grad_out,
                          const int64_t* gout_strides, const PullPrepOut& prep, int accumulate, cudaStream_t stream) {
  const bool g32 = grad_dtype == RAF_F32;
  switch (gout_dtype) {
    case RAF_F32: return strip_typed<float, float>(glv, a, grad_out, gout_strides, prep, accumulate, stream);
    case RAF_F16: return g32 ? strip_typed<__half, float>(glv, a, grad_out, gout_strides, prep, accumulate, stream)
                             : strip_typed<__half, __half>(glv, a, grad_out, gout_strides, prep, accumulate, stream);
    case RAF_BF16: return g32 ? strip_typed<__nv_bfloat16, float>(glv, a, grad_out, gout_strides, prep, accumulate, stream)
                              : strip_typed<__nv_bfloat16, __nv_bfloat16>(glv, a, grad_out, gout_strides, prep, accumulate, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
