// raf_backward_pull.cu -- K3d: deterministic PULL formulation of the RoIAlign backward
// (reading S12; H5: the backward's bytes are the gradient pyramid).
//
// Instead of scattering every tap with atomics into a zero-filled pyramid, every CTA OWNS a tile of
// the gradient pyramid -- (image n, level l, 8 rows x 8 columns, a chunk of 256 channels) -- sums
// everything that lands in it in registers, and writes each element exactly once (zero where
// nothing lands).  No memset, no atomics, every fp32 gradient element written once = the
// algorithmic byte count; the summation order is fixed (RoIs of the tile's (level, image) bucket in
// ascending k, taps in table order), so two runs give identical bits.
//
// The operator is separable: for RoI k, pixel (y, x),
//   g[y][x] += sum_{(ph,wy) in Y_k(y)} sum_{(pw,wx) in X_k(x)}  wy * wx * gout[k][ph][pw]
// where Y_k(y) lists the output-bin rows with a sample tap on pixel row y (weights of the same
// bin and pixel merged, 1/count folded in) and X_k(x) likewise for columns.  Those per-RoI, per-axis
// TAP TABLES are built once per call by the prep blocks (raf_pull_prep.cuh: same canonical fp32
// coordinates and weights as the forward) and live in the workspace (L2 resident: 448 B per RoI).
// The prep work -- stable (level, image) bucketing, a conservative pixel window per RoI, the tap
// tables -- runs either as pull_prep_kernel or, with RAF_REUSE_PREP, in the leading blocks of the
// forward launch.
//
// bwd_pull_kernel, per tile (TH x 8 pixels, TH = 8 on large levels, smaller on small dense ones):
//  (A) 256 threads test 512 bucket windows (bwin, bucket order) against the tile in one round trip
//      and keep the RoIs that meet it (ballot compaction, order preserved);
//  (B) per pass of <= 16 candidates, one warp per candidate holds the RoI's taps in its lanes and
//      ballots them against the tile's rows and columns: shared memory gets, per (candidate, row)
//      and (candidate, column), an ENTRY -- the premultiplied grad_out offset of the first bin with a
//      tap there, the weights of the first two (three) consecutive bins, the bin count -- and the
//      ballot masks for the (rarer) longer lists; then, lanes = pixels, one byte per (pixel,
//      candidate): no contribution / served by the entries / walk the masks;
//  (C) warp w owns pixel (i, (w + i) % 8) of every tile row i (one pixel per row and column: the
//      warps of a CTA carry about the same load); one pixel at a time, lanes spread over the 256
//      channels (two float4 accumulators per lane = 8 registers of state, 64 registers total, 4
//      CTAs per SM): a ballot over those bytes gives the candidates that hit the pixel; each hit =
//      two 16-byte shared loads (row entry, column entry), whose product gives up to 2 x 2 (3 x 3)
//      (offset, wy * wx) pairs, and two 128-bit grad_out loads + 8 FFMA per pair.  (An earlier
//      version expanded the pairs into a 34 KB table per CTA in (B); building them in the hit loop
//      instead leaves that shared memory to L1 -- 7 KB per CTA -- and is faster: config 2 backward
//      87.3 -> 85.9 us, config 4 84.2 -> 81.0 us.)  Candidates with longer lists (bins narrower
//      than half a pixel) walk the ballot masks instead (exact).  Tiles with more than 16
//      candidates take several passes, the partial sums parked in the gradient tensor itself.
// Tiles of the coarsest level are scheduled first (most RoIs per pixel).
#include "raf_device.cuh"
#include "raf_host.h"
#include "raf_pull_prep.cuh"

namespace raf {

constexpr int kPullThreads = 256;
constexpr int kTW = 8;   // tile columns (register accumulators per thread)
constexpr int kTH = 8;   // tile rows = warps per CTA

struct PullTiles {
  int32_t order[kMaxLevels];      // level processed at position i (coarsest first)
  int32_t start[kMaxLevels + 1];  // first block of position i
  int32_t tiles_y[kMaxLevels], tiles_x[kMaxLevels];
  int32_t th[kMaxLevels];         // tile rows of the level (1, 2, 4 or 8): small (dense) levels get
                                  // short tiles = more CTAs per RoI-heavy area, shorter critical path
  int32_t chunks;                 // channel chunks of 256
};

__global__ void __launch_bounds__(kPrepThreads, 1)
pull_prep_kernel(const LevelsParam lv, const RoiArgs a, const PullPrepOut o) {
  extern __shared__ int s_prep[];
  pull_prep_block(lv, a, o, (int)blockIdx.x, s_prep);
}

size_t bucket_smem_bytes(int L, int N) { return (size_t)(kPrepThreads / 32 + 1) * ((size_t)L * N + 1) * sizeof(int); }

int launch_pull_prep(const LevelsParam& lv, const RoiArgs& a, const PullPrepOut& prep, cudaStream_t stream) {
  const size_t smem = bucket_smem_bytes(lv.L, lv.n);
  if (smem > 200 * 1024) return RAF_ERR_UNSUPPORTED;
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(pull_prep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return RAF_ERR_CUDA;
  PullPrepOut o = prep;
  o.nblocks = pull_prep_blocks(a, kPrepThreads);
  pull_prep_kernel<<<(unsigned)o.nblocks, kPrepThreads, smem, stream>>>(lv, a, o);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

// ---------------------------------------------------------------------------------------------
// 8 channels of grad_out per lane as two float4 accumulands, 128 channels apart: every warp-wide
// access (16-byte fp32 / 8-byte 16-bit loads, 16-byte fp32 stores) covers contiguous bytes.
// chA / chB = channel of .x of the first / second float4.
// ---------------------------------------------------------------------------------------------
template <typename T> __device__ __forceinline__ float4 ldg4(const T* p);
template <> __device__ __forceinline__ float4 ldg4<float>(const float* p) {
  return __ldg(reinterpret_cast<const float4*>(p));
}
template <> __device__ __forceinline__ float4 ldg4<__half>(const __half* p) {
  const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
  const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
  return make_float4(a.x, a.y, b.x, b.y);
}
template <> __device__ __forceinline__ float4 ldg4<__nv_bfloat16>(const __nv_bfloat16* p) {
  const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
  return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u),
                     __uint_as_float(r.y << 16), __uint_as_float(r.y & 0xffff0000u));
}

// Raw (unconverted) 4-channel loads: the 16-bit types are widened at the use, after all loads of a hit are issued.
template <typename T> struct Raw4;
template <> struct Raw4<float> {
  typedef float4 type;
  static __device__ __forceinline__ float4 load(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
  static __device__ __forceinline__ float4 widen(const float4& r) { return r; }
};
template <> struct Raw4<__half> {
  typedef uint2 type;
  static __device__ __forceinline__ uint2 load(const __half* p) { return __ldg(reinterpret_cast<const uint2*>(p)); }
  static __device__ __forceinline__ float4 widen(const uint2& r) {
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
    const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
    return make_float4(a.x, a.y, b.x, b.y);
  }
};
template <> struct Raw4<__nv_bfloat16> {
  typedef uint2 type;
  static __device__ __forceinline__ uint2 load(const __nv_bfloat16* p) { return __ldg(reinterpret_cast<const uint2*>(p)); }
  static __device__ __forceinline__ float4 widen(const uint2& r) {
    return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u),
                       __uint_as_float(r.y << 16), __uint_as_float(r.y & 0xffff0000u));
  }
};

template <typename T> struct Gout8 {
  static constexpr int kChunk = 256;
  static __device__ __forceinline__ void channels(int lane, int& chA, int& chB) { chA = lane * 4; chB = 128 + lane * 4; }
  static __device__ __forceinline__ void load(const T* p, int chA, int chB, bool actA, bool actB, float4& a, float4& b) {
    a = actA ? ldg4<T>(p + chA) : make_float4(0.f, 0.f, 0.f, 0.f);
    b = actB ? ldg4<T>(p + chB) : make_float4(0.f, 0.f, 0.f, 0.f);
  }
};

// acc += w * v on 4 channels: two packed fp32x2 FMAs (sm_100; each half rounds exactly like fmaf)
__device__ __forceinline__ void fma4(float4& acc, float w, const float4& v) {
#ifndef RAF_NO_FFMA2
  const float2 ww = make_float2(w, w);
  const float2 lo = __ffma2_rn(ww, make_float2(v.x, v.y), make_float2(acc.x, acc.y));
  const float2 hi = __ffma2_rn(ww, make_float2(v.z, v.w), make_float2(acc.z, acc.w));
  acc = make_float4(lo.x, lo.y, hi.x, hi.y);
#else
  acc.x = fmaf(w, v.x, acc.x); acc.y = fmaf(w, v.y, acc.y);
  acc.z = fmaf(w, v.z, acc.z); acc.w = fmaf(w, v.w, acc.w);
#endif
}

// The NP (offset, weight) pairs of one hit as ONE basic block: every load is issued before the first FMA waits, so a
// hit exposes one memory latency, not one per pair (with a branch per pair the compiler keeps each pair's FMAs right
// behind its loads).  Summation order = pair order, as everywhere.
template <typename T, int NP>
__device__ __forceinline__ void hit_pairs(const T* goutA, int dAB, const int (&o)[4], const float (&w)[4], float4& accA, float4& accB) {
  typedef Raw4<T> R;
  typename R::type ra[NP], rb[NP];
#pragma unroll
  for (int i = 0; i < NP; ++i) { const T* q = goutA + o[i]; ra[i] = R::load(q); rb[i] = R::load(q + dAB); }
#pragma unroll
  for (int i = 0; i < NP; ++i) { fma4(accA, w[i], R::widen(ra[i])); fma4(accB, w[i], R::widen(rb[i])); }
}

#ifndef RAF_PULL_NC
#define RAF_PULL_NC 16
#endif
#ifndef RAF_PULL_MINB
#define RAF_PULL_MINB 4
#endif
constexpr int kNC = RAF_PULL_NC;   // candidates per build/consume pass
constexpr int kMaxTapChunks = 4;   // <= 128 taps per axis (eligibility checked on the host)
constexpr uint32_t kOffMask = 0x00ffffffu;

// Up to three entries of a (candidate, row) or (candidate, column): the bins with a tap on one pixel row /
// column are consecutive, so the entry is the element offset of the FIRST bin into grad_out (bin * stride,
// premultiplied, 24 bits), the weights of the first three bins, and the total entry count in m0's top
// byte (255 also when the bins turn out not to be consecutive).  More than three entries (bins narrower
// than about two thirds of a pixel) are served from the ballot masks.
struct __align__(16) PullInfo {
  uint32_t m0;   // off0 | count << 24
  float w0, w1, w2;
};

// kThree: also serve rows / columns with THREE consecutive bins from the entries (outputs finer than the
// pixel grid, e.g. 14 x 14 mask-head bins: config 4 backward 97.6 -> 90.9 us; on 7 x 7 outputs the extra
// code in the hit loop costs more than it saves: 87.7 -> 93.0 us, so it is off there).  With kThree the
// loads of a hit are also issued as a block before its FMAs (hit_pairs: 90.2 -> 84.1 us on config 4; the
// same grouping on 7 x 7 outputs is SLOWER, 87.1 -> 92.7 us -- profiles/r2_experiments.md -- and stays off).
template <typename T, typename G, bool kFull, bool kThree>
__global__ void __launch_bounds__(kPullThreads, RAF_PULL_MINB)
bwd_pull_kernel(const LevelsParam lv, const RoiArgs a, const T* __restrict__ gout, int gs_k,
                int gs_h, int gs_w, const uint32_t* __restrict__ hdr, const int32_t* __restrict__ bperm,
                const int32_t* __restrict__ boff, const int4* __restrict__ bwin,
                const PullTap* __restrict__ taps, const PullTiles tiles, int accumulate, const PrepFingerprint fp) {
  __shared__ int s_k[2 * kPullThreads];
  __shared__ int s_wcount[2 * kPullThreads / 32];
  __shared__ int s_goff[kNC];                          // k * gs_k
  __shared__ PullInfo s_info[kNC][16];                 // [c][0..7] rows, [c][8..15] columns
  __shared__ unsigned char s_pc[64][kNC];              // per (pixel, candidate): 0 no contribution, 1 from the entries, 255 walk the masks
  extern __shared__ uint32_t s_mask[];                 // [kNC][16][nq]

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int slots = 2 * a.sampling_ratio;
  const int nty = a.PH * slots, ntx = a.PW * slots;
  const int nq = (max(nty, ntx) + 31) >> 5;

  // ---- decode the tile: blockIdx.y = tile within the pyramid (coarsest level first),
  //      blockIdx.x = image * chunks + chunk (fastest, so heavy tiles of all images start first)
  int pos = 0;
  while (pos + 1 < lv.L && (int)blockIdx.y >= tiles.start[pos + 1]) ++pos;
  const int level = tiles.order[pos];
  const int trem = blockIdx.y - tiles.start[pos];
  const int tyi = trem / tiles.tiles_x[level], txi = trem - tyi * tiles.tiles_x[level];
  const int n = blockIdx.x / tiles.chunks, chunk = blockIdx.x - n * tiles.chunks;
  const int H = lv.h[level], W = lv.w[level];
  const int TH = tiles.th[level];
  const int y0 = tyi * TH, x0 = txi * kTW;
  const int y1 = min(y0 + TH, H) - 1, x1 = min(x0 + kTW, W) - 1;  // inclusive
  const int chA = chunk * 256 + lane * 4, chB = chA + 128;
  const bool actA = kFull || chA < lv.c, actB = kFull || chB < lv.c;
  // inactive lanes read channel 0 (valid memory) and never store: no predicates in the hot loop
  const T* goutA = gout + (actA ? chA : 0);
  const int dAB = kFull ? 128 : (actB ? chB : 0) - (actA ? chA : 0);
  const int sw = (int)lv.sw[level];
  const int sh = (int)lv.sh[level];
  G* gtile = reinterpret_cast<G*>(const_cast<void*>(lv.data[level])) + (int64_t)n * lv.sn[level] +
                 (int64_t)y0 * sh + (int64_t)x0 * sw + chA;
  const int npx = x1 - x0 + 1, npy = y1 - y0 + 1;

  const int key = level * lv.n + n;
  const int bbeg = __ldg(boff + key), bend = __ldg(boff + key + 1);
  // The workspace must hold the tables of exactly these arguments (RAF_REUSE_PREP contract): every warp
  // compares the fingerprint the prep left (same round trip as the bucket range); on a mismatch the
  // tile is poisoned with NaN instead of being computed from foreign tables.
  {
    const bool bad = lane < 8 && __ldg(hdr + lane) != fp.v[lane & 7];
    if (__any_sync(0xffffffffu, bad)) {
      const float qnan = __int_as_float(0x7fc00000);
      const float4 q4 = make_float4(qnan, qnan, qnan, qnan);
      for (int i = 0; i < npy; ++i) {
        const int j = (warp + i) & 7;
        if (j >= npx) continue;
        G* gp = gtile + i * sh + j * sw;
        if (actA) Grad4<G>::store(gp, q4);
        if (actB) Grad4<G>::store(gp + 128, q4);
      }
      return;   // (uniform over the CTA: every warp sees the same words)
    }
  }
  int npass = 0;

  for (int s0 = bbeg; s0 < bend; s0 += 2 * kPullThreads) {
    // ---- (A) candidates of this scan chunk (512 bucket entries, two per thread, all loads issued
    //      together), order preserved ------------------------------------------------------------
    const int ia = s0 + tid, ib = s0 + kPullThreads + tid;
    int4 wa = make_int4(0x7fffffff, -1, 0x7fffffff, -1), wb = wa;
    int ka = 0, kb = 0;
    if (ia < bend) { wa = __ldg(bwin + ia); ka = __ldg(bperm + ia); }   // {ymin, ymax, xmin, xmax}, conservative
    if (ib < bend) { wb = __ldg(bwin + ib); kb = __ldg(bperm + ib); }
    const bool hita = (wa.x <= y1) && (wa.y >= y0) && (wa.z <= x1) && (wa.w >= x0);
    const bool hitb = (wb.x <= y1) && (wb.y >= y0) && (wb.z <= x1) && (wb.w >= x0);
    const unsigned ma = __ballot_sync(0xffffffffu, hita), mb = __ballot_sync(0xffffffffu, hitb);
    if (lane == 0) { s_wcount[warp] = __popc(ma); s_wcount[kPullThreads / 32 + warp] = __popc(mb); }
    __syncthreads();
    int befa = 0, befb = 0, ncand = 0;
#pragma unroll
    for (int w = 0; w < 2 * kPullThreads / 32; ++w) {
      const int cnt = s_wcount[w];
      if (w < warp) befa += cnt;
      if (w < kPullThreads / 32 + warp) befb += cnt;
      ncand += cnt;
    }
    if (hita) s_k[befa + __popc(ma & ((1u << lane) - 1u))] = ka;
    if (hitb) s_k[befb + __popc(mb & ((1u << lane) - 1u))] = kb;
    __syncthreads();

    for (int p0 = 0; p0 < ncand; p0 += kNC) {
      const int nc = min(kNC, ncand - p0);
      // ---- (B) tables of this pass: warp per candidate, lanes = taps ---------------------------
      for (int c = warp; c < nc; c += kPullThreads / 32) {
        const int k = s_k[p0 + c];
        const PullTap* ty = taps + (int64_t)k * (nty + ntx);
        const PullTap* tx = ty + nty;
        int cnt = 0, e0 = -1, e1 = -1, e2 = -1;   // lanes 0..7: row `lane`; lanes 8..15: column `lane - 8`
        for (int q = 0; q < nq; ++q) {
          const int t = q * 32 + lane;
          const int rely = (t < nty) ? (int)(__ldg(&ty[t].pb) & kPixMask) - y0 : -1;
          const int relx = (t < ntx) ? (int)(__ldg(&tx[t].pb) & kPixMask) - x0 : -1;
          unsigned mine = 0;
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const unsigned my = __ballot_sync(0xffffffffu, rely == i);
            const unsigned mx = __ballot_sync(0xffffffffu, relx == i);
            if (lane == i) mine = my;
            if (lane == 8 + i) mine = mx;
          }
          if (lane < 16) {
            s_mask[(c * 16 + lane) * nq + q] = mine;
            cnt += __popc(mine);
            if (e0 < 0 && mine) { e0 = q * 32 + __ffs(mine) - 1; mine &= mine - 1; }
            if (e1 < 0 && mine) { e1 = q * 32 + __ffs(mine) - 1; mine &= mine - 1; }
            if (kThree && e2 < 0 && mine) e2 = q * 32 + __ffs(mine) - 1;
          }
        }
        if (lane < 16) {
          const PullTap* tb = lane < 8 ? ty : tx;
          const uint32_t stride = (uint32_t)(lane < 8 ? gs_h : gs_w);
          PullInfo inf;
          inf.m0 = 0; inf.w0 = 0.0f; inf.w1 = 0.0f; inf.w2 = 0.0f;
          if (e0 >= 0) {
            const PullTap e = tb[e0];
            const uint32_t bin0 = e.pb >> 24;
            int c8 = min(cnt, 255);
            inf.w0 = e.w;
            if (e1 >= 0) {
              const PullTap f = tb[e1];
              inf.w1 = f.w;
              if ((f.pb >> 24) != bin0 + 1) c8 = 255;   // not consecutive (degenerate box): walk the masks
            }
            if (e2 >= 0) {
              const PullTap f = tb[e2];
              inf.w2 = f.w;
              if ((f.pb >> 24) != bin0 + 2) c8 = 255;
            }
            inf.m0 = (bin0 * stride) | ((uint32_t)c8 << 24);
          }
          s_info[c][lane] = inf;
        }
        if (lane == 0) s_goff[c] = k * gs_k;
        __syncwarp();
        // lanes = pixels now: does candidate c land on the pixel, and can its entries serve it?
        for (int p = lane; p < 8 * npy; p += 32) {
          const uint32_t cy = s_info[c][p >> 3].m0 >> 24, cx = s_info[c][8 + (p & 7)].m0 >> 24;
          s_pc[p][c] = (cy == 0 || cx == 0) ? 0 : ((cy > (kThree ? 3 : 2) || cx > (kThree ? 3 : 2)) ? 255 : 1);
        }
      }
      __syncthreads();

      // ---- (C) consume: warp w takes pixel (row i, column (w + i) % 8) for every tile row i: one
      //      pixel of every row and (for 8-row tiles) of every column, so the warps of a CTA carry
      //      about the same load; one pixel at a time, lanes = channels -------------------------
      for (int i = 0; i < npy; ++i) {
        const int j = (warp + i) & 7;
        if (j >= npx) continue;
        const int p = i * 8 + j;
        G* gp = gtile + i * sh + j * sw;
        float4 accA = make_float4(0.f, 0.f, 0.f, 0.f), accB = accA;
        if (accumulate || npass) {
          if (actA) accA = Grad4<G>::load(gp);
          if (actB) accB = Grad4<G>::load(gp + 128);
        }
        // pair count of every candidate on this pixel: lane c holds candidate c's
        const unsigned pcv = (lane < nc) ? s_pc[p][lane] : 0u;
        unsigned mm = __ballot_sync(0xffffffffu, pcv != 0);
        while (mm) {
          const int c = __ffs(mm) - 1;
          mm &= mm - 1;
          const unsigned np = __shfl_sync(0xffffffffu, pcv, c);
          if (np != 255u) {   // (row entries) x (column entries) of the pixel, straight from the tables of (B)
            const PullInfo iy = s_info[c][i], ix = s_info[c][8 + j];
            const int cy = (int)(iy.m0 >> 24), cx = (int)(ix.m0 >> 24);
            const int o00 = s_goff[c] + (int)(iy.m0 & kOffMask) + (int)(ix.m0 & kOffMask);
            if (kThree) {
              for (int ai = 0; ai < cy; ++ai) {   // one bin row (up to three bins) per round, its loads issued as a block
                const float wy = ai == 0 ? iy.w0 : (ai == 1 ? iy.w1 : iy.w2);
                const int oy = o00 + ai * gs_h;
                const int o[4] = {oy, oy + gs_w, oy + 2 * gs_w, 0};
                const float w[4] = {wy * ix.w0, wy * ix.w1, wy * ix.w2, 0.0f};
                switch (cx) {
                  case 1: hit_pairs<T, 1>(goutA, dAB, o, w, accA, accB); break;
                  case 2: hit_pairs<T, 2>(goutA, dAB, o, w, accA, accB); break;
                  default: hit_pairs<T, 3>(goutA, dAB, o, w, accA, accB); break;
                }
              }
            } else {   // order (y0,x0) (y0,x1) (y1,x0) (y1,x1)
              const T* q = goutA + o00;
              { const float w = iy.w0 * ix.w0; fma4(accA, w, ldg4<T>(q)); fma4(accB, w, ldg4<T>(q + dAB)); }
              if (cx > 1) { const float w = iy.w0 * ix.w1; fma4(accA, w, ldg4<T>(q + gs_w)); fma4(accB, w, ldg4<T>(q + gs_w + dAB)); }
              if (cy > 1) {
                const T* q1 = q + gs_h;
                { const float w = iy.w1 * ix.w0; fma4(accA, w, ldg4<T>(q1)); fma4(accB, w, ldg4<T>(q1 + dAB)); }
                if (cx > 1) { const float w = iy.w1 * ix.w1; fma4(accA, w, ldg4<T>(q1 + gs_w)); fma4(accB, w, ldg4<T>(q1 + gs_w + dAB)); }
              }
            }
          } else {   // rare: more than two entries on an axis -> walk the ballot masks
            const int k = s_k[p0 + c];
            const T* gk = goutA + s_goff[c];
            const PullTap* ty = taps + (int64_t)k * (nty + ntx);
            const PullTap* tx = ty + nty;
            for (int qy = 0; qy < nq; ++qy) {
              unsigned my = s_mask[(c * 16 + i) * nq + qy];
              while (my) {
                const PullTap ey = ty[qy * 32 + __ffs(my) - 1];
                my &= my - 1;
                const T* gy = gk + (ey.pb >> 24) * (uint32_t)gs_h;
                for (int qx = 0; qx < nq; ++qx) {
                  unsigned mx = s_mask[(c * 16 + 8 + j) * nq + qx];
                  while (mx) {
                    const PullTap ex = tx[qx * 32 + __ffs(mx) - 1];
                    mx &= mx - 1;
                    const T* q = gy + (ex.pb >> 24) * (uint32_t)gs_w;
                    const float w = ey.w * ex.w;
                    fma4(accA, w, ldg4<T>(q)); fma4(accB, w, ldg4<T>(q + dAB));
                  }
                }
              }
            }
          }
        }
        if (actA) Grad4<G>::store(gp, accA);
        if (actB) Grad4<G>::store(gp + 128, accB);
      }
      ++npass;
      if (p0 + kNC < ncand || s0 + 2 * kPullThreads < bend)
        __syncthreads();  // tables and s_k are rewritten by the next pass / scan chunk
    }
  }

  if (npass == 0 && !accumulate) {   // nothing lands in this tile: zeros
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int i = 0; i < npy; ++i) {
      const int j = (warp + i) & 7;
      if (j >= npx) continue;
      G* gp = gtile + i * sh + j * sw;
      if (actA) Grad4<G>::store(gp, z);
      if (actB) Grad4<G>::store(gp + 128, z);
    }
  }
}

// Launch plan of the pull kernel; RAF_ERR_UNSUPPORTED when the arguments are outside its range
// (decided on the host before anything is launched).
struct PullPlan {
  PullTiles t;
  dim3 grid;
  size_t smem;
};

static int pull_plan(const LevelsParam& lv, const RoiArgs& a, const int64_t* gs, PullPlan* pl) {
  PullTiles& t = pl->t;
  if (a.sampling_ratio <= 0) return RAF_ERR_UNSUPPORTED;
  t.chunks = (lv.c + 255) / 256;
  int64_t total = 0;
  for (int i = 0; i < lv.L; ++i) {
    const int l = lv.L - 1 - i;  // coarsest level first
    t.order[i] = l;
#ifndef RAF_PULL_MINTILES
#define RAF_PULL_MINTILES 64
#endif
    int th = kTH;     // aim for >= RAF_PULL_MINTILES tiles per level and image
    while (th > 1 && (int64_t)lv.h[l] * lv.w[l] < (int64_t)RAF_PULL_MINTILES * th * kTW) th >>= 1;
    t.th[l] = th;
    t.tiles_y[l] = (lv.h[l] + th - 1) / th;
    t.tiles_x[l] = (lv.w[l] + kTW - 1) / kTW;
    t.start[i] = (int32_t)total;
    total += (int64_t)t.tiles_y[l] * t.tiles_x[l];
  }
  t.start[lv.L] = (int32_t)total;
  const int64_t gy = (int64_t)lv.n * t.chunks;
  const int ntaps = 2 * a.sampling_ratio * (a.PH > a.PW ? a.PH : a.PW);
  const int nq = (ntaps + 31) / 32;
  // 32-bit / 24-bit offset arithmetic inside the kernel: grad_out must fit
  const int64_t span = (int64_t)a.K * gs[0] + (int64_t)a.PH * gs[2] + (int64_t)a.PW * gs[3] + lv.c;
  if (total > 65535 || gy >= ((int64_t)1 << 31) || nq > kMaxTapChunks || span >= ((int64_t)1 << 31) ||
      (int64_t)a.PH * gs[2] >= (1 << 24) || (int64_t)a.PW * gs[3] >= (1 << 24))
    return RAF_ERR_UNSUPPORTED;
  for (int l = 0; l < lv.L; ++l)
    if (lv.h[l] >= 0xffffff || lv.w[l] >= 0xffffff ||   // tap tables keep pixel indices in 24 bits
        (int64_t)lv.w[l] * lv.sw[l] + (int64_t)kTH * lv.sh[l] >= ((int64_t)1 << 31))
      return RAF_ERR_UNSUPPORTED;
  pl->smem = sizeof(uint32_t) * kNC * 16 * nq;
  pl->grid = dim3((unsigned)gy, (unsigned)total);
  return RAF_OK;
}

int pull_eligible(const LevelsParam& glv, raf_dtype gout_dtype, const RoiArgs& a, const void* grad_out,
                  const int64_t* gout_strides) {
  (void)gout_dtype; (void)grad_out;
  PullPlan pl;
  return pull_plan(glv, a, gout_strides, &pl);
}

template <typename T, typename G>
static int pull_typed(const LevelsParam& lv, const RoiArgs& a, const void* gout, const int64_t* gs,
                      const PullPrepOut& prep, int accumulate, cudaStream_t stream) {
  PullPlan pl;
  const int rc = pull_plan(lv, a, gs, &pl);
  if (rc) return rc;
  const T* g = reinterpret_cast<const T*>(gout);
  const bool three = a.PH > 8 || a.PW > 8;
#define RAF_LAUNCH_PULL(FULL, THREE)                                                                                      \
  bwd_pull_kernel<T, G, FULL, THREE><<<pl.grid, kPullThreads, pl.smem, stream>>>(lv, a, g, (int)gs[0], (int)gs[2], (int)gs[3], \
                                                                                  prep.hdr, prep.bperm, prep.boff, prep.bwin, \
                                                                                  prep.taps, pl.t, accumulate, prep.fp)
  if (lv.c % 256 == 0) { if (three) RAF_LAUNCH_PULL(true, true); else RAF_LAUNCH_PULL(true, false); }
  else { if (three) RAF_LAUNCH_PULL(false, true); else RAF_LAUNCH_PULL(false, false); }
#undef RAF_LAUNCH_PULL
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

// grad_dtype: RAF_F32, or the 16-bit type of grad_out (checked by the caller).
int launch_backward_pull(const LevelsParam& glv, raf_dtype gout_dtype, raf_dtype grad_dtype, const RoiArgs& a, const void* grad_out,
                         const int64_t* gout_strides, const PullPrepOut& prep, int accumulate, cudaStream_t stream) {
  const bool g32 = grad_dtype == RAF_F32;
  switch (gout_dtype) {
    case RAF_F32: return pull_typed<float, float>(glv, a, grad_out, gout_strides, prep, accumulate, stream);
    case RAF_F16: return g32 ? pull_typed<__half, float>(glv, a, grad_out, gout_strides, prep, accumulate, stream)
                             : pull_typed<__half, __half>(glv, a, grad_out, gout_strides, prep, accumulate, stream);
    case RAF_BF16: return g32 ? pull_typed<__nv_bfloat16, float>(glv, a, grad_out, gout_strides, prep, accumulate, stream)
                              : pull_typed<__nv_bfloat16, __nv_bfloat16>(glv, a, grad_out, gout_strides, prep, accumulate, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
