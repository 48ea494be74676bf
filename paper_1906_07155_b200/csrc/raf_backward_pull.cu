// raf_backward_pull.cu -- K3d: deterministic PULL formulation of the RoIAlign backward
// (reading S12; H5: the backward's bytes are the gradient pyramid).
//
// Instead of scattering every tap with atomics into a zero-filled pyramid, every gradient TILE --
// (image n, level l, 8 rows x 8 columns, a chunk of 128 or 256 channels) -- is owned by one CTA at a
// time, kept whole in registers (a consumer warp = a tile row x 4 columns, a lane = 4 or 8 channels of
// each of those pixels), receives everything that lands in it, and is written exactly once (zero where
// nothing lands).  No memset, no atomics, every fp32 gradient element written once = the algorithmic
// byte count; the summation order is fixed (RoIs of the tile's (level, image) bucket in ascending k,
// bins in ascending order), so two runs give identical bits.
//
// The operator is separable: for RoI k, pixel (y, x),
//   g[y][x] += sum_{ph in Y_k(y)} wy[ph] * sum_{pw in X_k(x)} wx[pw] * gout[k][ph][pw]
// where Y_k(y) is the run of output-bin rows with a sample tap on pixel row y and X_k(x) likewise for
// columns: the INVERSE tap tables the prep builds once per call (raf_pull_prep.cuh; with
// RAF_REUSE_PREP they come out of the forward launch).
//
// bwd_pull_kernel is PERSISTENT (one CTA per SM) and warp-specialised; tiles are handed out heaviest
// first (coarsest level first; three fixed tiles per CTA, then an atomic counter):
//  * SCANNER warps: next tile -> bucket (level, image) -> test up to 512 RoI windows (bwin, bucket
//    order) against the tile in one round trip, ballot-compact the hits in order into a candidate buffer;
//  * LOADER warps: per pass of <= 16 candidates fetch the inverse-table entries of the tile's 8 rows and
//    8 columns (16 threads per candidate), reduce them to the block of bins [pa..pb] x [qa..qb] of
//    grad_out the candidate needs here, pack consecutive blocks into shared-memory STAGES, publish the
//    pass table to the consumers and stream the blocks in with bulk-async copies (TMA: cp.async.bulk +
//    mbarrier complete_tx).  Each grad_out vector crosses L2 -> SM once per tile that needs it, not once
//    per pixel;
//  * CONSUMER warps: wait on a stage's `full` barrier and run, for their pixels, the pair loop (rows of
//    bins x columns of bins) with 128-bit shared loads and FFMAs into the register accumulators, release
//    the stage (`empty` barrier), and store the tile after its last pass.  No global-load latency sits
//    in the consume loop.
// The three roles are decoupled by mbarrier rings (candidate buffers, pass tables, stages), so the
// scan / look-up / copy latencies of the coming tiles overlap the arithmetic of the current one.
#include "raf_device.cuh"
#include "raf_host.h"
#include "raf_pull_prep.cuh"
#include <cstdlib>

#ifndef RAF_COLSPLIT
#define RAF_COLSPLIT 2
#endif
#ifndef RAF_JLOOP
#define RAF_JLOOP 2
#endif
#ifndef RAF_ABLATE
#define RAF_ABLATE 0
#endif
#ifndef RAF_SETMAXNREG
#define RAF_SETMAXNREG 0
#endif
#ifndef RAF_PRODUCER_REGS
#define RAF_PRODUCER_REGS 56
#endif
#ifndef RAF_CONSUMER_REGS
#define RAF_CONSUMER_REGS 104
#endif

namespace raf {

constexpr int kRowWarps = 8;                            // = tile rows
constexpr int kColSplit = RAF_COLSPLIT;                 // consumer warps per tile row (column groups)
constexpr int kConsumerWarps = kRowWarps * kColSplit;
constexpr int kScanThreads = 64;                        // scanner role
constexpr int kLoadWarps = 1;                           // loader role: independent warps
constexpr int kPullThreads = 32 * kConsumerWarps + kScanThreads + 32 * kLoadWarps + 32;   // + the issuer warp
constexpr int kTW = 8;    // tile columns
constexpr int kJW = kTW / kColSplit;   // pixels (accumulator sets) per consumer lane
constexpr int kTH = 8;    // tile rows
constexpr int kNC = 16;   // candidates per pass
constexpr int kNB = 3;    // pass tables in flight
constexpr int kNCB = 4;   // candidate buffers in flight
constexpr int kStages = 4;
constexpr int kScanQ = 8;                               // bucket entries per scanner thread and chunk
constexpr int kScan = kScanQ * kScanThreads;            // bucket entries tested per scan chunk
constexpr int kBoffCache = 512;

struct PullTiles {
  int32_t order[kMaxLevels];      // level processed at position i (coarsest first)
  int32_t start[kMaxLevels + 1];  // first block of position i
  int32_t tiles_y[kMaxLevels], tiles_x[kMaxLevels];
  int32_t chunks;                 // channel chunks per pixel
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

// ---- mbarrier / bulk-async copy (TMA) wrappers ---------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t tx) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(tx) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "RAF_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra RAF_DONE_%=;\n"
      "bra RAF_WAIT_%=;\n"
      "RAF_DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ---- 4 channels of grad_out from a shared-memory stage, widened to fp32 --------------------------
template <typename T> __device__ __forceinline__ float4 lds_quad(const unsigned char* p);
template <> __device__ __forceinline__ float4 lds_quad<float>(const unsigned char* p) {
  return *reinterpret_cast<const float4*>(p);
}
template <> __device__ __forceinline__ float4 lds_quad<__half>(const unsigned char* p) {
  const uint2 r = *reinterpret_cast<const uint2*>(p);
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
  const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
  return make_float4(a.x, a.y, b.x, b.y);
}
template <> __device__ __forceinline__ float4 lds_quad<__nv_bfloat16>(const unsigned char* p) {
  const uint2 r = *reinterpret_cast<const uint2*>(p);
  return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u),
                     __uint_as_float(r.y << 16), __uint_as_float(r.y & 0xffff0000u));
}

template <typename T> __device__ __forceinline__ float4 ldg_quad(const T* p);
template <> __device__ __forceinline__ float4 ldg_quad<float>(const float* p) {
  return __ldg(reinterpret_cast<const float4*>(p));
}
template <> __device__ __forceinline__ float4 ldg_quad<__half>(const __half* p) {
  const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
  const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&r.x));
  const float2 b = __half22float2(*reinterpret_cast<const __half2*>(&r.y));
  return make_float4(a.x, a.y, b.x, b.y);
}
template <> __device__ __forceinline__ float4 ldg_quad<__nv_bfloat16>(const __nv_bfloat16* p) {
  const uint2 r = __ldg(reinterpret_cast<const uint2*>(p));
  return make_float4(__uint_as_float(r.x << 16), __uint_as_float(r.x & 0xffff0000u),
                     __uint_as_float(r.y << 16), __uint_as_float(r.y & 0xffff0000u));
}

__device__ __forceinline__ void fma4(float4& acc, float w, const float4& v) {
  acc.x = fmaf(w, v.x, acc.x); acc.y = fmaf(w, v.y, acc.y);
  acc.z = fmaf(w, v.z, acc.z); acc.w = fmaf(w, v.w, acc.w);
}

// Weight number `idx` of an inverse-table entry with more than kInvW bins on one pixel (bins narrower
// than 2/7 pixel): not stored, evaluated from the RoI geometry (same function as the prep).
__device__ __noinline__ float pull_slow_weight(const LevelsParam& lv, const RoiArgs& a, int k, int axis, int pix, int bin) {
  const RoiOnLevel r = roi_on_level(lv, a, k);
  const int n = axis ? lv.w[r.level] : lv.h[r.level];
  const int g = axis ? r.geo.gw : r.geo.gh;
  bool hit;
  return inv_bin_weight(axis ? r.geo.sx : r.geo.sy, axis ? r.geo.bw : r.geo.bh, bin, g, n,
                        axis ? 1.0f : r.geo.inv_count, pix, hit);
}

// Inverse-table entry of a pixel beyond the stored table (window wider than kInvCap pixels).
__device__ __noinline__ void pull_wide_entry(const LevelsParam& lv, const RoiArgs& a, int k, int axis, int pix,
                                             uint4& e0, uint4& e1) {
  const InvEntry e = inv_entry_compute(lv, a, roi_on_level(lv, a, k), axis, pix);
  e0 = make_uint4(e.meta, __float_as_uint(e.w[0]), __float_as_uint(e.w[1]), __float_as_uint(e.w[2]));
  e1 = make_uint4(__float_as_uint(e.w[3]), __float_as_uint(e.w[4]), __float_as_uint(e.w[5]), __float_as_uint(e.w[6]));
}

// copy_mode: how the producer fills a stage
enum { kCopyRows = 0,    // one bulk copy per row of bins (the chunk is the whole pixel vector and bins are adjacent)
       kCopyBins = 1,    // one bulk copy per bin
       kCopyManual = 2   // the producer's lanes copy with ordinary loads (16-byte alignment not given)
};

__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}

// acc += w * (the lane's Q quads of one bin in a stage)
template <typename T, int Q>
__device__ __forceinline__ void fma_bin(float4 (&acc)[Q], float w, const unsigned char* p) {
#if RAF_ABLATE == 2   // no FFMA: keep the loads alive with one add
#pragma unroll
  for (int q = 0; q < Q; ++q) { const float4 v = lds_quad<T>(p + q * 128 * sizeof(T)); acc[q].x += v.x + v.y + v.z + v.w; }
#elif RAF_ABLATE == 3  // no shared loads
#pragma unroll
  for (int q = 0; q < Q; ++q) fma4(acc[q], w, make_float4(w, 1.f, 2.f, 3.f));
#else
#pragma unroll
  for (int q = 0; q < Q; ++q) fma4(acc[q], w, lds_quad<T>(p + q * 128 * sizeof(T)));
#endif
}

template <int kId, int kCount>
__device__ __forceinline__ void role_sync() { asm volatile("bar.sync %0, %1;" ::"n"(kId), "n"(kCount) : "memory"); }

// Geometry of a work item (tile x image x channel chunk).
struct TileDesc {
  int level, n, chunk;
  int y0, x0, npy, npx;
};
enum { kFirst = 1, kLast = 2, kEnd = 4 };

// scanner -> loader: the RoIs of one scan chunk whose window meets the tile, in bucket order
struct __align__(16) CandBuf {
  TileDesc t;
  int flags;                 // kFirst / kLast scan chunk of the tile, kEnd
  int ncand;
  int pass_base;             // number of the first pass this buffer turns into
  int pad_;
  int k[kScan];
  uint2 win[kScan];          // {ymin | ymax << 16, xmin | xmax << 16}
};

// loader -> consumers: up to kNC candidates of one tile
enum { kNewItem = 1, kChunked = 2 };
struct __align__(16) PassTable {
  TileDesc t;
  int flags;                 // kFirst / kLast pass of the tile, kEnd
  int nc;
  int slow[2];               // != 0: some entry has more than kInvW bins on one pixel
  int k[kNC];                         // RoI index of every candidate
  // pa | pb << 8 | qa << 16 | ncols << 24 (0: nothing lands);  byte offset of the block in its stage;
  // rows of bins per stage item | (kNewItem / kChunked) << 16;  bytes of the stage item this candidate opens
  __align__(16) int blk[kNC][4];
  uint32_t xmeta[kNC][8];             // first bin | count << 8 of the column entries (info[c][8+j].meta is
                                      // rewritten to byte offset in a row of the block | stored weights << 24)
  __align__(16) InvEntry info[kNC][16];   // [c][0..7] tile rows, [c][8..15] tile columns
  // per (candidate, tile row): byte offset of the first row of bins that lands on it, relative to the
  // block | rows << 28 (0, 1, 2; 3 = more: generic loop), its weight, offset and weight of the second
  __align__(16) uint4 rowrec[kNC][8];
};

#ifdef RAF_PROFILE
#define RAF_T0(v) long long v = clock64()
#define RAF_ACC(slot, v) do { prof[slot] += clock64() - (v); } while (0)
#else
#define RAF_T0(v) do {} while (0)
#define RAF_ACC(slot, v) do {} while (0)
#endif

template <typename T, int CPL>
__global__ void __launch_bounds__(kPullThreads, 1)
bwd_pull_kernel(const __grid_constant__ LevelsParam lv, const __grid_constant__ RoiArgs a, const T* __restrict__ gout,
                int gs_k, int gs_h, int gs_w, uint32_t* __restrict__ hdr, const int32_t* __restrict__ bperm,
                const int32_t* __restrict__ boff, const int4* __restrict__ bwin, const InvEntry* __restrict__ inv,
                const __grid_constant__ PullTiles tiles, int accumulate, const __grid_constant__ PrepFingerprint fp,
                int stage_bytes, int copy_mode) {
  constexpr int Q = CPL / 4;           // float4 accumulators per pixel and lane
  constexpr int CH = 32 * CPL;         // channels per work item
  constexpr int kBinBytes = CH * (int)sizeof(T);   // one bin of the chunk in a stage
  __shared__ int s_wcount[kScanQ * kScanThreads / 32];
  __shared__ int s_next[3];
  __shared__ int s_boff[kBoffCache];   // bucket offsets boff[L*N + 1] when they fit (else read from global)
  __shared__ __align__(8) uint64_t s_full[kStages], s_empty[kStages], s_tfull[kNB], s_tempty[kNB], s_cfull[kNCB], s_cempty[kNCB];
  __shared__ int s_stale;
  extern __shared__ __align__(128) unsigned char s_dyn[];   // [stages][pass tables][candidate buffers]
  unsigned char* s_stage = s_dyn;
  PassTable* s_tab = reinterpret_cast<PassTable*>(s_dyn + (size_t)kStages * stage_bytes);
  CandBuf* s_cand = reinterpret_cast<CandBuf*>(s_tab + kNB);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
#ifdef RAF_PROFILE
  long long prof[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const long long prof_start = clock64();
#endif
  const int gx = lv.n * tiles.chunks;                       // work items per tile position
  const int total_items = tiles.start[lv.L] * gx;

  if (tid == 0) {
    uint32_t stale = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) stale |= __ldg(hdr + q) ^ fp.v[q];
    s_stale = stale != 0;
#pragma unroll
    for (int s = 0; s < kStages; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], kConsumerWarps); }
#pragma unroll
    for (int b = 0; b < kNB; ++b) { mbar_init(&s_tfull[b], 1); mbar_init(&s_tempty[b], kConsumerWarps + 1); }
#pragma unroll
    for (int b = 0; b < kNCB; ++b) { mbar_init(&s_cfull[b], kScanThreads); mbar_init(&s_cempty[b], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const bool boff_cached = lv.L * lv.n + 1 <= kBoffCache;
  if (boff_cached)
    for (int q = tid; q <= lv.L * lv.n; q += kPullThreads) s_boff[q] = __ldg(boff + q);
  __syncthreads();
  const bool stale = s_stale != 0;

  // work item t -> tile geometry
  auto decode = [&](int t, TileDesc& d) {
    const int tile = t / gx, x = t - tile * gx;
    int pos = 0;
    while (pos + 1 < lv.L && tile >= tiles.start[pos + 1]) ++pos;
    d.level = tiles.order[pos];
    const int trem = tile - tiles.start[pos];
    const int tyi = trem / tiles.tiles_x[d.level], txi = trem - tyi * tiles.tiles_x[d.level];
    d.n = x / tiles.chunks;
    d.chunk = x - d.n * tiles.chunks;
    d.y0 = tyi * kTH;
    d.x0 = txi * kTW;
    d.npy = min(d.y0 + kTH, lv.h[d.level]) - d.y0;
    d.npx = min(d.x0 + kTW, lv.w[d.level]) - d.x0;
  };

  if (warp == kConsumerWarps + kScanThreads / 32 + kLoadWarps) {
    // ================================== ISSUER WARP ===================================================
    // Walks the pass tables in order (like a consumer) and streams the candidates' blocks of grad_out
    // into the stage ring; the ring order is the order the consumers take the items in.
    if (stale) return;
    int stp = 0;
    uint32_t parp = 0;
    for (int pass = 0;; ++pass) {
      const int b = pass % kNB;
      mbar_wait(&s_tfull[b], (uint32_t)(pass / kNB) & 1u);
      const PassTable& tab = s_tab[b];
      if (tab.flags & kEnd) break;
      const int nc = tab.nc;
      const int ch0 = tab.t.chunk * CH;
      const int cbytes = min(CH, lv.c - ch0) * (int)sizeof(T);   // bytes of a bin that exist in this chunk
      int cur = 0;   // stage of the open item
      for (int c = 0; c < nc; ++c) {
        const int4 blk = *reinterpret_cast<const int4*>(tab.blk[c]);
        const int ncols = (int)((uint32_t)blk.x >> 24);
        if (ncols == 0) continue;
        const int pa = blk.x & 0xff, pb = (blk.x >> 8) & 0xff, qa = (blk.x >> 16) & 0xff;
        const int fl = blk.z >> 16, rpi = blk.z & 0xffff;
        const T* gsrc = gout + (int64_t)tab.k[c] * gs_k + qa * gs_w + ch0;
        for (int r0 = pa; r0 <= pb; r0 += rpi) {
          const int nr = min(rpi, pb - r0 + 1);
          if (fl) {   // this candidate (or chunk) opens a stage item
            cur = stp;
            { RAF_T0(te); if (lane == 0) mbar_wait(&s_empty[cur], parp ^ 1u); RAF_ACC(2, te); }
            __syncwarp();
            if (copy_mode != kCopyManual && lane == 0) {
              const uint32_t tx = (fl & kChunked) ? (uint32_t)(nr * ncols) * (uint32_t)(copy_mode == kCopyRows ? kBinBytes : cbytes)
                                                  : (copy_mode == kCopyRows ? (uint32_t)blk.w : (uint32_t)(blk.w / kBinBytes * cbytes));
              mbar_arrive_expect_tx(&s_full[cur], tx);
            }
            __syncwarp();
            if (++stp == kStages) { stp = 0; parp ^= 1u; }
          }
          unsigned char* dst = s_stage + cur * stage_bytes + ((fl & kChunked) ? 0 : blk.y);
          if (copy_mode == kCopyRows) {
            const uint32_t rowbytes = (uint32_t)(ncols * kBinBytes);
            if (lane < nr) tma_load_1d(dst + lane * rowbytes, gsrc + (int64_t)(r0 + lane) * gs_h, rowbytes, &s_full[cur]);
          } else if (copy_mode == kCopyBins) {
            const int nb = nr * ncols;
            for (int e = lane; e < nb; e += 32) {
              const int rr = e / ncols, cc = e - rr * ncols;
              tma_load_1d(dst + e * kBinBytes, gsrc + (int64_t)(r0 + rr) * gs_h + cc * gs_w, (uint32_t)cbytes, &s_full[cur]);
            }
          } else {
            const int wpb = cbytes / (4 * (int)sizeof(T));   // 4-channel words per bin
            const int nw = nr * ncols * wpb;
            for (int e = lane; e < nw; e += 32) {
              const int bb = e / wpb, wq4 = e - bb * wpb;
              const int rr = bb / ncols, cc = bb - rr * ncols;
              const T* src = gsrc + (int64_t)(r0 + rr) * gs_h + cc * gs_w + wq4 * 4;
              unsigned char* dd = dst + bb * kBinBytes + wq4 * 4 * sizeof(T);
              if (sizeof(T) == 4) *reinterpret_cast<float4*>(dd) = __ldg(reinterpret_cast<const float4*>(src));
              else *reinterpret_cast<uint2*>(dd) = __ldg(reinterpret_cast<const uint2*>(src));
            }
            if (fl & kChunked) {   // ordinary stores: a chunk is an item of its own
              __syncwarp();
              if (lane == 0) mbar_arrive(&s_full[cur]);
            }
          }
        }
        if (copy_mode == kCopyManual && !(fl & kChunked)) {
          // ordinary stores: a packed item is complete when its last candidate has been copied
          int c2 = c + 1;
          while (c2 < nc && ((uint32_t)tab.blk[c2][0] >> 24) == 0) ++c2;
          const bool closes = c2 >= nc || (tab.blk[c2][2] >> 16) != 0;
          __syncwarp();
          if (closes && lane == 0) mbar_arrive(&s_full[cur]);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&s_tempty[b]);
    }
#ifdef RAF_PROFILE
    if (lane == 0) atomicAdd(hdr + 18, (uint32_t)(prof[2] >> 6));
#endif
    return;
  }

  if (warp >= kConsumerWarps + kScanThreads / 32) {
    // ================================== LOADER WARPS ==================================================
    // Each loader warp works on its own: candidate buffers lw, lw + kLoadWarps, ...; the scanner has
    // numbered the passes they turn into, so the tables come out in order whoever fills them.
    if (stale) return;
    const int lw = warp - kConsumerWarps - kScanThreads / 32;
    const int r = lane & 15, axis = r >> 3, o = r & 7, csub = lane >> 4;
    // Table entries of kPre candidates (two per round): loaded one candidate buffer AHEAD, so that the
    // L2 round trip of the next tile's look-up overlaps the table building of the current one.
    constexpr int kPreR = 2, kPre = 2 * kPreR;
    struct Entries { uint4 e0[kPreR], e1[kPreR]; bool wide[kPreR]; };
    auto load_entries = [&](const CandBuf& cb, int p0, int nc, int c0, Entries& en) {
      const TileDesc& d = cb.t;
#pragma unroll
      for (int rd = 0; rd < kPreR; ++rd) {
        const int c = c0 + rd * 2 + csub;
        en.e0[rd] = make_uint4(0u, 0u, 0u, 0u);
        en.e1[rd] = en.e0[rd];
        en.wide[rd] = false;
        if (c < nc) {
          const int k = cb.k[p0 + c];
          const uint2 wn = cb.win[p0 + c];
          const int pix = axis ? d.x0 + o : d.y0 + o;
          const uint32_t wv = axis ? wn.y : wn.x;
          const int lo = (int)(wv & 0xffffu), hi = (int)(wv >> 16);
          if (o < (axis ? d.npx : d.npy) && pix >= lo && pix <= hi) {
            const int j = pix - lo;
            if (j < kInvCap) {
              const uint4* src = reinterpret_cast<const uint4*>(inv + ((int64_t)k * 2 + axis) * kInvCap + j);
              en.e0[rd] = __ldg(src);
              en.e1[rd] = __ldg(src + 1);
            } else {
              en.wide[rd] = true;   // window wider than the stored table: evaluated when used
            }
          }
        }
      }
    };
    Entries pre;
    bool have_pre = false;
    for (int cbn = lw;; cbn += kLoadWarps) {
      const int cbi = cbn % kNCB;
      { RAF_T0(tw); mbar_wait(&s_cfull[cbi], (uint32_t)(cbn / kNCB) & 1u); RAF_ACC(0, tw); }
      const CandBuf& cb = s_cand[cbi];
      const int cflags = cb.flags;
      if (cflags & kEnd) {
        if (cb.ncand) {   // the designated one closes the pass sequence
          const int pass = cb.pass_base, b = pass % kNB;
          mbar_wait(&s_tempty[b], ((uint32_t)(pass / kNB) & 1u) ^ 1u);
          if (lane == 0) s_tab[b].flags = kEnd;
          __syncwarp();
          if (lane == 0) mbar_arrive(&s_tfull[b]);
        }
        break;
      }
      const TileDesc d = cb.t;
      const int ncand = cb.ncand;
      const int npass = max(1, (ncand + kNC - 1) / kNC);
      Entries cur = pre;
      const bool have_cur = have_pre;
      have_pre = false;
      for (int pi = 0; pi < npass; ++pi) {
        const int pass = cb.pass_base + pi;
        const int p0 = pi * kNC, nc = min(kNC, ncand - p0);
        const int b = pass % kNB;
        RAF_T0(tl);
        bool slow = false;
        for (int c0 = 0; c0 < max(nc, 1); c0 += kPre) {
          if (!(have_cur && pi == 0 && c0 == 0)) load_entries(cb, p0, nc, c0, cur);
          if (pi == npass - 1 && c0 + kPre >= nc) {
            // last batch of this buffer: get the next buffer's first batch in flight (if it is there)
            const int nbn = cbn + kLoadWarps, nbi = nbn % kNCB;
            if (mbar_test(&s_cfull[nbi], (uint32_t)(nbn / kNCB) & 1u)) {
              const CandBuf& nb = s_cand[nbi];
              if (!(nb.flags & kEnd)) { load_entries(nb, 0, min(kNC, nb.ncand), 0, pre); have_pre = true; }
            }
          }
          if (c0 == 0) { RAF_T0(tw); mbar_wait(&s_tempty[b], ((uint32_t)(pass / kNB) & 1u) ^ 1u); RAF_ACC(3, tw); }
          PassTable& tab = s_tab[b];
#pragma unroll
          for (int rd = 0; rd < kPreR; ++rd) {
            if (c0 + rd * 2 >= nc) continue;   // (uniform)
            const int c = c0 + rd * 2 + csub;
            int first = 255, lastb = -1;
            uint4 e0 = cur.e0[rd], e1 = cur.e1[rd];
            if (c < nc) {
              if (cur.wide[rd]) pull_wide_entry(lv, a, cb.k[p0 + c], axis, axis ? d.x0 + o : d.y0 + o, e0, e1);
              const int cnt = (int)(e0.x >> 8);
              if (cnt) { first = (int)(e0.x & 0xffu); lastb = first + cnt - 1; }
              slow |= cnt > kInvW;
              if (r == 0) tab.k[c] = cb.k[p0 + c];
            }
            const int myfirst = first;
#pragma unroll
            for (int dd = 1; dd < 8; dd <<= 1) {
              first = min(first, __shfl_xor_sync(0xffffffffu, first, dd));
              lastb = max(lastb, __shfl_xor_sync(0xffffffffu, lastb, dd));
            }
            const int xf = __shfl_xor_sync(0xffffffffu, first, 8), xl = __shfl_xor_sync(0xffffffffu, lastb, 8);
            if (c < nc) {
              if (axis == 0) {   // row record (xf, xl: the candidate's range of bin columns, from the partner lanes)
                const int rowstep = max(xl - xf + 1, 0) * kBinBytes;
                const uint32_t cnt = e0.x >> 8;
                const uint32_t offA = cnt ? (uint32_t)((myfirst - first) * rowstep) : 0u;
                tab.rowrec[c][o] = make_uint4(offA | (min(cnt, 3u) << 28), e0.y, offA + (uint32_t)rowstep, e0.z);
              } else {   // column entries: the consumers want the byte offset inside a row of the block and
                         // the number of stored weights; the original meta goes to xmeta (slow path)
                tab.xmeta[c][o] = e0.x;
                const uint32_t cnt = e0.x >> 8;
                e0.x = cnt ? ((uint32_t)((myfirst - first) * kBinBytes) | (min(cnt, (uint32_t)kInvW) << 24)) : 0u;
              }
              uint4* dst = reinterpret_cast<uint4*>(&tab.info[c][r]);
              dst[0] = e0;
              dst[1] = e1;
              if (o == 0) tab.blk[c][1 + axis] = first | (max(lastb, 0) << 8) | ((lastb < first ? 1 : 0) << 16);   // (scratch)
            }
          }
        }
        PassTable& tab = s_tab[b];
        const bool anyslow = __any_sync(0xffffffffu, slow);
        __syncwarp();
        // ---- pack the candidates' blocks into stage items: lane c holds candidate c; the greedy scan
        //      over the <= kNC block sizes runs on shuffled registers -----------------------------------
        {
          int pa = 0, pb = 0, qa = 0, ncols = 0, nrows = 0, bytes = 0;
          if (lane < nc) {
            const int ry = tab.blk[lane][1], cx = tab.blk[lane][2];
            const bool empty = ((ry | cx) >> 16) != 0;
            pa = ry & 0xff; pb = (ry >> 8) & 0xff; qa = cx & 0xff;
            ncols = empty ? 0 : ((cx >> 8) & 0xff) - qa + 1;
            nrows = empty ? 0 : pb - pa + 1;
            bytes = nrows * ncols * kBinBytes;
          }
          int off = 0, open = -1, myoff = 0, myflag = 0, mytot = 0, tot = 0;
          for (int c = 0; c < nc; ++c) {
            const int bc = __shfl_sync(0xffffffffu, bytes, c);
            if (bc == 0) continue;
            if (bc > stage_bytes) {            // larger than a stage: split by rows of bins, own items
              if (lane == open) mytot = tot;
              open = -1;
              if (lane == c) myflag = kChunked;
            } else {
              if (open < 0 || off + bc > stage_bytes) {
                if (lane == open) mytot = tot;
                open = c; off = 0; tot = 0;
                if (lane == c) myflag = kNewItem;
              }
              if (lane == c) myoff = off;
              off += bc;
              tot += bc;
            }
          }
          if (lane == open) mytot = tot;
          __syncwarp();
          if (lane < nc) {
            const int rpi = (myflag & kChunked) ? max(1, stage_bytes / (ncols * kBinBytes)) : max(nrows, 1);
            *reinterpret_cast<int4*>(tab.blk[lane]) =
                make_int4(pa | (pb << 8) | (qa << 16) | (ncols << 24), myoff, rpi | (myflag << 16), mytot);
          }
        }
        if (lane == 0) {
          tab.t = d;
          tab.flags = (((cflags & kFirst) && pi == 0) ? kFirst : 0) | (((cflags & kLast) && pi == npass - 1) ? kLast : 0);
          tab.nc = nc;
          tab.slow[0] = anyslow;
          tab.slow[1] = 0;
        }
        RAF_ACC(1, tl);
        __syncwarp();
        if (lane == 0) mbar_arrive(&s_tfull[b]);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&s_cempty[cbi]);
    }
#ifdef RAF_PROFILE
    if (lw == 0 && lane == 0) {
      atomicAdd(hdr + 16, (uint32_t)(prof[0] >> 6));
      atomicAdd(hdr + 17, (uint32_t)(prof[1] >> 6));
      atomicAdd(hdr + 19, (uint32_t)(prof[3] >> 6));
      atomicAdd(hdr + 20, (uint32_t)((clock64() - prof_start) >> 6));
    }
#endif
    return;
  }

  if (warp >= kConsumerWarps) {
    // ================================== SCANNER WARPS =================================================
    if (stale) return;
    const int st = tid - 32 * kConsumerWarps, sw_ = st >> 5;
    uint32_t* counter = hdr + 8;   // next work item (zeroed by the prep, and by the last CTA of this kernel)
    auto bucket_off = [&](int key) { return boff_cached ? s_boff[key] : __ldg(boff + key); };
    // the first three items of every CTA are fixed (item order is heaviest first: the heavy ones are
    // dealt round-robin), the rest is handed out by the counter as CTAs run dry; the atomic for item
    // it+3 is in flight while item it is scanned
    const uint32_t nfixed = 3u * gridDim.x;
    uint32_t treg = 0;
    if (st == 0) {
      s_next[0] = (int)blockIdx.x;
      s_next[1] = (int)(blockIdx.x + gridDim.x);
      treg = blockIdx.x + 2u * gridDim.x;
    }
    role_sync<1, kScanThreads>();
    int cbn = 0, npass_total = 0;
    for (int it = 0;; ++it) {
      const int t = s_next[it % 3];
      if (st == 0) { s_next[(it + 2) % 3] = (int)treg; treg = nfixed + atomicAdd(counter, 1u); }
      if (t >= total_items) {   // one end marker per loader warp; the first also closes the pass sequence
        for (int e = 0; e < kLoadWarps; ++e, ++cbn) {
          const int cbi = cbn % kNCB;
          mbar_wait(&s_cempty[cbi], ((uint32_t)(cbn / kNCB) & 1u) ^ 1u);
          if (st == 0) { s_cand[cbi].flags = kEnd; s_cand[cbi].ncand = e == 0; s_cand[cbi].pass_base = npass_total; }
          mbar_arrive(&s_cfull[cbi]);
        }
        break;
      }
      TileDesc d{};
      decode(t, d);
      const int y1 = d.y0 + d.npy - 1, x1 = d.x0 + d.npx - 1;
      const int bbeg = bucket_off(d.level * lv.n + d.n), bend = bucket_off(d.level * lv.n + d.n + 1);
      int s0 = bbeg;
      do {   // one candidate buffer per scan chunk (an empty bucket still yields one, with no candidates)
        int4 wq[kScanQ];
        int kq[kScanQ];
        unsigned mq[kScanQ];
#pragma unroll
        for (int q = 0; q < kScanQ; ++q) {
          const int e = s0 + q * kScanThreads + st;
          wq[q] = make_int4(0x7fffffff, -1, 0x7fffffff, -1);
          kq[q] = 0;
          if (e < bend) { wq[q] = __ldg(bwin + e); kq[q] = __ldg(bperm + e); }   // {ymin, ymax, xmin, xmax}, conservative
        }
        const int cbi = cbn % kNCB;
        { RAF_T0(tw); mbar_wait(&s_cempty[cbi], ((uint32_t)(cbn / kNCB) & 1u) ^ 1u); RAF_ACC(0, tw); }
        CandBuf& cb = s_cand[cbi];
#pragma unroll
        for (int q = 0; q < kScanQ; ++q) {
          const bool hit = (wq[q].x <= y1) && (wq[q].y >= d.y0) && (wq[q].z <= x1) && (wq[q].w >= d.x0);
          mq[q] = __ballot_sync(0xffffffffu, hit);
          if (lane == 0) s_wcount[q * (kScanThreads / 32) + sw_] = __popc(mq[q]);
        }
        role_sync<1, kScanThreads>();
        int ncand = 0;
        int bef[kScanQ];
#pragma unroll
        for (int q = 0; q < kScanQ; ++q) bef[q] = 0;
#pragma unroll
        for (int w = 0; w < kScanQ * (kScanThreads / 32); ++w) {
          const int cnt = s_wcount[w];
#pragma unroll
          for (int q = 0; q < kScanQ; ++q)
            if (w < q * (kScanThreads / 32) + sw_) bef[q] += cnt;
          ncand += cnt;
        }
#pragma unroll
        for (int q = 0; q < kScanQ; ++q)
          if (mq[q] & (1u << lane)) {
            const int p = bef[q] + __popc(mq[q] & ((1u << lane) - 1u));
            cb.k[p] = kq[q];
            cb.win[p] = make_uint2((uint32_t)wq[q].x | ((uint32_t)wq[q].y << 16), (uint32_t)wq[q].z | ((uint32_t)wq[q].w << 16));
          }
        if (st == 0) {
          cb.t = d;
          cb.flags = (s0 == bbeg ? kFirst : 0) | (s0 + kScan >= bend ? kLast : 0);
          cb.ncand = ncand;
          cb.pass_base = npass_total;
        }
        npass_total += max(1, (ncand + kNC - 1) / kNC);
        mbar_arrive(&s_cfull[cbi]);
        ++cbn;
        s0 += kScan;
        role_sync<1, kScanThreads>();   // s_wcount is rewritten by the next chunk; orders the s_next accesses too
      } while (s0 < bend);
    }
    // the last CTA to run out of work re-arms the work counter for the next call
    if (st == 0) {
      __threadfence();
      if (atomicAdd(hdr + 9, 1u) == gridDim.x - 1) { hdr[8] = 0u; hdr[9] = 0u; }
    }
    return;
  }

  // ================================= CONSUMER WARPS ===================================================
  // warp = (tile row i, column group): acc[jj][q] = channels ch0 + q*128 + lane*4 .. +3 of pixel (i, j0 + jj)
  const int i = warp % kRowWarps, j0 = (warp / kRowWarps) * kJW;
  if (stale) {   // the workspace was not written for these arguments (RAF_REUSE_PREP misuse): poison, loudly
    const float qnan = __int_as_float(0x7fc00000);
    for (int t = blockIdx.x; t < total_items; t += gridDim.x) {
      TileDesc d{};
      decode(t, d);
      if (i >= d.npy) continue;
      float* grow = reinterpret_cast<float*>(const_cast<void*>(lv.data[d.level])) + (int64_t)d.n * lv.sn[d.level] +
                    (int64_t)(d.y0 + i) * lv.sh[d.level] + (int64_t)d.x0 * lv.sw[d.level] + d.chunk * CH + lane * 4;
      for (int j = j0; j < min(d.npx, j0 + kJW); ++j)
#pragma unroll
        for (int q = 0; q < Q; ++q)
          if (d.chunk * CH + q * 128 + lane * 4 < lv.c)
            *reinterpret_cast<float4*>(grow + j * lv.sw[d.level] + q * 128) = make_float4(qnan, qnan, qnan, qnan);
    }
    return;
  }

  float4 acc[kJW][Q];
  bool act[Q];
  float* grow = nullptr;
  int sw = 0, npx = 0;
  bool row_live = false;
  int st = 0;            // stage ring position: the item being consumed / the next one
  uint32_t par = 0;
  bool held = false;     // a stage item is open
  const unsigned char* lane_stage = s_stage + lane * 4 * sizeof(T);
  auto release = [&]() {
    if (held) {
      __syncwarp();
      if (lane == 0) mbar_arrive(&s_empty[st]);
      if (++st == kStages) { st = 0; par ^= 1u; }
      held = false;
    }
  };

  for (int pass = 0;; ++pass) {
    const int b = pass % kNB;
    { RAF_T0(tw); mbar_wait(&s_tfull[b], (uint32_t)(pass / kNB) & 1u); RAF_ACC(0, tw); }
    const PassTable& tab = s_tab[b];
    const int flags = tab.flags;
    if (flags & kEnd) break;
    RAF_T0(tpass);
    const int nc = tab.nc;
    const int y0 = tab.t.y0, x0 = tab.t.x0;
    const int ch0 = tab.t.chunk * CH;
    if (flags & kFirst) {
      const int level = tab.t.level;
      sw = (int)lv.sw[level];
      npx = tab.t.npx;
      row_live = i < tab.t.npy;
      grow = reinterpret_cast<float*>(const_cast<void*>(lv.data[level])) + (int64_t)tab.t.n * lv.sn[level] +
             (int64_t)(y0 + i) * lv.sh[level] + (int64_t)x0 * sw + ch0 + lane * 4;
#pragma unroll
      for (int q = 0; q < Q; ++q) act[q] = ch0 + q * 128 + lane * 4 < lv.c;
#pragma unroll
      for (int jj = 0; jj < kJW; ++jj)
#pragma unroll
        for (int q = 0; q < Q; ++q) {
          acc[jj][q] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (accumulate && row_live && j0 + jj < npx && act[q])
            acc[jj][q] = *reinterpret_cast<const float4*>(grow + (j0 + jj) * sw + q * 128);
        }
    }

    for (int c = 0; c < nc; ++c) {
      const int4 blk = *reinterpret_cast<const int4*>(tab.blk[c]);
      const int ncols = (int)((uint32_t)blk.x >> 24);
      if (ncols == 0) continue;   // nothing of this candidate lands in the tile
      const int pa = blk.x & 0xff, pb = (blk.x >> 8) & 0xff;
      const int fl = blk.z >> 16, rpi = blk.z & 0xffff;
      const InvEntry* info = tab.info[c];
      const uint4 rr = tab.rowrec[c][i];
      const uint32_t nrow = rr.x >> 28;
      if (!(fl & kChunked) && nrow <= 2u) {
        // ---- usual case: the whole block sits in a stage and at most two rows of bins land on my row ----
        if (fl) {   // this candidate opens a stage item
          release();
          { RAF_T0(tf); mbar_wait(&s_full[st], par); RAF_ACC(1, tf); }
          held = true;
        }
        if (nrow == 0u) continue;
        RAF_T0(tj);
        const unsigned char* rowA = lane_stage + st * stage_bytes + blk.y + (rr.x & 0xfffffffu);
        const int stepB = (int)(rr.z - (rr.x & 0xfffffffu));
        const float wyA = __uint_as_float(rr.y), wyB = __uint_as_float(rr.w);
#pragma unroll
        for (int jj = 0; jj < kJW; ++jj) {
          const uint4 x = *reinterpret_cast<const uint4*>(&info[8 + j0 + jj]);   // offset | count << 24, w0, w1, w2
          const int xcnt = (int)(x.x >> 24);
          if (xcnt == 0) continue;
          const unsigned char* p = rowA + (x.x & 0xffffffu);
          const float xw0 = __uint_as_float(x.y), xw1 = __uint_as_float(x.z);
          if (nrow == 2u) {
            fma_bin<T, Q>(acc[jj], wyA * xw0, p);
            fma_bin<T, Q>(acc[jj], wyB * xw0, p + stepB);
            if (xcnt > 1) {
              fma_bin<T, Q>(acc[jj], wyA * xw1, p + kBinBytes);
              fma_bin<T, Q>(acc[jj], wyB * xw1, p + kBinBytes + stepB);
            }
          } else {
            fma_bin<T, Q>(acc[jj], wyA * xw0, p);
            if (xcnt > 1) fma_bin<T, Q>(acc[jj], wyA * xw1, p + kBinBytes);
          }
          if (xcnt > 2) {
#pragma unroll 1
            for (int bq = 2; bq < xcnt; ++bq) {
              const float wx = info[8 + j0 + jj].w[bq];
              fma_bin<T, Q>(acc[jj], wyA * wx, p + bq * kBinBytes);
              if (nrow == 2u) fma_bin<T, Q>(acc[jj], wyB * wx, p + stepB + bq * kBinBytes);
            }
          }
        }
        RAF_ACC(4, tj);
        continue;
      }
      // ---- generic: blocks split over several stage items, or more than two rows of bins on my row ----
      const uint32_t rmeta = info[i].meta;
      const int rfirst = (int)(rmeta & 0xffu), rcnt = min((int)(rmeta >> 8), kInvW);
      const int rowstep = ncols * kBinBytes;
      // column records of my pixels, loaded once per candidate: byte offset of the first bin in a row of
      // the block | stored weights << 24, and the first two weights
      uint32_t xo[kJW];
      float xw0[kJW], xw1[kJW];
#pragma unroll
      for (int jj = 0; jj < kJW; ++jj) {
        const uint4 x = *reinterpret_cast<const uint4*>(&info[8 + j0 + jj]);
        xo[jj] = x.x;
        xw0[jj] = __uint_as_float(x.y);
        xw1[jj] = __uint_as_float(x.z);
      }
      for (int r0 = pa; r0 <= pb; r0 += rpi) {
        const int nr = min(rpi, pb - r0 + 1);
        if (fl) {   // this candidate (or chunk) opens a stage item
          release();
          { RAF_T0(tf); mbar_wait(&s_full[st], par); RAF_ACC(1, tf); }
          held = true;
        }
        const unsigned char* base = lane_stage + st * stage_bytes + ((fl & kChunked) ? 0 : blk.y);
        const int alo = max(rfirst, r0), ahi = min(rfirst + rcnt, r0 + nr);
        RAF_T0(tj);
        // rows of bins alo .. ahi-1 of this block land on my pixel row; two at a time
        for (int aa = alo; aa < ahi; aa += 2) {
          const bool two = aa + 1 < ahi;
          const float wyA = info[i].w[aa - rfirst];
          const float wyB = two ? info[i].w[aa + 1 - rfirst] : 0.0f;
          const unsigned char* rowA = base + (aa - r0) * rowstep;
#pragma unroll
          for (int jj = 0; jj < kJW; ++jj) {
            const int xcnt = (int)(xo[jj] >> 24);
            if (xcnt == 0) continue;
            const unsigned char* p = rowA + (xo[jj] & 0xffffffu);
            if (two) {
              fma_bin<T, Q>(acc[jj], wyA * xw0[jj], p);
              fma_bin<T, Q>(acc[jj], wyB * xw0[jj], p + rowstep);
              if (xcnt > 1) {
                fma_bin<T, Q>(acc[jj], wyA * xw1[jj], p + kBinBytes);
                fma_bin<T, Q>(acc[jj], wyB * xw1[jj], p + kBinBytes + rowstep);
              }
            } else {
              fma_bin<T, Q>(acc[jj], wyA * xw0[jj], p);
              if (xcnt > 1) fma_bin<T, Q>(acc[jj], wyA * xw1[jj], p + kBinBytes);
            }
            if (xcnt > 2) {
#pragma unroll 1
              for (int bq = 2; bq < xcnt; ++bq) {
                const float wx = info[8 + j0 + jj].w[bq];
                fma_bin<T, Q>(acc[jj], wyA * wx, p + bq * kBinBytes);
                if (two) fma_bin<T, Q>(acc[jj], wyB * wx, p + rowstep + bq * kBinBytes);
              }
            }
          }
        }
        RAF_ACC(4, tj);
      }
    }
    release();
    // ---- rare: runs of more than kInvW bins on one pixel (bins narrower than 2/7 pixel): the pairs
    //      beyond the stored weights, straight from global memory with weights evaluated on the fly
    if ((tab.slow[0] | tab.slow[1]) && row_live) {
      for (int c = 0; c < nc; ++c) {
        const uint32_t rmeta = tab.info[c][i].meta;
        const int rfirst = (int)(rmeta & 0xffu), rcnt = (int)(rmeta >> 8);
        if (rcnt == 0) continue;
        const int k = tab.k[c];
        for (int j = j0; j < min(npx, j0 + kJW); ++j) {
          const uint32_t xm = tab.xmeta[c][j];
          const int xfirst = (int)(xm & 0xffu), xcnt = (int)(xm >> 8);
          if (xcnt == 0 || (rcnt <= kInvW && xcnt <= kInvW)) continue;
          float4 tq[Q];
#pragma unroll
          for (int q = 0; q < Q; ++q) tq[q] = make_float4(0.f, 0.f, 0.f, 0.f);
          for (int ai = 0; ai < rcnt; ++ai)
            for (int bq = 0; bq < xcnt; ++bq) {
              if (ai < kInvW && bq < kInvW) continue;   // done by the fast loop
              const float wy = ai < kInvW ? tab.info[c][i].w[ai] : pull_slow_weight(lv, a, k, 0, y0 + i, rfirst + ai);
              const float wx = bq < kInvW ? tab.info[c][8 + j].w[bq] : pull_slow_weight(lv, a, k, 1, x0 + j, xfirst + bq);
              const T* src = gout + (int64_t)k * gs_k + (rfirst + ai) * gs_h + (xfirst + bq) * gs_w + ch0 + lane * 4;
#pragma unroll
              for (int q = 0; q < Q; ++q)
                if (act[q]) fma4(tq[q], wy * wx, ldg_quad<T>(src + q * 128));
            }
#pragma unroll
          for (int jj = 0; jj < kJW; ++jj)
            if (j0 + jj == j) {
#pragma unroll
              for (int q = 0; q < Q; ++q) {
                acc[jj][q].x += tq[q].x; acc[jj][q].y += tq[q].y; acc[jj][q].z += tq[q].z; acc[jj][q].w += tq[q].w;
              }
            }
        }
      }
    }
    RAF_T0(tst);
    if ((flags & kLast) && row_live) {
#pragma unroll
      for (int jj = 0; jj < kJW; ++jj)
        if (j0 + jj < npx) {
#pragma unroll
          for (int q = 0; q < Q; ++q)
            if (act[q]) *reinterpret_cast<float4*>(grow + (j0 + jj) * sw + q * 128) = acc[jj][q];
        }
    }
    RAF_ACC(2, tst);
    __syncwarp();
    if (lane == 0) mbar_arrive(&s_tempty[b]);
    RAF_ACC(3, tpass);
  }
#ifdef RAF_PROFILE
  if (tid == 0) {
    for (int q = 0; q < 4; ++q) atomicAdd(hdr + 24 + q, (uint32_t)(prof[q] >> 6));
    atomicAdd(hdr + 28, (uint32_t)((clock64() - prof_start) >> 6));
    atomicAdd(hdr + 29, (uint32_t)(prof[4] >> 6));
  }
#endif
}

static size_t pull_table_bytes() { return kNB * sizeof(PassTable) + kNCB * sizeof(CandBuf); }

// Launch plan of the pull kernel; RAF_ERR_UNSUPPORTED when the arguments are outside its range
// (decided on the host before anything is launched).
struct PullPlan {
  PullTiles t;
  int cpl, stage_bytes, copy_mode;
  dim3 grid;
};

static int pull_plan(const LevelsParam& lv, size_t esz, const RoiArgs& a, const void* gout, const int64_t* gs, PullPlan* pl) {
  PullTiles& t = pl->t;
  int64_t total = 0;
  for (int i = 0; i < lv.L; ++i) {
    const int l = lv.L - 1 - i;  // coarsest level first
    t.order[i] = l;
    t.tiles_y[l] = (lv.h[l] + kTH - 1) / kTH;
    t.tiles_x[l] = (lv.w[l] + kTW - 1) / kTW;
    t.start[i] = (int32_t)total;
    total += (int64_t)t.tiles_y[l] * t.tiles_x[l];
  }
  t.start[lv.L] = (int32_t)total;
  // channels per CTA: 256 (8 per lane, 2 CTAs per SM) when the pixel vector is a multiple of 256, else 128
  int cpl = (lv.c % 256 == 0) ? 8 : 4;
#ifdef RAF_EXPERIMENT
  if (const char* e = getenv("RAF_TUNE_CPL")) cpl = atoi(e);
#endif
  const int CH = 32 * cpl;
  t.chunks = (lv.c + CH - 1) / CH;
  const int64_t gx = (int64_t)lv.n * t.chunks;
  const int64_t binbytes = (int64_t)CH * esz;
  int stage_bytes = 32 * 1024;
#ifdef RAF_EXPERIMENT
  if (const char* e = getenv("RAF_TUNE_STAGE")) stage_bytes = atoi(e);
#endif
  while ((int64_t)a.PW * binbytes > stage_bytes) stage_bytes *= 2;   // a row of bins must fit a stage
  // 32-bit offset arithmetic inside the kernel: grad_out must fit; windows are packed in 16 bits
  const int64_t span = (int64_t)a.K * gs[0] + (int64_t)a.PH * gs[2] + (int64_t)a.PW * gs[3] + lv.c;
  if (total * gx >= ((int64_t)1 << 30) || span >= ((int64_t)1 << 31) || (int64_t)kStages * stage_bytes + pull_table_bytes() > 200 * 1024)
    return RAF_ERR_UNSUPPORTED;
  for (int l = 0; l < lv.L; ++l)
    if (lv.h[l] > 32767 || lv.w[l] > 32767 || (int64_t)lv.w[l] * lv.sw[l] + (int64_t)kTH * lv.sh[l] >= ((int64_t)1 << 31))
      return RAF_ERR_UNSUPPORTED;
  // bulk-async copies need 16-byte aligned sources and sizes
  const bool al16 = ((uintptr_t)gout % 16 == 0) && (gs[0] * esz % 16 == 0) && (gs[2] * esz % 16 == 0) &&
                    (gs[3] * esz % 16 == 0) && ((int64_t)lv.c * esz % 16 == 0);
  int copy_mode = !al16 ? kCopyManual : (t.chunks == 1 && gs[3] == CH ? kCopyRows : kCopyBins);
#ifdef RAF_EXPERIMENT
  if (const char* e = getenv("RAF_TUNE_COPY")) copy_mode = atoi(e);
#endif
  pl->cpl = cpl;
  pl->stage_bytes = stage_bytes;
  pl->copy_mode = copy_mode;
  int sms = 148, dev = 0;   // persistent CTAs, one per SM; work items are handed out by an atomic counter
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return RAF_ERR_CUDA;
  const int64_t items = total * gx;
  pl->grid = dim3((unsigned)(items < sms ? items : sms));
  return RAF_OK;
}

int pull_eligible(const LevelsParam& glv, raf_dtype gout_dtype, const RoiArgs& a, const void* grad_out,
                  const int64_t* gout_strides) {
  PullPlan pl;
  return pull_plan(glv, gout_dtype == RAF_F32 ? 4 : 2, a, grad_out, gout_strides, &pl);
}

template <typename T>
static int pull_typed(const LevelsParam& lv, const RoiArgs& a, const void* gout, const int64_t* gs,
                      const PullPrepOut& prep, int accumulate, cudaStream_t stream) {
  PullPlan pl;
  const int rc = pull_plan(lv, sizeof(T), a, gout, gs, &pl);
  if (rc) return rc;
  const size_t smem = (size_t)kStages * pl.stage_bytes + pull_table_bytes();
  const T* g = reinterpret_cast<const T*>(gout);
  cudaError_t err;
  if (pl.cpl == 8) {
    err = cudaFuncSetAttribute(bwd_pull_kernel<T, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err == cudaSuccess)
      bwd_pull_kernel<T, 8><<<pl.grid, kPullThreads, smem, stream>>>(lv, a, g, (int)gs[0], (int)gs[2], (int)gs[3], prep.hdr,
                                                                     prep.bperm, prep.boff, prep.bwin, prep.inv, pl.t, accumulate,
                                                                     prep.fp, pl.stage_bytes, pl.copy_mode);
  } else {
    err = cudaFuncSetAttribute(bwd_pull_kernel<T, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err == cudaSuccess)
      bwd_pull_kernel<T, 4><<<pl.grid, kPullThreads, smem, stream>>>(lv, a, g, (int)gs[0], (int)gs[2], (int)gs[3], prep.hdr,
                                                                     prep.bperm, prep.boff, prep.bwin, prep.inv, pl.t, accumulate,
                                                                     prep.fp, pl.stage_bytes, pl.copy_mode);
  }
  if (err != cudaSuccess) return RAF_ERR_CUDA;
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

int launch_backward_pull(const LevelsParam& glv, raf_dtype gout_dtype, const RoiArgs& a, const void* grad_out,
                         const int64_t* gout_strides, const PullPrepOut& prep, int accumulate, cudaStream_t stream) {
  switch (gout_dtype) {
    case RAF_F32: return pull_typed<float>(glv, a, grad_out, gout_strides, prep, accumulate, stream);
    case RAF_F16: return pull_typed<__half>(glv, a, grad_out, gout_strides, prep, accumulate, stream);
    case RAF_BF16: return pull_typed<__nv_bfloat16>(glv, a, grad_out, gout_strides, prep, accumulate, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
