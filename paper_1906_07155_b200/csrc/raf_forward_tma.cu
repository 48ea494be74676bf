// raf_forward_tma.cu -- K2, bulk-async variant of the channels-last forward.
//
// The direct gather (raf_forward.cu) is bound by what registers can keep in flight and by the L1
// load path (~2 cycles per 128-byte wavefront of a 128-bit load).  Here the bytes travel
// L2 -> shared memory by the async copy engine instead:
//   * persistent CTAs (one per SM), work item = (RoI, chunk of 512 bytes of channels per pixel);
//   * warp 0 = PRODUCER: builds the RoI's merged tap tables (same arithmetic as the direct kernel),
//     lists the UNIQUE pixel rows the RoI touches (taps are monotone for ordinary boxes) and streams
//     them, in order, into a ring of row slots with cp.async.bulk (one copy per pixel: 512 contiguous
//     bytes), completion signalled on the slot's `full` mbarrier;
//   * warps 1.. = CONSUMERS, one per output bin column pw: for every bin row ph they wait for the
//     <= 2g rows of its y taps, read the taps with 128-bit shared loads (conflict-free: lanes =
//     channel vectors), accumulate in fp32 and store the bin; rows no later bin needs are handed
//     back through the slot's `empty` mbarrier.  Every window pixel crosses L2 -> SM once per RoI.
// RoIs this scheme does not take (window wider than a slot, reversed boxes, too many rows per
// bin) are gathered by the consumers straight from global memory, same arithmetic ("direct" item).
//
// STATUS (round 1): EXPERIMENTAL, compiled always but dispatched only when the library is built
// with -DRAF_FWD_TMA (RAF_FWD_TMA=1 python -m paper_1906_07155_b200.build).  Parity-green under that
// build (all forward cases of tests/test_gpu_parity.py), but 2.5x SLOWER than the direct kernel on
// config 2 (fp32 167 us, bf16 92 us vs 57 / 39 us; profiles/r1_experiments.md).  Two persistent
// CTAs per SM with a 6-row ring each: every item is latency-bound row by row, and shared memory
// (~200 KB per SM) cannot hold more bytes in flight than the register file already does for the
// direct kernel (~118 KB per SM), so staging buys no extra memory-level parallelism here.
#include "raf_device.cuh"
#include "raf_host.h"

namespace raf {

constexpr int kTmaSlots = 6;           // ring of pixel-row slots (two CTAs per SM)
constexpr int kTmaSlotPx = 32;         // pixels per slot (window width limit of the staged path)
constexpr int kTmaChunkBytes = 512;    // channel bytes per pixel and work item
constexpr int kTmaMaxBins = 16;        // PH, PW <= 16 in this variant
constexpr int kTmaConsumers = 7;       // consumer warps
constexpr int kTmaThreads = 32 * (1 + kTmaConsumers);

struct TmaTap {   // merged tap: pixel index (y: row sequence index in .seq) and weight
  int pix;
  float w;
};

struct TmaTables {                      // one RoI, written by the producer, read by the consumers
  TmaTap ytap[kTmaMaxBins][4];
  TmaTap xtap[kTmaMaxBins][4];          // pix relative to xa
  unsigned char yseq[kTmaMaxBins][4];   // row sequence index of the y tap
  int ycnt[kTmaMaxBins], xcnt[kTmaMaxBins];
  int ylo[kTmaMaxBins + 1];             // first row sequence index bin row ph needs (ylo[PH] = nrows)
  int nrows;                            // unique rows (0: nothing to load / all-zero output)
  int direct;                           // 1: consumers gather from global memory
  int valid;                            // 0: invalid batch index -> zero rows
  int level, b, xa, npx;
  int k, chunk;
  unsigned g0;                          // global row counter at the start of this item
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(b)), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// 16 bytes of T widened to fp32 lanes (works for shared and global addresses).
template <typename T> struct Cvt16;
template <> struct Cvt16<float> {
  static constexpr int N = 4;
  static __device__ __forceinline__ void widen(const uint4& r, float (&v)[4]) {
    v[0] = __uint_as_float(r.x); v[1] = __uint_as_float(r.y); v[2] = __uint_as_float(r.z); v[3] = __uint_as_float(r.w);
  }
};
template <> struct Cvt16<__half> {
  static constexpr int N = 8;
  static __device__ __forceinline__ void widen(const uint4& r, float (&v)[8]) {
    const __half2* h = reinterpret_cast<const __half2*>(&r);
#pragma unroll
    for (int i = 0; i < 4; ++i) { const float2 f = __half22float2(h[i]); v[2 * i] = f.x; v[2 * i + 1] = f.y; }
  }
};
template <> struct Cvt16<__nv_bfloat16> {
  static constexpr int N = 8;
  static __device__ __forceinline__ void widen(const uint4& r, float (&v)[8]) {
    const uint32_t* u = reinterpret_cast<const uint32_t*>(&r);
#pragma unroll
    for (int i = 0; i < 4; ++i) { v[2 * i] = __uint_as_float(u[i] << 16); v[2 * i + 1] = __uint_as_float(u[i] & 0xffff0000u); }
  }
};

// Merged taps of one bin in registers (g <= 2): pix[q], w[q], q < cnt.
__device__ __forceinline__ int tma_bin_taps(float start, float bsz, int bin, int g, int n, float scale_w,
                                            int (&pix)[4], float (&w)[4]) {
  int cnt = 0;
#pragma unroll
  for (int q = 0; q < 4; ++q) { pix[q] = 0; w[q] = 0.f; }
  auto add = [&](int p, float v) {
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
    add(t.lo, t.wh * scale_w);
    add(t.hi, t.wl * scale_w);
  }
  return cnt;
}

// Producer warp: tables of work item (k, chunk) into T (shared).  Lanes = bins (PH + PW <= 32).
// s_flat / s_seq: 64-int scratch.  rowpix[i] = pixel row of row sequence index i.
__device__ __forceinline__ void tma_build_tables(const LevelsParam& lv, const RoiArgs& a, int k, int chunk,
                                                 unsigned g0, TmaTables& T, int* rowpix, int* s_flat, int* s_seq) {
  const int lane = threadIdx.x & 31;
  const int PH = a.PH, PW = a.PW, g = a.sampling_ratio;
  const float* r = a.rois + 5 * (int64_t)k;
  const float r0 = __ldg(r), x1 = __ldg(r + 1), y1 = __ldg(r + 2), x2 = __ldg(r + 3), y2 = __ldg(r + 4);
  const int level = level_of(x1, y1, x2, y2, lv.L, a.finest_scale);
  const RoiGeom geo = roi_geom(x1, y1, x2, y2, lv.scale[level], PH, PW, g, a.aligned);
  const int b = batch_index_of(r0, lv.n);
  const bool isy = lane < PH, isx = lane >= PH && lane < PH + PW;
  int pix[4];
  float w[4];
  int cnt = 0;
  if (isy) cnt = tma_bin_taps(geo.sy, geo.bh, lane, g, lv.h[level], geo.inv_count, pix, w);
  else if (isx) cnt = tma_bin_taps(geo.sx, geo.bw, lane - PH, g, lv.w[level], 1.0f, pix, w);
  else { pix[0] = pix[1] = pix[2] = pix[3] = 0; w[0] = w[1] = w[2] = w[3] = 0.f; }

  // x window [xa, xb]
  int xmin = 0x7fffffff, xmax = -1;
  if (isx)
#pragma unroll
    for (int q = 0; q < 4; ++q)
      if (q < cnt) { xmin = min(xmin, pix[q]); xmax = max(xmax, pix[q]); }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    xmin = min(xmin, __shfl_xor_sync(0xffffffffu, xmin, d));
    xmax = max(xmax, __shfl_xor_sync(0xffffffffu, xmax, d));
  }
  if (isx) {
    T.xcnt[lane - PH] = cnt;
#pragma unroll
    for (int q = 0; q < 4; ++q) { T.xtap[lane - PH][q].pix = (q < cnt) ? pix[q] - xmin : 0; T.xtap[lane - PH][q].w = w[q]; }
  }

  // flat list of the y taps in (ph, q) order -> unique row sequence
  const int ycnt = isy ? cnt : 0;
  int incl = ycnt;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += t;
  }
  const int n = __shfl_sync(0xffffffffu, incl, 31), s0 = incl - ycnt;
  if (isy) {
    T.ycnt[lane] = cnt;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      T.ytap[lane][q].pix = pix[q];
      T.ytap[lane][q].w = w[q];
      if (q < cnt) s_flat[s0 + q] = pix[q];
    }
  }
  __syncwarp();
  int nrows = 0;
  bool mono = true;
  for (int e0 = 0; e0 < n; e0 += 32) {
    const int e = e0 + lane;
    const bool in = e < n;
    const int p = in ? s_flat[e] : 0, prev = (in && e > 0) ? s_flat[e - 1] : -1;
    const bool isnew = in && (e == 0 || p != prev);
    if (in && e > 0 && p < prev) mono = false;
    const unsigned m = __ballot_sync(0xffffffffu, isnew);
    const int idx = nrows + __popc(m & ((2u << lane) - 1u)) - 1;
    if (in) s_seq[e] = idx;
    if (isnew) rowpix[idx] = p;
    nrows += __popc(m);
  }
  mono = __all_sync(0xffffffffu, mono);
  __syncwarp();
  if (isy) {
#pragma unroll
    for (int q = 0; q < 4; ++q) T.yseq[lane][q] = (unsigned char)((q < cnt) ? s_seq[s0 + q] : 0);
    T.ylo[lane] = (s0 < n) ? s_seq[s0] : nrows;
  }
  if (lane == 0) {
    T.ylo[PH] = nrows;
    const int npx = xmax - xmin + 1;
    T.valid = b >= 0;
    T.direct = (!mono || npx > kTmaSlotPx) ? 1 : 0;
    T.nrows = (b >= 0 && xmax >= 0 && n > 0) ? nrows : 0;
    T.level = level; T.b = b >= 0 ? b : 0; T.xa = xmax >= 0 ? xmin : 0; T.npx = xmax >= 0 ? npx : 0;
    T.k = k; T.chunk = chunk; T.g0 = g0;
  }
  __syncwarp();
}

// acc += sum_{a < NY, b < NX} (yw[a] * xw[b]) * row_a[xo[b]]: every 16-byte shared load is issued
// before the first use.  rp[a] already includes the lane's 16-byte offset; xo[b] = pixel * 512 bytes.
template <typename T, int NY, int NX>
__device__ __forceinline__ void tma_accumulate(const unsigned char* const (&rp)[4], const float (&yw)[4],
                                               const int (&xo)[4], const float (&xw)[4],
                                               float (&acc)[Cvt16<T>::N]) {
  constexpr int VN = Cvt16<T>::N;
  uint4 raw[NY][NX];
#pragma unroll
  for (int a = 0; a < NY; ++a)
#pragma unroll
    for (int b = 0; b < NX; ++b) raw[a][b] = *reinterpret_cast<const uint4*>(rp[a] + xo[b]);
#pragma unroll
  for (int a = 0; a < NY; ++a)
#pragma unroll
    for (int b = 0; b < NX; ++b) {
      float v[VN];
      Cvt16<T>::widen(raw[a][b], v);
      const float w = yw[a] * xw[b];
#pragma unroll
      for (int j = 0; j < VN; ++j) acc[j] = fmaf(w, v[j], acc[j]);
    }
}

template <typename T, int NY>
__device__ __forceinline__ void tma_dispatch_x(int nx, const unsigned char* const (&rp)[4], const float (&yw)[4],
                                               const int (&xo)[4], const float (&xw)[4],
                                               float (&acc)[Cvt16<T>::N]) {
  switch (nx) {
    case 1: tma_accumulate<T, NY, 1>(rp, yw, xo, xw, acc); break;
    case 2: tma_accumulate<T, NY, 2>(rp, yw, xo, xw, acc); break;
    case 3: tma_accumulate<T, NY, 3>(rp, yw, xo, xw, acc); break;
    default: tma_accumulate<T, NY, 4>(rp, yw, xo, xw, acc); break;
  }
}

struct TmaSmem {   // dynamic shared memory carve-up (ring first: 128-byte aligned slots)
  static constexpr int kSlotBytes = kTmaSlotPx * kTmaChunkBytes;
  unsigned char ring[kTmaSlots][kSlotBytes];
  TmaTables tab[2];
  int rowpix[2][64];
  int flat[64], seq[64];
  uint64_t full[kTmaSlots], empty[kTmaSlots], tfull[2], tempty[2];
};

template <typename T>
__global__ void __launch_bounds__(kTmaThreads, 2)
fwd_tma_kernel(const LevelsParam lv, const RoiArgs a, T* __restrict__ out, int64_t os_k, int64_t os_h,
               int64_t os_w, int chunks) {
  constexpr int VN = Cvt16<T>::N;
  constexpr int kChunkElems = kTmaChunkBytes / (int)sizeof(T);
  extern __shared__ __align__(128) unsigned char tma_smem_raw[];
  TmaSmem& S = *reinterpret_cast<TmaSmem*>(tma_smem_raw);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int PH = a.PH, PW = a.PW;
  const int64_t nitems = (int64_t)a.K * chunks;

  if (threadIdx.x == 0) {
    for (int i = 0; i < kTmaSlots; ++i) { mbar_init(&S.full[i], 1); mbar_init(&S.empty[i], kTmaConsumers); }
    for (int i = 0; i < 2; ++i) { mbar_init(&S.tfull[i], 1); mbar_init(&S.tempty[i], kTmaConsumers); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == 0) {
    // ================================ PRODUCER ================================================
    unsigned g0 = 0;
    int it = 0;
    for (int64_t item = blockIdx.x; item < nitems; item += gridDim.x, ++it) {
      const int buf = it & 1;
      mbar_wait(&S.tempty[buf], (uint32_t)(((it >> 1) & 1) ^ 1));
      const int k = (int)(item / chunks), chunk = (int)(item - (int64_t)k * chunks);
      TmaTables& Tb = S.tab[buf];
      tma_build_tables(lv, a, k, chunk, g0, Tb, S.rowpix[buf], S.flat, S.seq);
      const int nrows = Tb.nrows, direct = Tb.direct, npx = Tb.npx, xa = Tb.xa, level = Tb.level;
      __syncwarp();
      if (lane == 0) mbar_arrive(&S.tfull[buf]);
      if (nrows == 0 || direct) continue;   // nothing staged: g0 unchanged (consumers agree)
      const int cbytes = min(kTmaChunkBytes, (lv.c - chunk * kChunkElems) * (int)sizeof(T));
      const T* base = reinterpret_cast<const T*>(lv.data[level]) + (int64_t)Tb.b * lv.sn[level] +
                      (int64_t)xa * lv.sw[level] + chunk * kChunkElems;
      const int64_t sh = lv.sh[level], sw = lv.sw[level];
      for (int i = 0; i < nrows; ++i) {
        const unsigned G = g0 + (unsigned)i;
        const int slot = (int)(G % kTmaSlots);
        const unsigned gen = G / kTmaSlots;
        mbar_wait(&S.empty[slot], (gen & 1u) ^ 1u);
        if (lane == 0) mbar_expect_tx(&S.full[slot], (uint32_t)(npx * cbytes));
        __syncwarp();
        const T* row = base + (int64_t)S.rowpix[buf][i] * sh;
        if (sw * (int64_t)sizeof(T) == kTmaChunkBytes && cbytes == kTmaChunkBytes) {
          if (lane == 0)   // the chunk is the whole pixel: the row segment is one contiguous run
            bulk_g2s(&S.ring[slot][0], row, (uint32_t)(npx * kTmaChunkBytes), &S.full[slot]);
        } else {
          for (int px = lane; px < npx; px += 32)
            bulk_g2s(&S.ring[slot][px * kTmaChunkBytes], row + (int64_t)px * sw, (uint32_t)cbytes, &S.full[slot]);
        }
      }
      g0 += (unsigned)nrows;
    }
  } else {
    // ================================ CONSUMERS ===============================================
    const int cw = warp - 1;
    unsigned g0 = 0;
    int it = 0;
    for (int64_t item = blockIdx.x; item < nitems; item += gridDim.x, ++it) {
      const int buf = it & 1;
      mbar_wait(&S.tfull[buf], (uint32_t)((it >> 1) & 1));
      const TmaTables& Tb = S.tab[buf];
      const int nrows = Tb.nrows, direct = Tb.direct, level = Tb.level;
      const bool staged = nrows > 0 && !direct;
      const int k = Tb.k, chunk = Tb.chunk;
      const int ch0 = chunk * kChunkElems + lane * VN;
      const bool act = ch0 < lv.c;
      T* out_k = out + (int64_t)k * os_k + ch0;
      const T* gbase = reinterpret_cast<const T*>(lv.data[level]) + (int64_t)Tb.b * lv.sn[level] +
                       (int64_t)Tb.xa * lv.sw[level] + (act ? ch0 : 0);
      const int64_t sh = lv.sh[level], sw = lv.sw[level];
      int waited = 0, rel = 0;
      for (int ph = 0; ph < PH; ++ph) {
        const int ny = nrows > 0 ? Tb.ycnt[ph] : 0;
        if (staged && ny > 0) {
          const int need = (int)Tb.yseq[ph][ny - 1] + 1;
          while (waited < need) {
            const unsigned G = g0 + (unsigned)waited;
            mbar_wait(&S.full[G % kTmaSlots], (G / kTmaSlots) & 1u);
            ++waited;
          }
        }
        const unsigned char* rp[4];
        float yw[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {   // y taps of this bin row: row pointers (lane's 16 bytes) and weights
          const int sl = (staged && q < ny) ? (int)((g0 + Tb.yseq[ph][q]) % kTmaSlots) : 0;
          rp[q] = &S.ring[sl][lane * 16];
          yw[q] = Tb.ytap[ph][q].w;
        }
        for (int pw = cw; pw < PW; pw += kTmaConsumers) {
          const int nx = Tb.xcnt[pw];
          float acc[VN];
#pragma unroll
          for (int j = 0; j < VN; ++j) acc[j] = 0.0f;
          if (act && staged && ny > 0 && nx > 0) {
            int xo[4];
            float xw[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { const TmaTap e = Tb.xtap[pw][q]; xo[q] = e.pix * kTmaChunkBytes; xw[q] = e.w; }
            switch (ny) {
              case 1: tma_dispatch_x<T, 1>(nx, rp, yw, xo, xw, acc); break;
              case 2: tma_dispatch_x<T, 2>(nx, rp, yw, xo, xw, acc); break;
              case 3: tma_dispatch_x<T, 3>(nx, rp, yw, xo, xw, acc); break;
              default: tma_dispatch_x<T, 4>(nx, rp, yw, xo, xw, acc); break;
            }
            Vec16<T>::store(out_k + ph * os_h + pw * os_w, acc);
          } else if (act) {
            for (int qa = 0; qa < ny; ++qa) {
              const TmaTap ey = Tb.ytap[ph][qa];
              const unsigned char* srow = staged ? &S.ring[(g0 + Tb.yseq[ph][qa]) % kTmaSlots][lane * 16] : nullptr;
              const T* grow = gbase + (int64_t)ey.pix * sh;
              for (int qb = 0; qb < nx; ++qb) {
                const TmaTap ex = Tb.xtap[pw][qb];
                uint4 raw;
                if (staged) raw = *reinterpret_cast<const uint4*>(srow + ex.pix * kTmaChunkBytes);
                else raw = __ldg(reinterpret_cast<const uint4*>(grow + (int64_t)ex.pix * sw));
                float v[VN];
                Cvt16<T>::widen(raw, v);
                const float w = ey.w * ex.w;
#pragma unroll
                for (int j = 0; j < VN; ++j) acc[j] = fmaf(w, v[j], acc[j]);
              }
            }
            Vec16<T>::store(out_k + ph * os_h + pw * os_w, acc);
          }
        }
        if (staged) {   // hand back the rows no later bin row needs
          const int newrel = Tb.ylo[ph + 1];
          __syncwarp();
          while (rel < newrel) {
            if (lane == 0) mbar_arrive(&S.empty[(g0 + (unsigned)rel) % kTmaSlots]);
            ++rel;
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&S.tempty[buf]);
      if (staged) g0 += (unsigned)nrows;
    }
  }
}

template <typename T>
static int forward_tma_typed(const LevelsParam& lv, const RoiArgs& a, void* out, const int64_t* os,
                             cudaStream_t stream) {
  const int chunks = (lv.c * (int)sizeof(T) + kTmaChunkBytes - 1) / kTmaChunkBytes;
  const size_t smem = sizeof(TmaSmem) + 128;
  static int sm_count = 0;
  if (sm_count == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
      return RAF_ERR_CUDA;
  }
  if (cudaFuncSetAttribute(fwd_tma_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return RAF_ERR_CUDA;
  const int64_t items = (int64_t)a.K * chunks;
  const unsigned grid = (unsigned)(items < 2 * sm_count ? items : 2 * sm_count);
  fwd_tma_kernel<T><<<grid, kTmaThreads, smem, stream>>>(lv, a, reinterpret_cast<T*>(out), os[0], os[2], os[3], chunks);
  count_launch();
  return cudaGetLastError() == cudaSuccess ? RAF_OK : RAF_ERR_CUDA;
}

// Channels-last, sampling_ratio 1 or 2, PH + PW <= 32, PH, PW <= 16; RAF_ERR_UNSUPPORTED otherwise.
int launch_forward_tma(const LevelsParam& lv, raf_dtype dtype, const RoiArgs& a, void* out,
                       const int64_t* out_strides, cudaStream_t stream) {
  if (a.sampling_ratio < 1 || a.sampling_ratio > 2 || a.PH > kTmaMaxBins || a.PW > kTmaMaxBins || a.PH + a.PW > 32)
    return RAF_ERR_UNSUPPORTED;
  switch (dtype) {
    case RAF_F32: return forward_tma_typed<float>(lv, a, out, out_strides, stream);
    case RAF_F16: return forward_tma_typed<__half>(lv, a, out, out_strides, stream);
    case RAF_BF16: return forward_tma_typed<__nv_bfloat16>(lv, a, out, out_strides, stream);
  }
  return RAF_ERR_DTYPE;
}

}  // namespace raf
