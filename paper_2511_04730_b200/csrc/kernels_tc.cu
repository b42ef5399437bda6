// tcgen05 (5th-generation tensor core) kernels of the LLOID path, sm_100a only:
//   a2  corr_tc_kernel   Y^s = U^s x Hankel(d_{f^s})          (Eq. 5; delays Eq. 9, 167-185)
//   a3  recon_tc_kernel  rho = R x Yup, fused |z|^2 peak search (Eq. 6; peaks 199-201)
// Operands are fp16 (optionally hi + lo split), accumulation is fp32 in tensor memory.
// U and R tiles arrive by TMA (128-byte swizzle); the Hankel operand of a2 is built on chip as a strip of
// 8 element-shifted copies so that one shared-memory matrix descriptor with LBO = SBO = 128 B addresses it.
// Warp roles: warp 0 = TMA producer, warp 1 = MMA issuer (+ TMEM allocation), warps 2-5 = strip builders (a2)
// and epilogue (TMEM -> registers -> peaks / Y ring).  Synchronisation is by mbarriers only.
#include <cuda.h>

#include <algorithm>
#include <cstring>

#include "lloid_internal.h"
#include "tc_ptx.cuh"

namespace lloid {
using namespace ptx;

static constexpr int TC_THREADS = 192;       // 6 warps
static constexpr int TILE_M = 128;           // rows of U / templates of R per tile (= UMMA M, TMEM lanes)
static constexpr int TILE_N = 128;           // max columns (time samples) per tile
static constexpr int BK = 64;                // K elements per TMA box = one 128-byte swizzled row of fp16
static constexpr int TILE_BYTES = TILE_M * BK * 2;   // 16 KB

struct TcReconTile { int bank, det, m0, t0; };
struct TcReconBank {                         // device copy, 64-byte aligned (CUtensorMap needs it)
  CUtensorMap mapR;                          // [planes*2*Mpad rows][Kpad] fp16, box 64 x 128
  CUtensorMap mapY;                          // [planes*n_det*B rows][Kpad] fp16, box 64 x 128
  int M, Mpad, Kpad, tmpl_off;
  float inv_scale;
  int pad_[11];
};
struct TcCorrTile { int cls, det, row0, col0; };
struct TcCorrClass {
  CUtensorMap mapU;                          // [planes*Lpad rows][Npad] fp16, box 64 x 128
  int pad_[32];
};

// ------------------------------------------------------------------------------------------------
// a3 + a5.  Persistent CTAs; tile = 128 templates x 128 samples of one (bank, detector); accumulators
// re / im [128 x 128] fp32 each, double buffered in TMEM (512 columns).  Per K block of 64:
//   re += Rre_hi Y_hi (+ Rre_hi Y_lo + Rre_lo Y_hi),  im likewise  -> 2 or 6 MMAs of 128x128x16 per K step.
// ------------------------------------------------------------------------------------------------
template <int PLANES>
__global__ void __launch_bounds__(TC_THREADS, 1)
recon_tc_kernel(const TcReconBank *__restrict__ banks, const TcReconTile *__restrict__ tiles, int n_tiles, int n_det, int B,
                PeakPartial *__restrict__ partial, int Mtot, int n_tt, float *__restrict__ snr_debug, int debug_bank) {
  constexpr int STAGES = PLANES == 2 ? 2 : 4;
  constexpr int STAGE_BYTES = 3 * PLANES * TILE_BYTES;        // Rre, Rim, Y per plane
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint64_t *bars = (uint64_t *)(smem + STAGES * STAGE_BYTES);
  uint64_t *full = bars, *empty = bars + STAGES, *tfull = bars + 2 * STAGES, *tempty = bars + 2 * STAGES + 2;
  uint32_t *tmem_slot = (uint32_t *)(bars + 2 * STAGES + 4);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    for (int i = 0; i < STAGES; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull[i], 1); mbar_init(&tempty[i], 4); }
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, 512);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      for (int ti = blockIdx.x; ti < n_tiles; ti += gridDim.x) {
        const TcReconTile tl = tiles[ti];
        const TcReconBank *bk = &banks[tl.bank];
        const int nkb = bk->Kpad / BK;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(&empty[stage], phase ^ 1);
          mbar_arrive_expect_tx(&full[stage], STAGE_BYTES);
          uint8_t *s = smem + stage * STAGE_BYTES;
#pragma unroll
          for (int p = 0; p < PLANES; ++p) {
            tma_load_2d(s + (3 * p + 0) * TILE_BYTES, &bk->mapR, &full[stage], kb * BK, (p * 2 + 0) * bk->Mpad + tl.m0);
            tma_load_2d(s + (3 * p + 1) * TILE_BYTES, &bk->mapR, &full[stage], kb * BK, (p * 2 + 1) * bk->Mpad + tl.m0);
            tma_load_2d(s + (3 * p + 2) * TILE_BYTES, &bk->mapY, &full[stage], kb * BK, (p * n_det + tl.det) * B + tl.t0);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer
    if (lane == 0) {
      constexpr uint32_t idesc = idesc_f16_f32(TILE_M, TILE_N);
      int stage = 0; uint32_t phase = 0; int it = 0;
      for (int ti = blockIdx.x; ti < n_tiles; ti += gridDim.x, ++it) {
        const TcReconTile tl = tiles[ti];
        const int nkb = banks[tl.bank].Kpad / BK;
        const int buf = it & 1;
        mbar_wait(&tempty[buf], ((it >> 1) & 1) ^ 1);
        tc_fence_after_sync();
        const uint32_t d_re = tmem + buf * 256, d_im = d_re + 128;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(&full[stage], phase);
          tc_fence_after_sync();
          const uint32_t s = smem_u32(smem + stage * STAGE_BYTES);
#pragma unroll
          for (int k = 0; k < BK / 16; ++k) {
            const uint32_t ko = k * 32;
            const bool acc = (kb | k) != 0;
            const uint64_t re_hi = desc_kmajor_sw128(s + 0 * TILE_BYTES + ko), im_hi = desc_kmajor_sw128(s + 1 * TILE_BYTES + ko),
                           y_hi = desc_kmajor_sw128(s + 2 * TILE_BYTES + ko);
            mma_f16_ss(d_re, re_hi, y_hi, idesc, acc);
            mma_f16_ss(d_im, im_hi, y_hi, idesc, acc);
            if (PLANES == 2) {
              const uint64_t re_lo = desc_kmajor_sw128(s + 3 * TILE_BYTES + ko), im_lo = desc_kmajor_sw128(s + 4 * TILE_BYTES + ko),
                             y_lo = desc_kmajor_sw128(s + 5 * TILE_BYTES + ko);
              mma_f16_ss(d_re, re_hi, y_lo, idesc, true);
              mma_f16_ss(d_im, im_hi, y_lo, idesc, true);
              mma_f16_ss(d_re, re_lo, y_hi, idesc, true);
              mma_f16_ss(d_im, im_lo, y_hi, idesc, true);
            }
          }
          mma_commit(&empty[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        mma_commit(&tfull[buf]);
      }
    }
  } else {
    // ===== epilogue: thread = one template (TMEM lane), 128 columns in 4 chunks of 32
    const int q = warp & 3;                       // TMEM lane quadrant this warp may access
    int it = 0;
    for (int ti = blockIdx.x; ti < n_tiles; ti += gridDim.x, ++it) {
      const TcReconTile tl = tiles[ti];
      const TcReconBank *bk = &banks[tl.bank];
      const int buf = it & 1;
      mbar_wait(&tfull[buf], (it >> 1) & 1);
      tc_fence_after_sync();
      const int m = tl.m0 + q * 32 + lane;
      const float sc = bk->inv_scale;
      const bool dbg = snr_debug != nullptr && tl.bank == debug_bank && m < bk->M;
      float *dbg_re = dbg ? snr_debug + ((size_t)tl.det * 2 * bk->M + 2 * m) * B : nullptr;
      PeakPartial best; best.p = -1.f; best.idx = 0; best.re = 0.f; best.im = 0.f;
      const uint32_t t_re = tmem + ((uint32_t)(q * 32) << 16) + buf * 256;
#pragma unroll 1
      for (int c = 0; c < TILE_N / 32; ++c) {
        uint32_t vr[32], vi[32];
        tmem_ld_32x32(t_re + c * 32, vr);
        tmem_ld_32x32(t_re + 128 + c * 32, vi);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          const int t = tl.t0 + c * 32 + i;
          const float re = __uint_as_float(vr[i]) * sc, im = __uint_as_float(vi[i]) * sc;
          const float p = re * re + im * im;
          if (t < B) {
            if (p > best.p) { best.p = p; best.idx = t; best.re = re; best.im = im; }
            if (dbg) { dbg_re[t] = re; dbg_re[B + t] = im; }
          }
        }
      }
      tc_fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tempty[buf]);
      if (m < bk->M) partial[((size_t)tl.det * Mtot + bk->tmpl_off + m) * n_tt + tl.t0 / TILE_N] = best;
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 512);
}

// ------------------------------------------------------------------------------------------------
// a2.  One tile per CTA (2 CTAs per SM): 128 stacked basis rows x NT <= 128 columns of one (class, detector);
// K = the slice's taps, walked in chunks of KS = 512.  For each chunk warps 2-5 build the Hankel strip
//   strip[m][r][e] = x[c*KS + 8 m + r + e]   (fp16; m < (NT + ks)/8, r < 8, e < 8; 128 B per m)
// from the fp32 strain ring, so that B[n][k] = x[n + k] is the no-swizzle K-major operand with
// LBO = SBO = 128 B starting at strip + 128*(k/8) bytes.  U tiles come by TMA.  The accumulator
// [128 x NT] fp32 sits in 128 TMEM columns; the epilogue scales and writes the Y ring (time-major).
// ------------------------------------------------------------------------------------------------
static constexpr int KS = 512;
static constexpr int STRIP_BYTES = (TILE_N + KS) * 16;        // one plane, one buffer: 10240 B

template <int PLANES>
__global__ void __launch_bounds__(TC_THREADS, 2)
corr_tc_kernel(const CorrClass *__restrict__ classes, const TcCorrClass *__restrict__ maps, const TcCorrTile *__restrict__ tiles,
               const long long *__restrict__ n0_ptr) {
  constexpr int STAGES = 2;
  constexpr int STAGE_BYTES = PLANES * TILE_BYTES;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t *strips = smem + STAGES * STAGE_BYTES;                 // [2 buffers][PLANES][STRIP_BYTES]
  uint64_t *bars = (uint64_t *)(strips + 2 * PLANES * STRIP_BYTES);
  uint64_t *ufull = bars, *uempty = bars + STAGES, *sfull = bars + 2 * STAGES, *sempty = sfull + 2, *accfull = sempty + 2;
  uint32_t *tmem_slot = (uint32_t *)(accfull + 1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  const TcCorrTile tl = tiles[blockIdx.x];
  const CorrClass &c = classes[tl.cls];
  const int NT = min(TILE_N, (c.ncols - tl.col0 + 15) & ~15);    // MMA N: multiple of 16
  const int nkb = c.Npad / BK;                                   // 64-tap blocks
  const int nchunk = (c.Npad + KS - 1) / KS;

  if (warp == 0 && lane == 0) {
    for (int i = 0; i < STAGES; ++i) { mbar_init(&ufull[i], 1); mbar_init(&uempty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&sfull[i], 4); mbar_init(&sempty[i], 1); }
    mbar_init(accfull, 1);
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, 128);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = *tmem_slot;

  if (warp == 0) {
    if (lane == 0) {
      const CUtensorMap *mapU = &maps[tl.cls].mapU;
      int stage = 0; uint32_t phase = 0;
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait(&uempty[stage], phase ^ 1);
        mbar_arrive_expect_tx(&ufull[stage], STAGE_BYTES);
#pragma unroll
        for (int p = 0; p < PLANES; ++p)
          tma_load_2d(smem + stage * STAGE_BYTES + p * TILE_BYTES, mapU, &ufull[stage], kb * BK, p * c.Lpad + tl.row0);
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      const uint32_t idesc = idesc_f16_f32(TILE_M, NT);
      int stage = 0; uint32_t phase = 0;
      for (int ch = 0; ch < nchunk; ++ch) {
        const int sb = ch & 1;
        mbar_wait(&sfull[sb], (ch >> 1) & 1);
        tc_fence_after_sync();
        const uint32_t strip = smem_u32(strips + sb * PLANES * STRIP_BYTES);
        const int kb_end = min(nkb, (ch + 1) * (KS / BK));
        for (int kb = ch * (KS / BK); kb < kb_end; ++kb) {
          mbar_wait(&ufull[stage], phase);
          tc_fence_after_sync();
          const uint32_t us = smem_u32(smem + stage * STAGE_BYTES);
#pragma unroll
          for (int k = 0; k < BK / 16; ++k) {
            const uint32_t koff = (uint32_t)((kb - ch * (KS / BK)) * BK + k * 16) * 16;   // 128 B per 8 taps
            const uint64_t u_hi = desc_kmajor_sw128(us + k * 32);
            const uint64_t x_hi = desc_kmajor_nosw(strip + koff, 128, 128);
            mma_f16_ss(tmem, u_hi, x_hi, idesc, (kb | k) != 0);
            if (PLANES == 2) {
              const uint64_t u_lo = desc_kmajor_sw128(us + TILE_BYTES + k * 32);
              const uint64_t x_lo = desc_kmajor_nosw(strip + STRIP_BYTES + koff, 128, 128);
              mma_f16_ss(tmem, u_hi, x_lo, idesc, true);
              mma_f16_ss(tmem, u_lo, x_hi, idesc, true);
            }
          }
          mma_commit(&uempty[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        mma_commit(&sempty[sb]);
      }
      mma_commit(accfull);
    }
  } else {
    // ===== strip builders, then epilogue (128 threads)
    const int tid = threadIdx.x - 64;
    const long long n0 = *n0_ptr;
    const long long j0 = n0 / c.D + c.H + tl.col0;                   // first column of this tile
    const long long first = j0 - c.delay - c.N + 1 + c.lag;          // ring index of tap 0 of column j0
    const int p0 = (int)(((first % c.rlen) + c.rlen) % c.rlen);
    const float *x = c.ring2 + (size_t)tl.det * c.ring_det_stride + p0;   // mirrored ring: the window is contiguous
    for (int ch = 0; ch < nchunk; ++ch) {
      const int sb = ch & 1;
      mbar_wait(&sempty[sb], ((ch >> 1) & 1) ^ 1);
      const int ks = min(KS, c.Npad - ch * KS);
      const int n_ent = NT + ks;                                      // (NT + ks)/8 core matrices x 8 rows
      uint8_t *dst = strips + sb * PLANES * STRIP_BYTES;
      const float *xs = x + ch * KS;
      for (int e = tid; e < n_ent; e += 128) {                        // entry e = 8 m + r holds x[e .. e+8)
        float v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = xs[e + i];
        __half2 h[4], l[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          h[i] = __floats2half2_rn(v[2 * i], v[2 * i + 1]);
          if (PLANES == 2) {
            float2 b = __half22float2(h[i]);
            l[i] = __floats2half2_rn(v[2 * i] - b.x, v[2 * i + 1] - b.y);
          }
        }
        *reinterpret_cast<uint4 *>(dst + (size_t)e * 16) = *reinterpret_cast<uint4 *>(h);
        if (PLANES == 2) *reinterpret_cast<uint4 *>(dst + STRIP_BYTES + (size_t)e * 16) = *reinterpret_cast<uint4 *>(l);
      }
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(&sfull[sb]);
    }
    // epilogue
    mbar_wait(accfull, 0);
    tc_fence_after_sync();
    const int q = warp & 3;
    const int row = tl.row0 + q * 32 + lane;
    float *yr = c.yring + (size_t)tl.det * c.ydet_stride;
    const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16);
    for (int cc = 0; cc < NT; cc += 32) {
      uint32_t v[32];
      tmem_ld_32x32(taddr + cc, v);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 32; ++i) {
        const int col = tl.col0 + cc + i;
        if (col < c.ncols && row < c.Lstack) {
          const int slot = (int)((j0 + cc + i + 64) % c.ylen);
          yr[(size_t)slot * c.Lpad + row] = __uint_as_float(v[i]) * c.u_scale_inv;
        }
      }
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 128);
}

// ------------------------------------------------------------------------------------------------ host side
struct TcPlan {
  int planes, n_det, B, n_tt;
  TcReconBank *rbanks_dev; TcReconTile *rtiles_dev; int n_rtiles;
  TcCorrClass *cmaps_dev; TcCorrTile *ctiles_dev; int n_ctiles;
  const CorrClass *classes_dev;
  int recon_grid, recon_smem, corr_smem;
  std::vector<void *> allocs;
};

int tc_time_splits(int B) { return (B + TILE_N - 1) / TILE_N; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

// fp16 row-major [rows][cols] (cols % 64 == 0), box = 64 columns x 128 rows, 128-byte swizzle
static bool make_map(CUtensorMap *m, const void *base, uint64_t rows, uint64_t cols) {
  EncodeTiledFn enc = get_encode();
  if (!enc) { set_error("stream_create: cuTensorMapEncodeTiled is not available from the driver"); return false; }
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols * 2};
  cuuint32_t box[2] = {BK, TILE_M};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("stream_create: cuTensorMapEncodeTiled failed (%d) for [%llu][%llu]", (int)r,
                                     (unsigned long long)rows, (unsigned long long)cols); return false; }
  return true;
}

template <typename T>
static bool plan_upload(TcPlan *p, T **dst, const std::vector<T> &h) {
  void *q = nullptr;
  size_t bytes = std::max<size_t>(h.size() * sizeof(T), 256);
  if (cudaMalloc(&q, bytes) != cudaSuccess) { set_error("stream_create: cudaMalloc of the tensor-core plan failed"); return false; }
  p->allocs.push_back(q);
  if (!h.empty() && cudaMemcpy(q, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) {
    set_error("stream_create: upload of the tensor-core plan failed"); return false;
  }
  *dst = (T *)q;
  return true;
}

void tc_plan_destroy(TcPlan *p) {
  if (!p) return;
  for (void *q : p->allocs) cudaFree(q);
  delete p;
}

int tc_plan_create(TcPlan **out, const std::vector<CorrClass> &classes, const CorrClass *classes_dev,
                   const std::vector<ReconBank> &banks, const ReconBank *, int n_det, int B, int planes) {
  *out = nullptr;
  TcPlan *p = new TcPlan();
  p->planes = planes; p->n_det = n_det; p->B = B; p->n_tt = tc_time_splits(B); p->classes_dev = classes_dev;
  // ---- a2: one tensor map per class, tiles ordered by decreasing K so the long ones start first
  std::vector<TcCorrClass> cm(classes.size());
  std::vector<TcCorrTile> ct;
  std::vector<int> order(classes.size());
  for (size_t i = 0; i < classes.size(); ++i) order[i] = (int)i;
  std::sort(order.begin(), order.end(), [&](int a, int b) { return classes[a].Npad > classes[b].Npad; });
  for (int ci : order) {
    const CorrClass &c = classes[ci];
    memset(&cm[ci], 0, sizeof(TcCorrClass));
    if (!make_map(&cm[ci].mapU, c.U16, (uint64_t)planes * c.Lpad, (uint64_t)c.Npad)) { tc_plan_destroy(p); return LLOID_ECUDA; }
    for (int det = 0; det < n_det; ++det)
      for (int r0 = 0; r0 < c.Lstack; r0 += TILE_M)
        for (int c0 = 0; c0 < c.ncols; c0 += TILE_N) ct.push_back({ci, det, r0, c0});
  }
  p->n_ctiles = (int)ct.size();
  // ---- a3: two tensor maps per bank; tiles ordered (bank, template tile, detector, time tile)
  std::vector<TcReconBank> rb(banks.size());
  std::vector<TcReconTile> rt;
  for (size_t b = 0; b < banks.size(); ++b) {
    const ReconBank &k = banks[b];
    memset(&rb[b], 0, sizeof(TcReconBank));
    if (!make_map(&rb[b].mapR, k.R16, (uint64_t)planes * 2 * k.Mpad, (uint64_t)k.Kpad) ||
        !make_map(&rb[b].mapY, k.yup, (uint64_t)planes * n_det * B, (uint64_t)k.Kpad)) { tc_plan_destroy(p); return LLOID_ECUDA; }
    rb[b].M = k.M; rb[b].Mpad = k.Mpad; rb[b].Kpad = k.Kpad; rb[b].tmpl_off = k.tmpl_off; rb[b].inv_scale = k.inv_scale;
    for (int m0 = 0; m0 < k.M; m0 += TILE_M)
      for (int det = 0; det < n_det; ++det)
        for (int t0 = 0; t0 < B; t0 += TILE_N) rt.push_back({(int)b, det, m0, t0});
  }
  p->n_rtiles = (int)rt.size();
  if (!plan_upload(p, &p->cmaps_dev, cm) || !plan_upload(p, &p->ctiles_dev, ct) || !plan_upload(p, &p->rbanks_dev, rb) ||
      !plan_upload(p, &p->rtiles_dev, rt)) { tc_plan_destroy(p); return LLOID_ENOMEM; }
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  p->recon_grid = std::min(p->n_rtiles, sms);
  const int rstages = planes == 2 ? 2 : 4;
  p->recon_smem = rstages * 3 * planes * TILE_BYTES + 1024 + 256;
  p->corr_smem = 2 * planes * TILE_BYTES + 2 * planes * STRIP_BYTES + 1024 + 256;
  cudaError_t e;
  if (planes == 2) {
    e = cudaFuncSetAttribute(recon_tc_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->recon_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(corr_tc_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->corr_smem);
  } else {
    e = cudaFuncSetAttribute(recon_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->recon_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(corr_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->corr_smem);
  }
  if (e != cudaSuccess) { set_error("stream_create: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); tc_plan_destroy(p); return LLOID_ECUDA; }
  *out = p;
  return LLOID_OK;
}

cudaError_t tc_launch_corr(TcPlan *p, const long long *n0, cudaStream_t st) {
  if (p->n_ctiles == 0) return cudaSuccess;
  if (p->planes == 2) corr_tc_kernel<2><<<p->n_ctiles, TC_THREADS, p->corr_smem, st>>>(p->classes_dev, p->cmaps_dev, p->ctiles_dev, n0);
  else corr_tc_kernel<1><<<p->n_ctiles, TC_THREADS, p->corr_smem, st>>>(p->classes_dev, p->cmaps_dev, p->ctiles_dev, n0);
  return cudaGetLastError();
}

cudaError_t tc_launch_recon(TcPlan *p, PeakPartial *partial, int Mtot, float *snr_debug, int debug_bank, cudaStream_t st) {
  if (p->planes == 2)
    recon_tc_kernel<2><<<p->recon_grid, TC_THREADS, p->recon_smem, st>>>(p->rbanks_dev, p->rtiles_dev, p->n_rtiles, p->n_det, p->B,
                                                                         partial, Mtot, p->n_tt, snr_debug, debug_bank);
  else
    recon_tc_kernel<1><<<p->recon_grid, TC_THREADS, p->recon_smem, st>>>(p->rbanks_dev, p->rtiles_dev, p->n_rtiles, p->n_det, p->B,
                                                                         partial, Mtot, p->n_tt, snr_debug, debug_bank);
  return cudaGetLastError();
}

}  // namespace lloid
