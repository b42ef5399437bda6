// a1 decimator (Eq. 4), the basis-domain polyphase upsampler (Eqs. 7-9)
// and the peak finalisation.  FP32 CUDA-core kernels shared by every precision mode:
// they are latency/HBM-bound stages, not contractions.
#include <cmath>

#include <cuda_fp8.h>

#include "lloid_internal.h"

namespace lloid {

// ------------------------------------------------------------------------------------------------
// K1: append the pushed strain to the f0 ring and decimate it to every lower rate.
//   d_r[j] = sum_k taps[k] * d[j*D + c - k], taps = sqrt(D)*ghat (host, float64 -> fp32), zero phase.
//   New outputs of a push: j in [n0/D - n_down, (n0+B)/D - n_down)  (needs c future f0 samples).
//   DEC_PER_CTA outputs per CTA; thread t sums taps t, t+256, ... then a fixed-order reduction: deterministic.
// ------------------------------------------------------------------------------------------------
#define DEC_PER_CTA 8
#define DEC_WIN (2 * 32 * 64 + 1 + (DEC_PER_CTA - 1) * 64 + 3)   // staged strain span: n_down = 32, D <= 64
__global__ void __launch_bounds__(256) decimate_kernel(const DecimParams P, const float *__restrict__ strain,
                                                       const long long *__restrict__ n0_ptr) {
  const long long n0 = *n0_ptr;
  const int det = blockIdx.y;
  const float *sd = strain + (size_t)det * P.B;
  const RateDev &r0 = P.r[0];
  float *ring0 = r0.ring2 + (size_t)det * 2 * r0.rlen;
  if ((int)blockIdx.x < P.copy_blocks) {
    // f0 ring append (both mirror halves)
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.B; i += P.copy_blocks * blockDim.x) {
      int slot = (int)((n0 + i) % r0.rlen);
      float v = sd[i];
      ring0[slot] = v;
      ring0[slot + r0.rlen] = v;
    }
    return;
  }
  // DEC_PER_CTA consecutive outputs of ONE rate per CTA (out_begin is padded to a multiple of DEC_PER_CTA).  The 256
  // threads split the taps; each thread carries all DEC_PER_CTA accumulators so its loads are independent.  Partial
  // sums are reduced in a fixed order (lane tree, then warps 0..7): deterministic.
  __shared__ float part[DEC_PER_CTA][8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int o0 = (blockIdx.x - P.copy_blocks) * DEC_PER_CTA;
  if (o0 >= P.total_out) return;
  int ri = 1;
  while (ri + 1 < P.n_rates && o0 >= P.r[ri + 1].out_begin) ++ri;
  const RateDev &r = P.r[ri];
  const int first = o0 - r.out_begin;                      // first output of this CTA within the push
  if (first >= r.n_out) return;
  const long long j0 = n0 / r.D - r.lag + first;
  const long long top0 = j0 * r.D + r.c;                   // f0 index read by tap k = 0 of output j0
  const int ntap = 2 * r.c + 1, D = r.D, rlen0 = r0.rlen;
  const float *__restrict__ taps = r.taps;
  float acc[DEC_PER_CTA];
#pragma unroll
  for (int oi = 0; oi < DEC_PER_CTA; ++oi) acc[oi] = 0.f;
  // The CTA's outputs read the contiguous strain span [top0 - 2c, top0 + (DEC_PER_CTA-1) D] (<= 4545 samples for D = 64):
  // stage it in shared memory with one round of coalesced loads (below n0 it lives in the f0 ring, below 0 it is zero),
  // then every (output, tap) product reads shared memory.  win[i] = d[top0 - 2c + i].
  __shared__ float win[DEC_WIN];
  const long long base = top0 - 2LL * r.c;                 // stream index of win[0]
  const int nwin = ntap + (DEC_PER_CTA - 1) * D;
  const int ring_base = (int)(((n0 % rlen0) + rlen0) % rlen0);   // ring slot of stream sample n0
  auto strain_at = [&](long long idx) {
    const long long rel = idx - n0;
    if (rel >= 0) return rel < P.B ? sd[rel] : 0.f;       // beyond the pushed buffer: outputs that do not exist (discarded)
    if (idx < 0) return 0.f;
    long long sl = ring_base + rel;                        // rel in (-rlen0, 0): one wrap at most
    if (sl < 0) sl += rlen0;
    return ring0[sl];
  };
  if (nwin > DEC_WIN) {
    // very long filters (n_down * D beyond the staged window): read the strain directly
    for (int k = threadIdx.x; k < ntap; k += 256) {
      const float t = taps[k];
#pragma unroll
      for (int oi = 0; oi < DEC_PER_CTA; ++oi) acc[oi] = fmaf(t, strain_at(top0 + (long long)oi * D - k), acc[oi]);
    }
  } else {
  for (int i = threadIdx.x; i < nwin; i += 256) {
    const long long idx = base + i, rel = idx - n0;
    float v;
    if (rel >= 0) v = rel < P.B ? sd[rel] : 0.f;            // never read past the caller's [n_det][B] buffer
    else if (idx < 0) v = 0.f;
    else {
      long long sl = ring_base + rel;                      // rel in (-rlen0, 0): one wrap at most
      if (sl < 0) sl += rlen0;
      v = ring0[sl];
    }
    win[i] = v;
  }
  __syncthreads();
  for (int k = threadIdx.x; k < ntap; k += 256) {
    const float t = taps[k];
    const int w0 = 2 * r.c - k;                            // tap k of output oi reads d[top0 + oi D - k] = win[w0 + oi D]
#pragma unroll
    for (int oi = 0; oi < DEC_PER_CTA; ++oi) acc[oi] = fmaf(t, win[w0 + oi * D], acc[oi]);
  }
  }
#pragma unroll
  for (int oi = 0; oi < DEC_PER_CTA; ++oi) {
    float a = acc[oi];
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) a += __shfl_xor_sync(0xffffffffu, a, s);
    if (lane == 0) part[oi][warp] = a;
  }
  __syncthreads();
  if (threadIdx.x < DEC_PER_CTA && first + (int)threadIdx.x < r.n_out) {
    const long long j = j0 + threadIdx.x;
    float a = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) a += part[threadIdx.x][w];
    int slot = (int)((j + r.lag) % r.rlen);
    float *ring = r.ring2 + (size_t)det * 2 * r.rlen;
    ring[slot] = a;
    ring[slot + r.rlen] = a;
  }
}

cudaError_t launch_decimate(const DecimParams &P, const float *strain, const long long *n0, cudaStream_t st) {
  int dec_blocks = (P.total_out + DEC_PER_CTA - 1) / DEC_PER_CTA;
  dim3 grid(P.copy_blocks + dec_blocks, P.n_det);
  decimate_kernel<<<grid, 256, 0, st>>>(P, strain, n0);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// K_up: polyphase upsample chain applied in the BASIS domain.
//   Up_f is linear and acts along time, R^s acts along rows, so  Up(R^s Y^s) = R^s Up(Y^s):  the chain of
//   Eq. 9 is applied to the L^s basis outputs (not to the 2M template rows) and the reconstruction of all
//   slices becomes one contraction over the concatenated basis axis at f0.
//   Stage h -> h-1 with factor f:  out[i] = in[i/f] if i mod f == 0 (Eq. 8 case 1), else
//   sum_{k=0}^{15} in[floor(i/f) + 8 - k] * g_f[k f + (i mod f)]   (Eq. 7-8, zero-phase form).
//   CTA = (time chunk of `chunk` f0 samples, item = 32 basis rows sharing one upsample chain, detector).
//   lane = basis row (of any slice / bank with that chain: UpRow gives its source ring row and destination row).
//   Output, tensor-core modes (HALF_PLANES 1 / 2): one row of samples per basis row (fp16 plane; correction plane = two byte
//   rows per basis row).  A store instruction that fills only part of a 32-byte sector costs as much as 2-3 full ones
//   (measured: 1.3-3.0 TB/s against 6.3-7.4), and rows of one chain are never 16 neighbours on the basis axis -- so the
//   samples of a row are contiguous and the CTA stages UP_TT samples x 32 rows in shared memory, then writes them with
//   16-byte vectors, whole sectors only.  FFMA mode (HALF_PLANES 0) keeps fp32 [sample][Kpad] and stores directly.
// ------------------------------------------------------------------------------------------------
#define UP_THREADS 256
#define UP_RUN 8
#define UP_LD 8      // ring columns loaded per round and warp
#define UP_CHUNK 512  // f0 samples per CTA
// Staged levels: w_h <= (w_{h-1} - 1) / f + 18, f >= 2, so level 1 has <= chunk/2 + 17 columns and level 2 <= 154 (chunk
// 512).  Odd levels live in buffer A, even ones and the output tile in the smaller buffer B: 55 KB, four CTAs per SM.
#define UP_WA (UP_CHUNK / 2 + 20)
#define UP_WB (UP_CHUNK / 4 + 28)
#define UP_SMEM ((UP_WA + UP_WB) * 32 * 4)
#define UP_TT 128                     // samples per output tile (tensor-core layouts)
#define UP_P16 (UP_TT * 2 + 16)       // tile row pitches in bytes: odd multiples of 16, so 16-byte accesses by lane = row do not conflict
#define UP_P8 (UP_TT + 16)
#define UP_T8 (32 * UP_P16)           // byte rows start here: row = term * 32 + lane
static_assert(UP_T8 + 64 * UP_P8 <= UP_WB * 32 * 4, "the output tile must fit staging buffer B");

// the two correction bytes of DESIGN.md section 4 for a value v whose fp16 rounding is hf: e5m2(4 (v - hf)), e5m2(hf / 256)
__device__ __forceinline__ unsigned short up_pair_lo(float v0, float h0, float v1, float h1) {
  return __nv_cvt_float2_to_fp8x2(make_float2((v0 - h0) * 4.f, (v1 - h1) * 4.f), __NV_SATFINITE, __NV_E5M2);
}
__device__ __forceinline__ unsigned short up_pair_hi(float h0, float h1) {
  return __nv_cvt_float2_to_fp8x2(make_float2(h0 * (1.f / 256.f), h1 * (1.f / 256.f)), __NV_SATFINITE, __NV_E5M2);
}
// one sample of row `lane` into the tile
template <int HALF_PLANES>
__device__ __forceinline__ void tile_put(unsigned char *tile, int lane, int tc, float v) {
  const __half h = __float2half_rn(v);
  *reinterpret_cast<__half *>(tile + lane * UP_P16 + tc * 2) = h;
  if (HALF_PLANES == 2) {
    const float hf = __half2float(h);
    tile[UP_T8 + lane * UP_P8 + tc] = (unsigned char)__nv_cvt_float_to_fp8((v - hf) * 4.f, __NV_SATFINITE, __NV_E5M2);
    tile[UP_T8 + (32 + lane) * UP_P8 + tc] = (unsigned char)__nv_cvt_float_to_fp8(hf * (1.f / 256.f), __NV_SATFINITE, __NV_E5M2);
  }
}
// eight consecutive samples (tc a multiple of 8): one 16-byte and two 8-byte shared stores
template <int HALF_PLANES>
__device__ __forceinline__ void tile_put8(unsigned char *tile, int lane, int tc, const float (&v)[8]) {
  uint32_t w[4], a[2], b[2];
  unsigned short pa[4], pb[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const __half2 h2 = __floats2half2_rn(v[2 * i], v[2 * i + 1]);
    w[i] = *reinterpret_cast<const uint32_t *>(&h2);
    if (HALF_PLANES == 2) {
      const float2 f = __half22float2(h2);
      pa[i] = up_pair_lo(v[2 * i], f.x, v[2 * i + 1], f.y);
      pb[i] = up_pair_hi(f.x, f.y);
    }
  }
  *reinterpret_cast<uint4 *>(tile + lane * UP_P16 + tc * 2) = make_uint4(w[0], w[1], w[2], w[3]);
  if (HALF_PLANES == 2) {
    a[0] = pa[0] | ((uint32_t)pa[1] << 16); a[1] = pa[2] | ((uint32_t)pa[3] << 16);
    b[0] = pb[0] | ((uint32_t)pb[1] << 16); b[1] = pb[2] | ((uint32_t)pb[3] << 16);
    *reinterpret_cast<uint2 *>(tile + UP_T8 + lane * UP_P8 + tc) = make_uint2(a[0], a[1]);
    *reinterpret_cast<uint2 *>(tile + UP_T8 + (32 + lane) * UP_P8 + tc) = make_uint2(b[0], b[1]);
  }
}
// FFMA mode: fp32 [sample][Kpad]
__device__ __forceinline__ void up_store_f32(void *yup, size_t o, float v) { reinterpret_cast<float *>(yup)[o] = v; }

template <int HALF_PLANES>
__global__ void __launch_bounds__(UP_THREADS, HALF_PLANES == 0 ? 3 : 4) upsample_kernel(const UpItem *__restrict__ items, const UpRow *__restrict__ rows, int B, int chunk,
                                                          const float *__restrict__ uptaps,
                                                          const int *__restrict__ uptap_off,
                                                          const long long *__restrict__ n0_ptr, const UpTaps2 taps2) {
  static_assert(UP_LD == 8, "tile_put8 takes the UP_LD columns of one load round");
  extern __shared__ __align__(16) float up_dyn[];
  float(*bufA)[32] = reinterpret_cast<float(*)[32]>(up_dyn), (*bufB)[32] = bufA + UP_WA;    // level h: A if h is odd, else B
  __shared__ int s_r0[LLOID_MAX_GROUPS + 1], s_w[LLOID_MAX_GROUPS + 1], s_lf[LLOID_MAX_GROUPS + 1], s_slot0;
  __shared__ unsigned char *s_dst16[32], *s_dst8[32];     // tensor-core layouts: where sample ka of each lane's row goes
  const UpItem *it = &items[blockIdx.y];
  const int det = blockIdx.z;
  const int ka = blockIdx.x * chunk;
  const int kb = min(ka + chunk, B);
  constexpr int nwarp = UP_THREADS / 32;                       // compile-time: the run partition divides by it
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int G = it->g, nl = it->nl;
  const bool active = lane < nl;
  const UpRow *rw = &rows[it->row0 + (active ? lane : 0)];     // this lane's row: source ring row and destination
  const int ylen = it->ylen, ypitch = rw->ypitch;
  const int kpitch = rw->kpitch;                               // FFMA: Kpad (sample pitch); tensor-core layouts: yup_pitch(B) (row pitch)
  void *yup = rw->yup;
  const size_t rowoff = (size_t)det * rw->yup_det_stride + (size_t)rw->dst0;
  const size_t out0 = rowoff + (size_t)ka * kpitch;            // FFMA: element (sample ka, this row's column)
  if (HALF_PLANES > 0 && warp == 0) {
    s_dst16[lane] = reinterpret_cast<unsigned char *>(yup) + 2 * (rowoff + ka);
    s_dst8[lane] = reinterpret_cast<unsigned char *>(yup) + 2 * ((size_t)rw->yup_plane_stride + rowoff) + ka;
  }
  // Level h covers the absolute index range [lo_h, hi_h) at its rate (64-bit, thread 0 only); everything the
  // loops below need is relative and fits 32 bits: width w_h, phase r0_h = lo_{h-1} mod f_h of the first output of
  // stage h, and the Y-ring slot of column lo_G.  lo_h = floor(lo_{h-1} / f_h) - 8, hi_h = floor((hi_{h-1} - 1) / f_h) + 9.
  if (threadIdx.x == 0) {
    long long lo = *n0_ptr + ka, hi = *n0_ptr + kb;
    s_w[0] = (int)(hi - lo);
    for (int h = 1; h <= G; ++h) {
      const int lf = it->log2f[h];
      s_lf[h] = lf;
      s_r0[h] = (int)(lo & ((1 << lf) - 1));
      lo = (lo >> lf) - LLOID_NUP;                   // arithmetic shift = floor division
      hi = ((hi - 1) >> lf) + LLOID_NUP + 1;
      s_w[h] = (int)(hi - lo);
    }
    s_slot0 = (int)((lo + 64) % ylen);
  }
  __syncthreads();
  const float *yr = rw->ysrc + (size_t)det * rw->ydet_stride;
  const int nseg = rw->nseg;
  const size_t yseg = (size_t)rw->yseg_stride;
  // UP_LD consecutive ring columns from c0 on: all (column, tap segment) loads are issued before any add (memory-level
  // parallelism is what the load phase needs); the split-K partial sums are then added in segment order (deterministic,
  // the same order for every caller).  Columns never computed at stream start are the ring's zeros.
  auto load_yn = [&](int c0, int c_end, float (&v)[UP_LD]) {
    unsigned off[UP_LD];                                      // element offsets inside one (segment, detector) ring: < 2^31 (checked at create)
    const int slot = (s_slot0 + c0) % ylen;
    const int nok = active ? min(UP_LD, c_end - c0) : 0;      // columns [c0, c0 + nok) exist
#pragma unroll
    for (int i = 0; i < UP_LD; ++i) {
      const int sl = slot + i >= ylen ? slot + i - ylen : slot + i;
      off[i] = (unsigned)sl * (unsigned)ypitch;
      v[i] = 0.f;
    }
    const float *ys = yr;
    for (int sg0 = 0; sg0 < nseg; sg0 += 2, ys += 2 * yseg) {
      const float *ys1 = ys + yseg;
      float t[UP_LD][2];
      if (nok == UP_LD && sg0 + 1 < nseg) {                   // the common case: no per-load predicate
#pragma unroll
        for (int i = 0; i < UP_LD; ++i) t[i][0] = __ldg(ys + off[i]);
#pragma unroll
        for (int i = 0; i < UP_LD; ++i) t[i][1] = __ldg(ys1 + off[i]);
      } else {
        const int nok1 = sg0 + 1 < nseg ? nok : 0;
#pragma unroll
        for (int i = 0; i < UP_LD; ++i) t[i][0] = i < nok ? __ldg(ys + off[i]) : 0.f;
#pragma unroll
        for (int i = 0; i < UP_LD; ++i) t[i][1] = i < nok1 ? __ldg(ys1 + off[i]) : 0.f;
      }
#pragma unroll
      for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int i = 0; i < UP_LD; ++i) v[i] += t[i][j];
    }
  };
  // tile -> global: 16-byte vectors, a warp instruction covers UP_TT samples of 32 / (UP_TT / 8) fp16 rows or twice as many byte rows
  auto flush = [&](const unsigned char *tile, int c_lo, int ncol) {
    constexpr int L16 = UP_TT / 8, L8 = UP_TT / 16;          // lanes per row
    constexpr int R16 = nwarp * (32 / L16), R8 = nwarp * (32 / L8);   // rows per pass of the CTA
    const bool whole = ncol == UP_TT;                        // (a ragged tile: buffer_len not a multiple of UP_TT)
    const int tc16 = (lane % L16) * 8, tc8 = (lane % L8) * 16;
#pragma unroll
    for (int p = 0; p < 32 / R16; ++p) {
      const int r = p * R16 + warp * (32 / L16) + lane / L16;
      if (r < nl) {
        unsigned char *dst = s_dst16[r] + 2 * (c_lo + tc16);
        const unsigned char *src = tile + r * UP_P16 + 2 * tc16;
        if (whole || tc16 + 8 <= ncol) *reinterpret_cast<uint4 *>(dst) = *reinterpret_cast<const uint4 *>(src);
        else
          for (int j = 0; j < 8; ++j)
            if (tc16 + j < ncol) reinterpret_cast<unsigned short *>(dst)[j] = reinterpret_cast<const unsigned short *>(src)[j];
      }
    }
    if (HALF_PLANES == 2) {
#pragma unroll
      for (int p = 0; p < 64 / R8; ++p) {
        const int rr = p * R8 + warp * (32 / L8) + lane / L8;                // rr = term * 32 + row
        const int r = rr & 31;
        if (r < nl) {
          unsigned char *dst = s_dst8[r] + (size_t)(rr >> 5) * kpitch + c_lo + tc8;
          const unsigned char *src = tile + UP_T8 + rr * UP_P8 + tc8;
          if (whole || tc8 + 16 <= ncol) *reinterpret_cast<uint4 *>(dst) = *reinterpret_cast<const uint4 *>(src);
          else
            for (int j = 0; j < 16; ++j)
              if (tc8 + j < ncol) dst[j] = src[j];
        }
      }
    }
  };

  if (G == 0) {                                              // full-rate rows: converted and stored as they are
    const int w0 = s_w[0];
    if (HALF_PLANES == 0) {
      for (int c0 = warp * UP_LD; c0 < w0; c0 += UP_LD * nwarp) {
        float v[UP_LD];
        load_yn(c0, w0, v);
#pragma unroll
        for (int i = 0; i < UP_LD; ++i)
          if (active && c0 + i < w0) up_store_f32(yup, out0 + (size_t)(c0 + i) * kpitch, v[i]);
      }
    } else {
      unsigned char *tile = reinterpret_cast<unsigned char *>(bufB);
      for (int c_lo = 0; c_lo < w0; c_lo += UP_TT) {
        const int c_hi = min(c_lo + UP_TT, w0);
        for (int c0 = c_lo + warp * UP_LD; c0 < c_hi; c0 += UP_LD * nwarp) {
          float v[UP_LD];
          load_yn(c0, c_hi, v);
          if (c0 + UP_LD <= c_hi) tile_put8<HALF_PLANES>(tile, lane, c0 - c_lo, v);
          else {
#pragma unroll
            for (int i = 0; i < UP_LD; ++i)
              if (c0 + i < c_hi) tile_put<HALF_PLANES>(tile, lane, c0 + i - c_lo, v[i]);
          }
        }
        __syncthreads();
        flush(tile, c_lo, c_hi - c_lo);
        if (c_hi < w0) __syncthreads();
      }
    }
    return;
  }

  // level G from the Y ring
  const int wg = s_w[G];
  float(*lvG)[32] = (G & 1) ? bufA : bufB;
  for (int c0 = warp * UP_LD; c0 < wg; c0 += UP_LD * nwarp) {
    float v[UP_LD];
    load_yn(c0, wg, v);
#pragma unroll
    for (int i = 0; i < UP_LD; ++i)
      if (c0 + i < wg) lvG[c0 + i][lane] = v[i];
  }
  __syncthreads();
  // The run of one warp: UP_RUN consecutive inputs qq = q0 + u of a stage, held in registers with their 15 neighbours:
  // in[qq + 8 - k] = X[u + 15 - k] (in[qq] sits at buffer index qq + 8): ~3 shared loads per 16 FMA, no per-tap index arithmetic.
  // x2 stage: taps g_2[2k+1] come from the kernel parameter (constant bank), FFMA with a constant operand.
#define UP_LOAD_RUN()                                                                              \
  const int nrun = min(UP_RUN, qb - q0);                                                           \
  float X[UP_RUN + 15];                                                                            \
  if (nrun == UP_RUN) {                                     /* warp-uniform: no per-element predicate */   \
    _Pragma("unroll") for (int j = 0; j < UP_RUN + 15; ++j) X[j] = in[q0 + 1 + j][lane];           \
  } else {                                                                                         \
    _Pragma("unroll") for (int j = 0; j < UP_RUN + 15; ++j) X[j] = (j < nrun + 15) ? in[q0 + 1 + j][lane] : 0.f; \
  }                                                                                                \
  const int cbase = (q0 << lf) - r0;                        /* output index of (u = 0, phase 0) */
#define UP_ODD_X2()                                                                                \
  float odd[UP_RUN];                                                                               \
  _Pragma("unroll") for (int u = 0; u < UP_RUN; ++u) {                                             \
    float v0 = 0.f, v1 = 0.f;                                                                      \
    _Pragma("unroll") for (int k = 0; k < 16; k += 2) {                                            \
      v0 = fmaf(X[u + 15 - k], taps2.t[k], v0);                                                    \
      v1 = fmaf(X[u + 14 - k], taps2.t[k + 1], v1);                                                \
    }                                                                                              \
    odd[u] = v0 + v1;                                                                              \
  }

  for (int h = G; h >= 2; --h) {                             // stages that stay in shared memory
    const int lf = s_lf[h], f = 1 << lf, r0 = s_r0[h], wout = s_w[h - 1];
    // Output c (relative to lo_{h-1}) has input index qq = (r0 + c) >> lf relative to floor(lo_{h-1}/f) and phase
    // (r0 + c) & (f-1).  Each warp takes consecutive qq in runs of UP_RUN (a multiple of UP_RUN per warp, so only the
    // last warp's last run is ragged).
    const int nq = ((r0 + wout - 1) >> lf) + 1, per = ((nq + nwarp - 1) / nwarp + UP_RUN - 1) / UP_RUN * UP_RUN;
    const int qa = warp * per, qb = min(qa + per, nq);
    const float(*in)[32] = (h & 1) ? bufA : bufB;
    float(*out)[32] = (h & 1) ? bufB : bufA;
    for (int q0 = qa; q0 < qb; q0 += UP_RUN) {
      UP_LOAD_RUN()
      if (f == 2) {
        UP_ODD_X2()
        if (nrun == UP_RUN && cbase >= 0 && cbase + 2 * UP_RUN <= wout) {    // warp-uniform
#pragma unroll
          for (int u = 0; u < UP_RUN; ++u) {
            out[cbase + 2 * u][lane] = X[u + 7];                                 // phase 0: the copy of Eq. 8 case 1
            out[cbase + 2 * u + 1][lane] = odd[u];
          }
        } else {
#pragma unroll
          for (int u = 0; u < UP_RUN; ++u) {
            const int c0 = cbase + 2 * u;
            if (u < nrun) {
              if (c0 >= 0 && c0 < wout) out[c0][lane] = X[u + 7];
              if (c0 + 1 >= 0 && c0 + 1 < wout) out[c0 + 1][lane] = odd[u];
            }
          }
        }
      } else {
        const float *g = uptaps + uptap_off[lf];
#pragma unroll
        for (int u = 0; u < UP_RUN; ++u) {
          if (u < nrun) {
            for (int ph = 0; ph < f; ++ph) {
              float v0 = 0.f, v1 = 0.f;
              if (ph == 0) v0 = X[u + 7];
              else {
#pragma unroll
                for (int k = 0; k < 16; k += 2) {
                  v0 = fmaf(X[u + 15 - k], g[k * f + ph], v0);
                  v1 = fmaf(X[u + 14 - k], g[(k + 1) * f + ph], v1);
                }
              }
              const int c = cbase + (u << lf) + ph;
              if (c >= 0 && c < wout) out[c][lane] = v0 + v1;
            }
          }
        }
      }
    }
    __syncthreads();
  }

  // last stage (to f0).  FFMA mode stores every output directly; the tensor-core layouts go through the tile, UP_TT output
  // samples at a time (the staging buffer not read by this stage), every warp taking its share of each tile's runs.
  {
    const int lf = s_lf[1], f = 1 << lf, r0 = s_r0[1], wout = s_w[0];
    const float(*in)[32] = bufA;
    unsigned char *tile = reinterpret_cast<unsigned char *>(bufB);
    const float *g = uptaps + uptap_off[lf];
    const int tt = HALF_PLANES == 0 ? wout : UP_TT;
    for (int c_lo = 0; c_lo < wout; c_lo += tt) {
      const int c_hi = min(c_lo + tt, wout);
      const int q_lo = (r0 + c_lo) >> lf, q_hi = ((r0 + c_hi - 1) >> lf) + 1;
      const int per = ((q_hi - q_lo + nwarp - 1) / nwarp + UP_RUN - 1) / UP_RUN * UP_RUN;
      const int qa = q_lo + warp * per, qb = min(qa + per, q_hi);
      for (int q0 = qa; q0 < qb; q0 += UP_RUN) {
        UP_LOAD_RUN()
        if (f == 2) {
          UP_ODD_X2()
          const bool full = nrun == UP_RUN && cbase >= c_lo && cbase + 2 * UP_RUN <= c_hi;    // warp-uniform
          if (HALF_PLANES == 0) {
            if (active) {
#pragma unroll
              for (int u = 0; u < UP_RUN; ++u) {
                const int c0 = cbase + 2 * u;
                if (u < nrun) {
                  if (full || (c0 >= c_lo && c0 < c_hi)) up_store_f32(yup, out0 + (size_t)c0 * kpitch, X[u + 7]);
                  if (full || (c0 + 1 >= c_lo && c0 + 1 < c_hi)) up_store_f32(yup, out0 + (size_t)(c0 + 1) * kpitch, odd[u]);
                }
              }
            }
          } else if (full && ((cbase - c_lo) & 7) == 0) {
#pragma unroll
            for (int hh = 0; hh < 2; ++hh) {
              float v[8];
#pragma unroll
              for (int u = 0; u < 4; ++u) { v[2 * u] = X[4 * hh + u + 7]; v[2 * u + 1] = odd[4 * hh + u]; }
              tile_put8<HALF_PLANES>(tile, lane, cbase - c_lo + 8 * hh, v);
            }
          } else {
#pragma unroll
            for (int u = 0; u < UP_RUN; ++u) {
              const int c0 = cbase + 2 * u;
              if (u < nrun) {
                if (c0 >= c_lo && c0 < c_hi) tile_put<HALF_PLANES>(tile, lane, c0 - c_lo, X[u + 7]);
                if (c0 + 1 >= c_lo && c0 + 1 < c_hi) tile_put<HALF_PLANES>(tile, lane, c0 + 1 - c_lo, odd[u]);
              }
            }
          }
        } else {
#pragma unroll
          for (int u = 0; u < UP_RUN; ++u) {
            if (u < nrun) {
              for (int ph = 0; ph < f; ++ph) {
                float v0 = 0.f, v1 = 0.f;
                if (ph == 0) v0 = X[u + 7];
                else {
#pragma unroll
                  for (int k = 0; k < 16; k += 2) {
                    v0 = fmaf(X[u + 15 - k], g[k * f + ph], v0);
                    v1 = fmaf(X[u + 14 - k], g[(k + 1) * f + ph], v1);
                  }
                }
                const int c = cbase + (u << lf) + ph;
                if (c >= c_lo && c < c_hi) {
                  if (HALF_PLANES == 0) { if (active) up_store_f32(yup, out0 + (size_t)c * kpitch, v0 + v1); }
                  else tile_put<HALF_PLANES>(tile, lane, c - c_lo, v0 + v1);
                }
              }
            }
          }
        }
      }
      if (HALF_PLANES > 0) {
        __syncthreads();
        flush(tile, c_lo, c_hi - c_lo);
        if (c_hi < wout) __syncthreads();
      }
    }
  }
#undef UP_LOAD_RUN
#undef UP_ODD_X2
}

// Per-device kernel attributes (dynamic shared memory opt-in) and the x2 taps: called by every lloid_stream_create on
// its current device (the attribute is per device/context, not per process).
cudaError_t upsample_configure(UpTaps2 *t2) {
  const int smem = UP_SMEM;
  cudaError_t e = cudaFuncSetAttribute(upsample_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(upsample_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(upsample_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  for (int k = 0; k < 16; ++k) {                         // Eq. 4 with f = 2, c = 16 (same float64 -> fp32 values as uptaps)
    const double x = (2 * k + 1) - 16.0, a = M_PI * x / 2.0, b = M_PI * x / 16.0;
    t2->t[k] = (float)((sin(a) / a) * (sin(b) / b));
  }
  return e;
}

cudaError_t launch_upsample(const UpItem *items_dev, const UpRow *rows_dev, int n_items, int n_det, int B, int chunk, const float *uptaps,
                            const int *uptap_off, const long long *n0, int out_half_planes, const UpTaps2 &t2, cudaStream_t st) {
  dim3 grid((B + chunk - 1) / chunk, n_items, n_det);
  const int smem = UP_SMEM;
  if (out_half_planes == 0) upsample_kernel<0><<<grid, UP_THREADS, smem, st>>>(items_dev, rows_dev, B, chunk, uptaps, uptap_off, n0, t2);
  else if (out_half_planes == 1) upsample_kernel<1><<<grid, UP_THREADS, smem, st>>>(items_dev, rows_dev, B, chunk, uptaps, uptap_off, n0, t2);
  else upsample_kernel<2><<<grid, UP_THREADS, smem, st>>>(items_dev, rows_dev, B, chunk, uptaps, uptap_off, n0, t2);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a5 finalisation: reduce the per-time-tile partial peaks of every template in ascending time order
// (strict '>' keeps the first maximum), then snr = sqrt(p), phase = atan2(im, re).
// Thread 0 also advances the device-side stream clock n0 by B.
// ------------------------------------------------------------------------------------------------
// With overlapped trigger windows (Fig. 5) the window of a push is [n0 - overlap, n0 + B): `tail` holds, per
// template, the peak of the PREVIOUS buffer's last `overlap` samples (index relative to that buffer); it competes with
// the current buffer's peak (being earlier it wins a tie; reported sample = index - B < 0) and is then replaced by the
// reduction of `tail_partial`, the current buffer's own tail peak.
template <int g>
__global__ void __launch_bounds__(256) finalize_kernel(const PeakPartial *__restrict__ partial, int n_det, int Mtot, int n_tt,
                                float threshold, lloid_peak *__restrict__ peaks, long long *n0, int B,
                                PeakPartial *__restrict__ tail, const PeakPartial *__restrict__ tail_partial, int overlap) {
  // The partial peaks are laid out [detector][slot][template]: for one slot the threads of a warp read consecutive
  // templates (coalesced 16-byte loads).  A block takes 256 / g (detector, template) pairs; thread (li, jj) reduces the slots
  // li, li + g, ... of pair jj, the g results meet in shared memory (g = 1 when there are enough pairs to fill the GPU).
  // "Better" = larger |z|^2, ties -> lower sample index (= the first maximum in time), so the order of the reduction is free.
  __shared__ PeakPartial red[g > 1 ? 256 : 1];
  constexpr int tpb = 256 / g;
  const int li = threadIdx.x / tpb, jj = threadIdx.x - li * tpb;
  const long long t = (long long)blockIdx.x * tpb + jj;
  if (blockIdx.x == 0 && threadIdx.x == 0) *n0 += B;
  const bool valid = t < (long long)n_det * Mtot;
  const int det = valid ? (int)(t / Mtot) : 0, j = valid ? (int)(t - (long long)det * Mtot) : 0;
  PeakPartial best;
  best.p = -2.f; best.idx = 0x7fffffff; best.re = 0.f; best.im = 0.f;
  if (valid) {
    const PeakPartial *pp = partial + (size_t)det * n_tt * Mtot + j;
#pragma unroll 4
    for (int i = li; i < n_tt; i += g) {
      const PeakPartial c = pp[(size_t)i * Mtot];
      if (c.p > best.p || (c.p == best.p && c.idx < best.idx)) best = c;
    }
  }
  if (g > 1) {
    red[threadIdx.x] = best;
    __syncthreads();
    if (li != 0) return;
    for (int i = 1; i < g; ++i) {
      const PeakPartial c = red[i * tpb + jj];
      if (c.p > best.p || (c.p == best.p && c.idx < best.idx)) best = c;
    }
  }
  if (!valid) return;
  if (tail != nullptr) {
    const PeakPartial tp = tail[t];
    if (tp.idx >= B - overlap && tp.idx < B && tp.p >= best.p) { best = tp; best.idx = tp.idx - B; }
    PeakPartial nt;
    nt.p = -3.f; nt.idx = 0x7fffffff; nt.re = 0.f; nt.im = 0.f;
    for (int i = 0; i < 4; ++i) {
      const PeakPartial c = tail_partial[((size_t)det * 4 + i) * Mtot + j];
      if (c.p > nt.p || (c.p == nt.p && c.idx < nt.idx)) nt = c;
    }
    tail[t] = nt;
  }
  lloid_peak o;
  o.snr = sqrtf(fmaxf(best.p, 0.f));
  o.sample = best.idx;
  o.phase = atan2f(best.im, best.re);
  if (threshold > 0.f && o.snr < threshold) { o.snr = 0.f; o.sample = LLOID_NO_TRIGGER; o.phase = 0.f; }
  peaks[t] = o;
}

// xi^2 support: copy this push's upsampled Y into slot `slot` of the three-buffer history ring (16-byte vectors)
__global__ void yup_copy_kernel(const YupCopy *__restrict__ table, int slot) {
  const YupCopy c = table[blockIdx.y];
  uint4 *dst = c.dst + (long long)slot * c.row16;            // rows of 3 B samples: this push's B samples go to columns slot * B ...
  const long long n16 = c.n_rows * c.row16;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (long long)gridDim.x * blockDim.x) {
    const long long r = i / c.row16;
    dst[r * c.dst_pitch16 + (i - r * c.row16)] = c.src[i];
  }
}
cudaError_t launch_yup_copy(const YupCopy *table_dev, int n_pieces, int slot, cudaStream_t st) {
  if (n_pieces == 0) return cudaSuccess;
  yup_copy_kernel<<<dim3(8, n_pieces), 256, 0, st>>>(table_dev, slot);
  return cudaGetLastError();
}
// xi^2 = sum of the four column-slice partial numerators (fixed order) / sum_t (2 - 2 |R|^2); -1 where there is no trigger
__global__ void xi2_finalize_kernel(const float *__restrict__ part, const lloid_peak *__restrict__ peaks, const float *__restrict__ den,
                                    long long n, int Mtot, float *__restrict__ out) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const float4 p = reinterpret_cast<const float4 *>(part)[t];
  out[t] = peaks[t].sample == LLOID_NO_TRIGGER ? -1.f : (((p.x + p.y) + p.z) + p.w) / den[t % Mtot];
}
cudaError_t launch_xi2_finalize(const float *xi_partial, const lloid_peak *peaks, const float *den, int n_det, int Mtot, float *xi2_out,
                                cudaStream_t st) {
  const long long n = (long long)n_det * Mtot;
  xi2_finalize_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(xi_partial, peaks, den, n, Mtot, xi2_out);
  return cudaGetLastError();
}

__global__ void fill_partial_kernel(PeakPartial *partial, size_t n) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { PeakPartial e; e.p = -3.f; e.idx = 0x7fffffff; e.re = 0.f; e.im = 0.f; partial[i] = e; }
}
cudaError_t launch_fill_partial(PeakPartial *partial, size_t n, cudaStream_t st) {
  if (n == 0) return cudaSuccess;
  fill_partial_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(partial, n);
  return cudaGetLastError();
}

cudaError_t launch_finalize(const PeakPartial *partial, int n_det, int Mtot, int n_tt, float threshold,
                            lloid_peak *peaks, long long *n0, int B, PeakPartial *tail, const PeakPartial *tail_partial, int overlap,
                            cudaStream_t st) {
  const long long n = (long long)n_det * Mtot;
  int g = 1;                                                  // threads per (detector, template) pair: up to 8 while the grid is small
  while (g < 8 && 2 * g <= n_tt && n * g < 148LL * 2048) g <<= 1;
  const int tpb = 256 / g;
  const unsigned grid = (unsigned)((n + tpb - 1) / tpb);
  if (g == 1) finalize_kernel<1><<<grid, 256, 0, st>>>(partial, n_det, Mtot, n_tt, threshold, peaks, n0, B, tail, tail_partial, overlap);
  else if (g == 2) finalize_kernel<2><<<grid, 256, 0, st>>>(partial, n_det, Mtot, n_tt, threshold, peaks, n0, B, tail, tail_partial, overlap);
  else if (g == 4) finalize_kernel<4><<<grid, 256, 0, st>>>(partial, n_det, Mtot, n_tt, threshold, peaks, n0, B, tail, tail_partial, overlap);
  else finalize_kernel<8><<<grid, 256, 0, st>>>(partial, n_det, Mtot, n_tt, threshold, peaks, n0, B, tail, tail_partial, overlap);
  return cudaGetLastError();
}

}  // namespace lloid
