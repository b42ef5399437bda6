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
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <queue>
#include <type_traits>

#include <cuda_fp8.h>

#include "lloid_internal.h"
#include "tc_ptx.cuh"

namespace lloid {
using namespace ptx;

static constexpr int EPI_THREADS = 512;      // a3: 16 epilogue warps
static constexpr int RECON_THREADS = 64 + EPI_THREADS + 32;   // a3: warps 0 TMA, 1 and 18 MMA (even / odd tiles), 2-17 epilogue
static constexpr int RECON_MMA2 = RECON_THREADS / 32 - 1;     // the second MMA warp
static constexpr int PK_CHUNK = 4;           // samples per peak-search chunk
static constexpr int REC_BYTES = EPI_THREADS * PK_CHUNK * 8;   // saved record chunk (re, im) per epilogue thread: 16 KB
static constexpr int TILE_M = 128;           // rows of U / templates of R per tile (= UMMA M, TMEM lanes)
static constexpr int TILE_N = 128;           // max columns (time samples) per tile
static constexpr int BK = 64;                // K elements per TMA box = one 128-byte swizzled row of fp16
static constexpr int TILE_BYTES = TILE_M * BK * 2;   // 16 KB
static constexpr int RSTEP_BYTES = 4 * 128 * 16 * 2;   // a3 resident variant: R of ONE K step (16 of K): [Rre, Rim, Rre corr, Rim corr] x 128 rows x 32 B
static constexpr int RBK_RES = 32;           // a3 resident variant: K elements per TMA box (64-byte swizzled rows)
static constexpr int RBK_STR = 64;           // a3 streaming variant: 128-byte swizzled rows (fewer barrier round trips per K)
static constexpr int RES_KMAX = 144;         // resident-R variant: the item's R tile (Kpad / 16 K steps of 16 KB) <= 144 KB
static constexpr int RMAX_STAGES = 8;        // a3 operand ring: at most 8 stages
static constexpr int RECON_SMEM_BUDGET = 232448 - 1024 - 256;   // dynamic shared memory per CTA minus alignment and barriers

struct TcReconTile { int bank, det, ndet, m0, t0, nt, slot; };   // detectors det..det+ndet-1 x nt consecutive time tiles from sample t0; partial slot
struct TcReconBank {                         // device copy, 64-byte aligned (CUtensorMap needs it)
  CUtensorMap mapR;                          // [planes*2*Mpad rows][Kpad] fp16, box 16 x 128, 32-byte swizzle (resident variant: one K step per box)
  CUtensorMap mapR64;                        // the same array, box 64 x 128, 128-byte swizzle (streaming variant)
  // upsampled Y, sample-contiguous rows: plane 0 fp16 [n_det*Kpad rows][Bp], boxes of 64 samples x
  // 32 / 64 rows; correction plane bytes [n_det*2*Kpad rows][Bp], boxes of 128 samples x 64 / 128 rows; 128-byte swizzle
  CUtensorMap mapY, mapY64, mapY8, mapY8_64;
  CUtensorMap mapYh, mapYh8;                 // xi^2: the history ring, rows of 3 B samples, boxes of the streaming variant
  const float2 *acorr;                       // xi^2: [M][2 xi_delta + 1] autocorrelations
  int M, Mpad, Kpad, tmpl_off;
  float inv_scale;
  int xi_delta;
  int pad_[8];
};
static_assert(sizeof(TcReconBank) % 64 == 0, "CUtensorMap members need 64-byte alignment");
struct XiArgs {                              // xi^2 pass (template XI): triggers of the target buffer, output, ring position
  const lloid_peak *peaks; float *partial; int row_base, ring_rows;
};
struct TcCorrClass {
  CUtensorMap mapU;                          // [planes*Lpad rows][Npad] fp16, box 64 x 128
  int pad_[32];
};

// ------------------------------------------------------------------------------------------------
// a3 + a5.  Persistent CTAs; tile = 128 templates x 128 samples of one (bank, detector); accumulators re / im
// [128 x 128] fp32 each, double buffered in TMEM (512 columns).  Per 16 of K: re += Rre_hi Y_hi, im += Rim_hi Y_hi (fp16)
// and, in split mode, one fp8 MMA each carrying both hi/lo cross terms.
// The kernel is bound by operand delivery from L2 unless R is reused (measured), so a work item is a
// (bank, 128-template tile) with a run of (detector, time tile) pairs and, in the RES variant (split mode, Kpad <=
// RES_KMAX), all K blocks of the item's R tile are loaded ONCE into a resident shared-memory region; only the
// upsampled-Y blocks stream through the ring.  The streaming variant (any Kpad) moves R and Y blocks together.
// ------------------------------------------------------------------------------------------------
template <int PLANES, bool RES, bool XI = false>
__global__ void __launch_bounds__(RECON_THREADS, 1)
recon_tc_kernel(const TcReconBank *__restrict__ banks, const TcReconTile *__restrict__ tiles, const int *__restrict__ cta_begin,
                int n_det, int B,
                PeakPartial *__restrict__ partial, int Mtot, int n_tt, float *__restrict__ snr_debug, int debug_bank,
                int ring_off, int n_stages, int t_min, XiArgs xi = XiArgs()) {
  constexpr int RBK = RES ? RBK_RES : RBK_STR;
  constexpr int RTILE_BYTES = TILE_M * RBK * 2;
  // Operand ring of K blocks of RBK (tiles of 128 rows x RBK fp16).  Streaming: NT = 3 * PLANES tiles
  // per stage (Rre, Rim, Y per plane), 4 or 8 stages.  RES: 2 tiles per stage (Y fp16, Y correction), 3 stages, after the
  // resident R region [K block][Rre, Rim, Rre corr, Rim corr].
  constexpr int NT = RES ? 2 : 3 * PLANES;
  constexpr int STAGE_BYTES = NT * RTILE_BYTES;
  const int STAGES = n_stages;                                  // <= RMAX_STAGES; the resident region [0, ring_off) comes first
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // 1024-byte aligned; stays a shared-space pointer
  uint8_t *ring = smem + ring_off;
  float4 *rec = (float4 *)(ring + STAGES * STAGE_BYTES);       // [re, im][PK_CHUNK / 4][EPI_THREADS] float4
  uint64_t *bars = (uint64_t *)((uint8_t *)rec + REC_BYTES);
  uint64_t *full = bars, *empty = bars + RMAX_STAGES, *tfull = bars + 2 * RMAX_STAGES, *tempty = tfull + 2, *rfull = tempty + 2, *rfree = rfull + 1;
  uint32_t *tmem_slot = (uint32_t *)(rfree + 1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    for (int i = 0; i < STAGES; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], 2); }   // released by both MMA warps
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull[i], 1); mbar_init(&tempty[i], EPI_THREADS / 32); }
    mbar_init(rfull, 1); mbar_init(rfree, 2);                     // both MMA warps are done with the item's R
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, 512);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = *tmem_slot;
  const int i_begin = cta_begin[blockIdx.x], i_end = cta_begin[blockIdx.x + 1];

  if (warp == 0) {
    // ===== TMA producer
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      for (int ti = i_begin; ti < i_end; ++ti) {
        const TcReconTile tl = tiles[ti];
        const TcReconBank *bk = &banks[tl.bank];
        const int nkb = (bk->Kpad + RBK - 1) / RBK;
        if (RES) {
          if (ti > i_begin) mbar_wait(rfree, (uint32_t)(ti - i_begin - 1) & 1);    // the previous item's MMAs have read R
          // resident R: one 16 KB group per K step of 16 (Kpad / 16 groups: no padding to the 32-row Y blocks, which leaves the
          // ring one more stage at Kpad = 144)
          const int nst = bk->Kpad / 16;
          mbar_arrive_expect_tx(rfull, nst * RSTEP_BYTES);
          for (int ks = 0; ks < nst; ++ks)
#pragma unroll
            for (int j = 0; j < 4; ++j) tma_load_2d(smem + ks * RSTEP_BYTES + j * (RSTEP_BYTES / 4), &bk->mapR, rfull, ks * 16, j * bk->Mpad + tl.m0);
        }
        for (int d = 0; d < tl.ndet; ++d)
        for (int tt = 0; tt < tl.nt; ++tt) {
          int ycol = tl.t0 + tt * TILE_N;                          // first sample of the tile = innermost TMA coordinate
          const int yrow = (tl.det + d) * bk->Kpad;                // first row of the detector in the fp16 plane (x2 in the byte plane)
          if (XI) {
            // history ring: sample t of the target buffer sits at column (row_base + t) mod ring_rows (t may be negative)
            ycol = (xi.row_base + ycol) % xi.ring_rows;
            if (ycol < 0) ycol += xi.ring_rows;
          }
          for (int kb = 0; kb < nkb; ++kb) {
            mbar_wait(&empty[stage], phase ^ 1);
            mbar_arrive_expect_tx(&full[stage], STAGE_BYTES);
            uint8_t *sdst = ring + stage * STAGE_BYTES;
            // Y tile = two boxes of 64 samples x RBK rows (fp16) / one box of 128 samples x 2 RBK rows (correction bytes)
            if (RES) {
              tma_load_2d(sdst, &bk->mapY, &full[stage], ycol, yrow + kb * RBK);
              tma_load_2d(sdst + RTILE_BYTES / 2, &bk->mapY, &full[stage], ycol + 64, yrow + kb * RBK);
              tma_load_2d(sdst + RTILE_BYTES, &bk->mapY8, &full[stage], ycol, 2 * (yrow + kb * RBK));
            } else {
#pragma unroll
              for (int p = 0; p < PLANES; ++p) {
                tma_load_2d(sdst + (3 * p + 0) * RTILE_BYTES, &bk->mapR64, &full[stage], kb * RBK, (p * 2 + 0) * bk->Mpad + tl.m0);
                tma_load_2d(sdst + (3 * p + 1) * RTILE_BYTES, &bk->mapR64, &full[stage], kb * RBK, (p * 2 + 1) * bk->Mpad + tl.m0);
              }
              const CUtensorMap *my = XI ? &bk->mapYh : &bk->mapY64, *my8 = XI ? &bk->mapYh8 : &bk->mapY8_64;
              tma_load_2d(sdst + 2 * RTILE_BYTES, my, &full[stage], ycol, yrow + kb * RBK);
              tma_load_2d(sdst + 2 * RTILE_BYTES + RTILE_BYTES / 2, my, &full[stage], ycol + 64, yrow + kb * RBK);
              if (PLANES == 2) tma_load_2d(sdst + 5 * RTILE_BYTES, my8, &full[stage], ycol, 2 * (yrow + kb * RBK));
            }
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
        }
      }
    }
  } else if (warp == 1 || warp == RECON_MMA2) {
    // ===== MMA issuers.  One thread keeps the tensor pipe busy only while it issues an MMA every ~64 cycles (measured: the
    // pipe queues about one instruction ahead), and each barrier round trip between K blocks or tiles (wait, fence, elect,
    // commit) is ~300 cycles of one thread's latency.  So TWO warps issue: warp 1 the even tiles of the CTA (TMEM buffer
    // 0), warp 18 the odd ones (buffer 1) -- every accumulator is still written by one thread in program order (the
    // result does not depend on timing), and one warp's round trips hide behind the other's MMAs.
    // The whole warp runs the loops (uniform control flow keeps the descriptors in uniform registers), one elected lane
    // issues the MMAs of a K block and the commits.
    // R (A operand) is K-major, upsampled Y (B operand) MN-major: rows of the Y tiles are K, samples are contiguous
    const int par = warp == 1 ? 0 : 1;
    constexpr uint32_t idesc = idesc_f16_f32(TILE_M, TILE_N) | IDESC_B_MN_MAJOR, idesc8 = idesc_f8_f32(TILE_M, TILE_N) | IDESC_B_MN_MAJOR;
    constexpr uint32_t T16 = RTILE_BYTES >> 4;                    // operand tile size in 16-byte descriptor units
    constexpr uint32_t YK16 = 2048 >> 4, YK8 = 4096 >> 4;          // one MMA of K: 16 fp16 rows / 32 byte rows of 128 B
    int stage = 0; uint32_t phase = 0; int it = 0;
    const uint64_t ring_d = desc_kmajor_sw(smem_u32(ring), RBK), res_d = desc_kmajor_sw(smem_u32(smem), 16);
    const uint64_t ring_y16 = desc_mnmajor_sw128(smem_u32(ring), RTILE_BYTES / 2), ring_y8 = desc_mnmajor_sw128(smem_u32(ring), 16);
    for (int ti = i_begin; ti < i_end; ++ti) {
      const TcReconTile tl = tiles[ti];
      const int Kpad = banks[tl.bank].Kpad, nkb = (Kpad + RBK - 1) / RBK;
      if (RES) { mbar_wait(rfull, (uint32_t)(ti - i_begin) & 1); tc_fence_after_sync(); }
      const int ntile = tl.ndet * tl.nt;
      // this warp's last tile of the item (the MMAs that read the item's resident R last), -1: it has none
      const int my_last = ntile - 1 - ((((it + ntile - 1) & 1) != par) ? 1 : 0);
      for (int tn = 0; tn < ntile; ++tn, ++it) {
        if ((it & 1) != par) {
          // The other warp's tile.  A parity wait is only sound for a waiter that cannot fall two phases behind, so this warp
          // takes part in the hand-shake of EVERY K block: it waits for the block to land and gives the stage its second
          // release (empty[] counts two arrivals: the consumer's tcgen05.commit and this one).  The blocks land before this
          // warp's own next block anyway (the producer loads in tile order), so nothing waits for the observer.
          for (int kb = 0; kb < nkb; ++kb) {
            mbar_wait(&full[stage], phase);
            if (lane == 0) mbar_arrive(&empty[stage]);
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
          continue;
        }
        const int buf = par;
        mbar_wait(&tempty[buf], ((it >> 1) & 1) ^ 1);
        tc_fence_after_sync();
        const uint32_t d_re = tmem + buf * 256, d_im = d_re + 128;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(&full[stage], phase);
          tc_fence_after_sync();
          // base descriptors; every operand tile / K step is a constant added to the 16-byte address field
          const uint64_t sd = ring_d + (uint64_t)(stage * (STAGE_BYTES >> 4));
          const uint64_t sy16 = ring_y16 + (uint64_t)(stage * (STAGE_BYTES >> 4)), sy8 = ring_y8 + (uint64_t)(stage * (STAGE_BYTES >> 4));
          const uint64_t rd = RES ? res_d + (uint64_t)(kb * 2 * (RSTEP_BYTES >> 4)) : sd;   // two K steps per Y block
          const int nk = min(RBK / 16, (Kpad - kb * RBK) / 16);    // K is padded to 16: the last box may be partly zero fill
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < RBK / 16; ++k) {
              if (k >= nk) break;
              const bool acc = (kb | k) != 0;
              if (RES) {
                const uint64_t y_hi = sy16 + YK16 * k, y_8 = sy8 + (T16 + YK8 * k);
                constexpr uint32_t RS = RSTEP_BYTES >> 4, RP = RS / 4;   // K step and plane strides of the resident R, 16-byte units
                mma_f16_ss(d_re, rd + (k * RS + 0 * RP), y_hi, idesc, acc);
                mma_f16_ss(d_im, rd + (k * RS + 1 * RP), y_hi, idesc, acc);
                mma_f8_ss(d_re, rd + (k * RS + 2 * RP), y_8, idesc8, true);
                mma_f8_ss(d_im, rd + (k * RS + 3 * RP), y_8, idesc8, true);
              } else {
                const uint64_t y_hi = sy16 + (2 * T16 + YK16 * k);
                mma_f16_ss(d_re, sd + (0 * T16 + 2 * k), y_hi, idesc, acc);
                mma_f16_ss(d_im, sd + (1 * T16 + 2 * k), y_hi, idesc, acc);
                if (PLANES == 2) {
                  // the correction planes: 16 of K as (e4m3, e4m3) pairs of R x two e5m2 byte rows of Y per basis row -> one
                  // fp8 MMA adds both cross terms R_hi Y_lo + R_lo Y_hi
                  const uint64_t y_8 = sy8 + (5 * T16 + YK8 * k);
                  mma_f8_ss(d_re, sd + (3 * T16 + 2 * k), y_8, idesc8, true);
                  mma_f8_ss(d_im, sd + (4 * T16 + 2 * k), y_8, idesc8, true);
                }
              }
            }
            mma_commit(&empty[stage]);
            if (kb == nkb - 1) mma_commit(&tfull[buf]);
            if (RES && kb == nkb - 1 && tn == my_last) mma_commit(rfree);
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
      if (RES && my_last < 0 && lane == 0) mbar_arrive(rfree);      // no tile of this item was ours: nothing of its R is in flight here
    }
  } else {
    // ===== epilogue (16 warps, four per scheduler): thread = one template (TMEM lane) x one 32-sample slice of the tile.
    // Peak search (first maximum of |z|^2): per 8-sample chunk the thread computes |z|^2 with packed
    // fp32x2 arithmetic and the chunk maximum (3-input max); only when that beats the running maximum (strict >, so an
    // earlier chunk keeps a tie) it saves the chunk's (re, im) to its shared-memory slot.  The first sample attaining the
    // maximum is located once per run from the saved chunk with the same arithmetic (bit-identical p).  The raw
    // accumulators are compared: the operand scale is a power of two, so the order is unchanged.
    const int q = warp & 3, cs = (warp - 2) >> 2, etid = threadIdx.x - 64;
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    float4 *rec_re = rec + etid, *rec_im = rec + (PK_CHUNK / 4) * EPI_THREADS + etid;   // conflict-free 16-byte slots
    const uint32_t rec_re_s = smem_u32(rec_re), rec_im_s = smem_u32(rec_im);
    int it = 0;
    for (int ti = i_begin; ti < i_end; ++ti) {
      const TcReconTile tl = tiles[ti];
      const TcReconBank *bk = &banks[tl.bank];
      const int m = tl.m0 + q * 32 + lane, M = bk->M, tmpl_off = bk->tmpl_off;
      const float sc = bk->inv_scale;
      if (XI) {
        // xi^2 pass (Eq. 10): the item covers samples [t0, t0 + 128 nt) around the target buffer; this
        // thread accumulates |z[t] - z0 R_j[t - k0]|^2 over the window of ITS template's trigger (raw accumulator scale)
        const int det = tl.det, delta = bk->xi_delta;
        lloid_peak pk; pk.snr = 0.f; pk.sample = LLOID_NO_TRIGGER; pk.phase = 0.f;
        if (m < M) pk = xi.peaks[(size_t)det * Mtot + tmpl_off + m];
        const bool has = pk.sample != LLOID_NO_TRIGGER;
        const int k0 = has ? pk.sample : 0;
        float sn, cs_;
        sincosf(pk.phase, &sn, &cs_);
        const float z0r = pk.snr * cs_ / sc, z0i = pk.snr * sn / sc;
        const float2 *R = bk->acorr + (size_t)(m < M ? m : 0) * (2 * delta + 1);
        float num = 0.f;
        for (int tt = 0; tt < tl.nt; ++tt, ++it) {
          const int buf = it & 1;
          const int tbase = tl.t0 + tt * TILE_N + cs * 32;
          mbar_wait(&tfull[buf], (it >> 1) & 1);
          tc_fence_after_sync();
          const uint32_t t_re = tmem + lane_base + buf * 256 + cs * 32;
          uint32_t vr[32], vi[32];
          tmem_ld_32x32(t_re, vr);
          tmem_ld_32x32(t_re + 128, vi);
          tmem_ld_wait();
          tc_fence_before_sync();
          __syncwarp();
          if (lane == 0) mbar_arrive(&tempty[buf]);
          if (has && tbase + 31 >= k0 - delta && tbase <= k0 + delta) {
            // sample i of the slice is autocorrelation lag u0 + i: one base pointer, constant offsets, and the window as a range
            // of i (no per-sample index arithmetic); the pointer is only dereferenced inside the row
            const int u0 = tbase - k0 + delta;
            const int i_lo = max(0, -u0), i_hi = min(32, 2 * delta + 1 - u0);
            const float2 *Rp = reinterpret_cast<const float2 *>(reinterpret_cast<const char *>(R) + (long long)u0 * (long long)sizeof(float2));
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              if (i >= i_lo && i < i_hi) {
                const float2 a = __ldg(Rp + i);
                const float dr = __uint_as_float(vr[i]) - (z0r * a.x - z0i * a.y), di = __uint_as_float(vi[i]) - (z0r * a.y + z0i * a.x);
                num = fmaf(dr, dr, fmaf(di, di, num));
              }
            }
          }
        }
        if (m < M) xi.partial[((size_t)det * Mtot + tmpl_off + m) * 4 + cs] = num * sc * sc;
        continue;
      }
      const bool dbg = snr_debug != nullptr && tl.bank == debug_bank && m < M;
      for (int d = 0; d < tl.ndet; ++d) {
      const int det = tl.det + d;
      float bp = -1.f;                               // running first maximum over the run's nt tiles (ascending time)
      int bt0 = 0;
      for (int tt = 0; tt < tl.nt; ++tt, ++it) {
        const int buf = it & 1;
        const int tbase = tl.t0 + tt * TILE_N + cs * 32;
        mbar_wait(&tfull[buf], (it >> 1) & 1);
        tc_fence_after_sync();
        const uint32_t t_re = tmem + lane_base + buf * 256 + cs * 32;
        // the slice is loaded as two halves of 16 columns: the second load is in flight while the first half is scanned
        uint32_t vr[32], vi[32];
        tmem_ld_32x16(t_re, *reinterpret_cast<uint32_t(*)[16]>(&vr[0]));
        tmem_ld_32x16(t_re + 128, *reinterpret_cast<uint32_t(*)[16]>(&vi[0]));
        tmem_ld_wait();
        tmem_ld_32x16(t_re + 16, *reinterpret_cast<uint32_t(*)[16]>(&vr[16]));
        tmem_ld_32x16(t_re + 128 + 16, *reinterpret_cast<uint32_t(*)[16]>(&vi[16]));
        // chunk maxima are independent; the running-maximum chain is one compare + select per chunk and the record
        // stores are predicated (no vote / branch on the chain).  Only a buffer's last tile can be ragged: the masked
        // loop is a separate copy, chosen once per tile.
        auto scan = [&](auto ragged_tag, int c_lo, int c_hi) {
          constexpr bool RAGGED = decltype(ragged_tag)::value;
#pragma unroll
          for (int c = 0; c < 32 / PK_CHUNK; ++c) {
            if (c < c_lo || c >= c_hi) continue;
            const int t0c = tbase + c * PK_CHUNK;
            float p[PK_CHUNK];
#pragma unroll
            for (int i = 0; i < PK_CHUNK; i += 2)
              abs2_x2(__uint_as_float(vr[c * PK_CHUNK + i]), __uint_as_float(vr[c * PK_CHUNK + i + 1]),
                      __uint_as_float(vi[c * PK_CHUNK + i]), __uint_as_float(vi[c * PK_CHUNK + i + 1]), p[i], p[i + 1]);
            if (RAGGED) {
#pragma unroll
              for (int i = 0; i < PK_CHUNK; ++i) if (t0c + i >= B || t0c + i < t_min) p[i] = -1.f;
            }
            float cm = p[0];
#pragma unroll
            for (int i = 1; i + 1 < PK_CHUNK; i += 2) cm = fmaxf(cm, fmaxf(p[i], p[i + 1]));
            cm = fmaxf(cm, p[PK_CHUNK - 1]);
            if (cm > bp) {                             // strict: an earlier chunk keeps a tie (first maximum)
              bp = cm; bt0 = t0c;
#pragma unroll
              for (int j = 0; j < PK_CHUNK / 4; ++j) {  // the loaded registers are consecutive: plain 16-byte stores
                const int o = c * PK_CHUNK + 4 * j;
                // explicit st.shared (through the generic pointer the compiler emits generic stores)
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(rec_re_s + j * EPI_THREADS * 16), "r"(vr[o]), "r"(vr[o + 1]), "r"(vr[o + 2]), "r"(vr[o + 3]) : "memory");
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(rec_im_s + j * EPI_THREADS * 16), "r"(vi[o]), "r"(vi[o + 1]), "r"(vi[o + 2]), "r"(vi[o + 3]) : "memory");
              }
            }
          }
        };
        // (t_min > 0: the tail pass of the overlapped trigger windows looks at samples [t_min, B) only)
        const bool masked = tl.t0 + tt * TILE_N + TILE_N > B || t_min > 0;
        constexpr int HALF_CHUNKS = 16 / PK_CHUNK;
        if (masked) scan(std::true_type(), 0, HALF_CHUNKS); else scan(std::false_type(), 0, HALF_CHUNKS);
        tmem_ld_wait();
        tc_fence_before_sync();                        // this warp's part of the accumulators is in registers: release the buffer
        __syncwarp();
        if (lane == 0) mbar_arrive(&tempty[buf]);
        if (masked) scan(std::true_type(), HALF_CHUNKS, 2 * HALF_CHUNKS); else scan(std::false_type(), HALF_CHUNKS, 2 * HALF_CHUNKS);
        if (dbg) {
          float *o = snr_debug + ((size_t)det * 2 * M + 2 * m) * B;
#pragma unroll
          for (int i = 0; i < 32; ++i)
            if (tbase + i < B) { o[tbase + i] = __uint_as_float(vr[i]) * sc; o[B + tbase + i] = __uint_as_float(vi[i]) * sc; }
        }
      }
      if (m < M) {
        PeakPartial best;
        best.p = -1.f; best.idx = 0; best.re = 0.f; best.im = 0.f;
        if (bp >= 0.f) {
          bool found = false;
#pragma unroll
          for (int j = 0; j < PK_CHUNK / 4; ++j) {
            const float4 a = rec_re[j * EPI_THREADS], b = rec_im[j * EPI_THREADS];
            const float re4[4] = {a.x, a.y, a.z, a.w}, im4[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float pp = __fmaf_rn(im4[i], im4[i], __fmul_rn(re4[i], re4[i]));
              if (!found && pp == bp) { found = true; best.idx = bt0 + 4 * j + i; best.re = re4[i] * sc; best.im = im4[i] * sc; }
            }
          }
          best.p = best.re * best.re + best.im * best.im;
        }
        partial[((size_t)det * n_tt + tl.slot * 4 + cs) * Mtot + tmpl_off + m] = best;   // [detector][slot][template]: a warp writes 512 contiguous bytes
      }
      }
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 512);
}

// ------------------------------------------------------------------------------------------------
// a2.  Persistent CTAs (one per SM) over work UNITS = (class, 128 stacked basis rows, tap segment of <= 1024 taps,
// up to 4 sub-tiles), a sub-tile being 128 (or fewer) output columns of one detector.  All sub-tiles of a unit share
// the U tiles (read once from L2 for up to 512 output columns); the tap segments (split K) of a slice balance the
// load and their partial sums go to separate planes of the Y ring, added in order by the reader (deterministic).
// For each chunk of KS = 128 taps warps 2-5 build, per sub-tile, the Hankel strip
//   strip[m][r][e] = x[k + 8 m + r + e]   (fp16; m < (NT + KS)/8, r < 8, e < 8; 128 B per m)
// from the strain window staged in shared memory, so that B[n][k] = x[n + k] is a no-swizzle K-major operand with
// LBO = SBO = 128 B starting at strip + 16*k bytes.  Accumulators: 4 x [128 x 128] fp32 = all 512 TMEM columns.
// ------------------------------------------------------------------------------------------------
static constexpr int KS = 128;                                // taps per strip chunk (2 U stages)
static constexpr int KSEG_MAX = 1024;                         // taps per unit (split-K segment)
static constexpr int MAX_SUB = 4;                             // sub-tiles per unit, packed into 256 accumulator columns
static constexpr int UNIT_N = 256;                            // accumulator columns per unit (x2 TMEM buffers)
static constexpr int SUB_W = 256;                             // widest sub-tile: one MMA of N = 256 (operand reads < math cycles)
static constexpr int STRIP_PLANE = (UNIT_N + MAX_SUB * KS) * 16;   // strips of all sub-tiles of a unit, one plane, one buffer: 12 KB
static constexpr int XWIN_TOTAL = UNIT_N + MAX_SUB * (KSEG_MAX + 8);  // staged strain windows of all sub-tiles (floats)
static constexpr int CORR_THREADS = 448;                      // warps: 0 TMA, 1 MMA, 2-5 + 10-13 epilogue, 6-9 strip builders

struct TcCorrUnit {
  int cls, row0, k0, k1;                                      // taps [k0, k1), multiples of 64
  int seg, nsub;
  int det[MAX_SUB], col0[MAX_SUB];
  int nt[MAX_SUB];                                            // MMA N of the sub-tile: columns rounded up to 16, sum <= UNIT_N
  int tcol[MAX_SUB];                                          // first accumulator column of the sub-tile (prefix sum of nt)
  int soff[MAX_SUB];                                          // byte offset of the sub-tile's strip inside a plane: 16 * (tcol + sb * KS)
  int xoff[MAX_SUB];                                          // float offset of the sub-tile's staged strain window
};

int tc_k_segments(int Npad) { return (Npad + KSEG_MAX - 1) / KSEG_MAX; }

template <int PLANES>
__global__ void __launch_bounds__(CORR_THREADS, 1)
corr_tc_kernel(const CorrClass *__restrict__ classes, const TcCorrClass *__restrict__ maps, const TcCorrUnit *__restrict__ units,
               const int *__restrict__ cta_begin, const long long *__restrict__ n0_ptr) {
  constexpr int STAGES = PLANES == 2 ? 4 : 6;
  constexpr int STAGE_BYTES = PLANES * TILE_BYTES;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t *smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);   // 1024-byte aligned; stays a shared-space pointer
  uint8_t *strips = smem + STAGES * STAGE_BYTES;                 // [2 buffers][PLANES][STRIP_PLANE]
  float *xwin = (float *)(strips + 2 * PLANES * STRIP_PLANE);    // [XWIN_TOTAL]
  uint64_t *bars = (uint64_t *)(xwin + XWIN_TOTAL);
  uint64_t *ufull = bars, *uempty = bars + STAGES, *sfull = bars + 2 * STAGES, *sempty = sfull + 2, *tfull = sempty + 2,
           *tempty = tfull + 2;
  uint32_t *tmem_slot = (uint32_t *)(tempty + 2);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    for (int i = 0; i < STAGES; ++i) { mbar_init(&ufull[i], 1); mbar_init(&uempty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&sfull[i], 4); mbar_init(&sempty[i], 1); mbar_init(&tfull[i], 1); mbar_init(&tempty[i], 8); }
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, 512);
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer: U tiles of 128 rows x 64 taps (x planes), in unit order
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      for (int ui = cta_begin[blockIdx.x]; ui < cta_begin[blockIdx.x + 1]; ++ui) {
        const TcCorrUnit *u = &units[ui];
        const CUtensorMap *mapU = &maps[u->cls].mapU;
        const int Lpad = classes[u->cls].Lpad, row0 = u->row0, k1 = u->k1;
        for (int k = u->k0; k < k1; k += BK) {
          mbar_wait(&uempty[stage], phase ^ 1);
          mbar_arrive_expect_tx(&ufull[stage], STAGE_BYTES);
#pragma unroll
          for (int p = 0; p < PLANES; ++p)
            tma_load_2d(smem + stage * STAGE_BYTES + p * TILE_BYTES, mapU, &ufull[stage], k, p * Lpad + row0);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer.  Descriptors differ only in their 14-bit address field (16-byte units): one 64-bit add each.
    // The whole warp runs the loops (uniform control flow: descriptors stay in uniform registers); one elected lane
    // issues the MMAs of a 64-tap block and the commits.
    int stage = 0; uint32_t phase = 0; int it = 0, chunk_it = 0;
    for (int ui = cta_begin[blockIdx.x]; ui < cta_begin[blockIdx.x + 1]; ++ui, ++it) {
      const TcCorrUnit *u = &units[ui];
      const int nsub = u->nsub, k0 = u->k0, k1 = u->k1;
      uint32_t idesc[MAX_SUB], dcol[MAX_SUB], sdesc[MAX_SUB];
#pragma unroll
      for (int sb = 0; sb < MAX_SUB; ++sb) {
        idesc[sb] = idesc_f16_f32(TILE_M, sb < nsub ? u->nt[sb] : 16);
        dcol[sb] = sb < nsub ? u->tcol[sb] : 0;
        sdesc[sb] = sb < nsub ? (uint32_t)(u->soff[sb] >> 4) : 0;
      }
      const int buf = it & 1;
      mbar_wait(&tempty[buf], ((it >> 1) & 1) ^ 1);
      tc_fence_after_sync();
      const uint32_t d0 = tmem + buf * UNIT_N;
      // the chunk / k loops, specialised on the number of sub-tiles so the issuing lane runs straight-line code
      auto issue = [&](auto ns_tag) {
        constexpr int NS = decltype(ns_tag)::value;
        for (int kc = k0; kc < k1; kc += KS, ++chunk_it) {
          const int sbuf = chunk_it & 1;
          mbar_wait(&sfull[sbuf], (chunk_it >> 1) & 1);
          tc_fence_after_sync();
          const uint64_t xd = desc_kmajor_nosw(smem_u32(strips + sbuf * PLANES * STRIP_PLANE), 128, 128);
          const int kend = min(kc + KS, k1);
          for (int kb = kc; kb < kend; kb += BK) {
            mbar_wait(&ufull[stage], phase);
            tc_fence_after_sync();
            const uint64_t ud = desc_kmajor_sw128(smem_u32(smem + stage * STAGE_BYTES));
            const uint64_t xk = xd + (uint64_t)(kb - kc);              // 16 B per tap
            if (elect_one()) {
#pragma unroll
              for (int k = 0; k < BK / 16; ++k) {
                const bool acc = (kb > k0) || (k > 0);
                const uint64_t u_hi = ud + 2 * k, u_lo = u_hi + (TILE_BYTES >> 4);
#pragma unroll
                for (int sb = 0; sb < NS; ++sb) {
                  const uint64_t x_hi = xk + 16 * k + sdesc[sb], x_8 = x_hi + (STRIP_PLANE >> 4);
                  mma_f16_ss(d0 + dcol[sb], u_hi, x_hi, idesc[sb], acc);
                  // correction planes: 16 taps = 32 bytes of (e4m3, e4m3) x (e5m2, e5m2) pairs: one fp8 MMA adds U_hi x_lo + U_lo x_hi
                  if (PLANES == 2) mma_f8_ss(d0 + dcol[sb], u_lo, x_8, idesc[sb] | (1u << 10), true);
                }
              }
              mma_commit(&uempty[stage]);
              if (kb + BK >= kend) mma_commit(&sempty[sbuf]);
              if (kb + BK >= k1) mma_commit(&tfull[buf]);
            }
            __syncwarp();
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
        }
      };
      if (nsub == 1) issue(std::integral_constant<int, 1>());
      else if (nsub == 2) issue(std::integral_constant<int, 2>());
      else if (nsub == 3) issue(std::integral_constant<int, 3>());
      else issue(std::integral_constant<int, 4>());
    }
  } else if (warp >= 6 && warp < 10) {
    // ===== strip builders (128 threads): stage the strain windows of a unit, then build its strips chunk by chunk
    const int tid = threadIdx.x - 192;
    const long long n0 = *n0_ptr;
    int chunk_it = 0;
    for (int ui = cta_begin[blockIdx.x]; ui < cta_begin[blockIdx.x + 1]; ++ui) {
      const TcCorrUnit *u = &units[ui];
      const CorrClass &c = classes[u->cls];
      const int nsub = u->nsub, k0 = u->k0, klen = u->k1 - k0;
      asm volatile("bar.sync 1, 128;" ::: "memory");             // every builder is done with the previous unit's windows
      for (int sb = 0; sb < nsub; ++sb) {
        // sub-tile sb needs x[first + k0 + i], i in [0, NT + klen): contiguous in the mirrored ring
        const long long first = n0 / c.D + c.H + u->col0[sb] - c.delay - c.N + 1 + c.lag;
        const int p0 = (int)(((first % c.rlen) + c.rlen) % c.rlen);
        const float *x = c.ring2 + (size_t)u->det[sb] * c.ring_det_stride + p0 + k0;
        float *w = xwin + u->xoff[sb];
        const int nw = u->nt[sb] + klen + 8;
        for (int i = tid; i < nw; i += 4 * 128) {
          float v[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) v[j] = (i + j * 128 < nw) ? x[i + j * 128] : 0.f;
#pragma unroll
          for (int j = 0; j < 4; ++j) if (i + j * 128 < nw) w[i + j * 128] = v[j];
        }
      }
      asm volatile("bar.sync 1, 128;" ::: "memory");
      int nt_r[MAX_SUB], soff_r[MAX_SUB], xoff_r[MAX_SUB];        // the unit's sub-tile table in registers
#pragma unroll
      for (int sb = 0; sb < MAX_SUB; ++sb) {
        nt_r[sb] = sb < nsub ? u->nt[sb] : 0; soff_r[sb] = sb < nsub ? u->soff[sb] : 0; xoff_r[sb] = sb < nsub ? u->xoff[sb] : 0;
      }
      for (int kc = 0; kc < klen; kc += KS, ++chunk_it) {
        const int sbuf = chunk_it & 1;
        mbar_wait(&sempty[sbuf], ((chunk_it >> 1) & 1) ^ 1);
#pragma unroll
        for (int sb = 0; sb < MAX_SUB; ++sb) {
          if (sb >= nsub) break;
          const int n_ent = nt_r[sb] + min(KS, klen - kc);         // entry e = 8 m + r holds x[kc + e .. kc + e + 8)
          uint8_t *dst = strips + sbuf * PLANES * STRIP_PLANE + soff_r[sb];
          const float *xs = xwin + xoff_r[sb] + kc;
          for (int e = tid; e < n_ent; e += 128) {
            float v[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) v[i] = xs[e + i];
            __half2 h[4];
            uint32_t l[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              h[i] = __floats2half2_rn(v[2 * i], v[2 * i + 1]);
              if (PLANES == 2) {
                // correction strip: per tap 16 bits = { e5m2(4 x_lo), e5m2(x_hi / 256) }
                const float2 bb = __half22float2(h[i]);
                const uint32_t p0 = __nv_cvt_float2_to_fp8x2(make_float2((v[2 * i] - bb.x) * 4.f, bb.x * (1.f / 256.f)), __NV_SATFINITE, __NV_E5M2);
                const uint32_t p1 = __nv_cvt_float2_to_fp8x2(make_float2((v[2 * i + 1] - bb.y) * 4.f, bb.y * (1.f / 256.f)), __NV_SATFINITE, __NV_E5M2);
                l[i] = p0 | (p1 << 16);
              }
            }
            *reinterpret_cast<uint4 *>(dst + (size_t)e * 16) = *reinterpret_cast<uint4 *>(h);
            if (PLANES == 2) *reinterpret_cast<uint4 *>(dst + STRIP_PLANE + (size_t)e * 16) = *reinterpret_cast<uint4 *>(l);
          }
        }
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(&sfull[sbuf]);
      }
    }
  } else {
    // ===== epilogue (warps 2-5 and 10-13): thread = basis row (TMEM lane); the two warp groups take alternate chunks of
    // 32 columns; partial sums of this tap segment -> plane `seg` of the Y ring (time-major: 128 B per warp store)
    const int q = warp & 3;
    const int grp = warp >= 10 ? 1 : 0;
    const long long n0 = *n0_ptr;
    int it = 0;
    for (int ui = cta_begin[blockIdx.x]; ui < cta_begin[blockIdx.x + 1]; ++ui, ++it) {
      const TcCorrUnit *u = &units[ui];
      const CorrClass &c = classes[u->cls];
      const int nsub = u->nsub, buf = it & 1;
      const int ylen = c.ylen, ncols = c.ncols;
      const size_t Lpad = (size_t)c.Lpad;
      const float sc = c.u_scale_inv;
      const int row = u->row0 + q * 32 + lane;
      const bool row_ok = row < c.Lstack;
      const long long jbase = n0 / c.D + c.H + 64;
      float *ybase = c.yring + (size_t)u->seg * c.yseg_stride + row;
      mbar_wait(&tfull[buf], (it >> 1) & 1);
      tc_fence_after_sync();
      const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + buf * UNIT_N;
      for (int sb = 0; sb < nsub; ++sb) {
        const int col0 = u->col0[sb], NT = u->nt[sb];
        float *yr = ybase + (size_t)u->det[sb] * c.ydet_stride;
        const int slot0 = (int)((jbase + col0) % ylen);
        const int nvalid = min(NT, ncols - col0);                 // columns of this sub-tile that exist
        for (int cc = grp * 32; cc < nvalid; cc += 64) {
          uint32_t v[32];
          tmem_ld_32x32(taddr + u->tcol[sb] + cc, v);
          tmem_ld_wait();
          int slot = slot0 + cc;
          if (slot >= ylen) slot -= ylen;
          float *p = yr + (size_t)slot * Lpad;
          float *const pend = yr + (size_t)ylen * Lpad;
          if (row_ok) {
            if (cc + 32 <= nvalid) {
#pragma unroll
              for (int i = 0; i < 32; ++i) {
                *p = __uint_as_float(v[i]) * sc;
                p += Lpad;
                if (p >= pend) p -= (size_t)ylen * Lpad;
              }
            } else {
#pragma unroll
              for (int i = 0; i < 32; ++i) {
                if (cc + i < nvalid) *p = __uint_as_float(v[i]) * sc;
                p += Lpad;
                if (p >= pend) p -= (size_t)ylen * Lpad;
              }
            }
          }
        }
      }
      tc_fence_before_sync();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tempty[buf]);
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 512);
}

// ------------------------------------------------------------------------------------------------ host side
struct TcPlan {
  int planes, n_det, B, n_tt;
  TcReconBank *rbanks_dev; TcReconTile *rtiles_dev; int n_rtiles;
  // resident-R a3: up to 3 launches, the banks grouped by the size of their R tile, so that small-K banks get the deep operand
  // ring their small resident region leaves room for (one launch sized for Kpad = 144 gave every bank 3 stages)
  TcReconTile *res_items_dev[3]; int *res_begin_dev[3]; int n_res[3], res_grid[3], res_ring_off[3], res_stages[3], n_res_classes;
  int n_res_items, str_stages;
  // the a3 launches of one push are independent (disjoint partial-peak slots): all but the first go to side streams between a
  // fork and a join event, so that the CTAs of the next launch fill the SMs the previous one's tail leaves idle
  cudaStream_t side[3]; cudaEvent_t fork_ev, join_ev[3]; bool side_ready;
  TcReconTile *tail_dev; int *tail_begin_dev; int n_tail, tail_grid, tail_tmin;   // tail pass of overlapped trigger windows
  TcReconTile *xi_dev; int *xi_begin_dev; int n_xi, xi_grid;   // xi^2 pass
  int *rbegin_dev, *cbegin_dev;
  TcCorrClass *cmaps_dev; TcCorrUnit *cunits_dev; int n_cunits, corr_grid;
  int n_phase; std::vector<int> clist_off, clist_n;          // a2 unit lists: one per phase + one with every class
  const CorrClass *classes_dev;
  int recon_grid, recon_smem, corr_smem;
  std::vector<void *> allocs;
};

// Consecutive time tiles one CTA visit covers for a fixed (bank, detector, template tile): as long as possible while
// the persistent grid still gets >= 3 units per SM.  The peak is carried in registers across the run.
static int recon_run_tiles(int B, long long n_mtile_units) {
  const int ntile = (B + TILE_N - 1) / TILE_N;
  int nt = 1;
  while (nt * 2 <= ntile && n_mtile_units * ((ntile + 2 * nt - 1) / (2 * nt)) >= 3 * 148) nt *= 2;
  return nt;
}
int tc_time_splits(int B, long long n_mtile_units) {          // partial peaks per template: 4 column slices per run
  const int ntile = (B + TILE_N - 1) / TILE_N, nt = recon_run_tiles(B, n_mtile_units);
  return 4 * ((ntile + nt - 1) / nt);
}

// Longest-processing-time assignment of work items to `grid` persistent CTAs: items sorted by decreasing cost, each given
// to the least loaded CTA; returns the items regrouped per CTA and the per-CTA begin offsets.
template <typename T, typename CostFn>
static void lpt_assign(std::vector<T> &items, int grid, CostFn cost, std::vector<int> &begin) {
  std::vector<int> order(items.size());
  for (size_t i = 0; i < order.size(); ++i) order[i] = (int)i;
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cost(items[a]) > cost(items[b]); });
  std::vector<long long> load(grid, 0);
  std::vector<std::vector<int>> mine(grid);
  typedef std::pair<long long, int> Q;
  std::priority_queue<Q, std::vector<Q>, std::greater<Q>> heap;
  for (int c = 0; c < grid; ++c) heap.push({0, c});
  for (int i : order) {
    Q q = heap.top(); heap.pop();
    mine[q.second].push_back(i);
    q.first += cost(items[i]);
    heap.push(q);
  }
  std::vector<T> out;
  out.reserve(items.size());
  begin.assign(grid + 1, 0);
  for (int c = 0; c < grid; ++c) {
    begin[c] = (int)out.size();
    for (int i : mine[c]) out.push_back(items[i]);
  }
  begin[grid] = (int)out.size();
  items.swap(out);
}

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

// fp16 row-major [rows][cols], box = box_cols (64 / 32 / 16) columns x box_rows rows, swizzle = the box's row width (128 / 64 / 32 B)
static bool make_map(CUtensorMap *m, const void *base, uint64_t rows, uint64_t cols, int box_rows, int box_cols) {
  EncodeTiledFn enc = get_encode();
  if (!enc) { set_error("stream_create: cuTensorMapEncodeTiled is not available from the driver"); return false; }
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols * 2};
  cuuint32_t box[2] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows};
  const CUtensorMapSwizzle sw = box_cols == 16 ? CU_TENSOR_MAP_SWIZZLE_32B : (box_cols == 32 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B);
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("stream_create: cuTensorMapEncodeTiled failed (%d) for [%llu][%llu]", (int)r,
                                     (unsigned long long)rows, (unsigned long long)cols); return false; }
  return true;
}

// upsampled-Y planes: rows of `cols` elements (fp16: bytes = false, correction plane: bytes = true), boxes of 128 B x box_rows, 128-byte swizzle
static bool make_map_y(CUtensorMap *m, const void *base, bool bytes, uint64_t rows, uint64_t cols, int box_rows) {
  EncodeTiledFn enc = get_encode();
  if (!enc) { set_error("stream_create: cuTensorMapEncodeTiled is not available from the driver"); return false; }
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {cols * (bytes ? 1 : 2)};
  cuuint32_t box[2] = {(cuuint32_t)(bytes ? 128 : 64), (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(m, bytes ? CU_TENSOR_MAP_DATA_TYPE_UINT8 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void *>(base), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("stream_create: cuTensorMapEncodeTiled failed (%d) for the upsampled-Y plane [%llu][%llu]", (int)r,
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
  if (p->side_ready) {
    cudaEventDestroy(p->fork_ev);
    for (int i = 0; i < 3; ++i) { cudaStreamSynchronize(p->side[i]); cudaEventDestroy(p->join_ev[i]); cudaStreamDestroy(p->side[i]); }
  }
  for (void *q : p->allocs) cudaFree(q);
  delete p;
}

int tc_plan_create(TcPlan **out, const std::vector<CorrClass> &classes, const CorrClass *classes_dev,
                   const std::vector<ReconBank> &banks, const ReconBank *, int n_det, int B, int planes, int overlap, int xi_delta, int n_phase) {
  *out = nullptr;
  TcPlan *p = new TcPlan();
  p->planes = planes; p->n_det = n_det; p->B = B; p->classes_dev = classes_dev;
  {
    bool ok = cudaEventCreateWithFlags(&p->fork_ev, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < 3 && ok; ++i)
      ok = cudaStreamCreateWithFlags(&p->side[i], cudaStreamNonBlocking) == cudaSuccess &&
           cudaEventCreateWithFlags(&p->join_ev[i], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { set_error("stream_create: cannot create the side streams / events of a3"); delete p; return LLOID_ECUDA; }
    p->side_ready = true;
  }
  // ---- a2: one tensor map per class; units = (row tile, tap segment, group of <= 4 (detector, column tile) sub-tiles),
  //      dealt to the persistent CTAs in order of decreasing cost
  std::vector<TcCorrClass> cm(classes.size());
  std::vector<TcCorrUnit> cu;
  for (size_t ci = 0; ci < classes.size(); ++ci) {
    const CorrClass &c = classes[ci];
    memset(&cm[ci], 0, sizeof(TcCorrClass));
    if (!make_map(&cm[ci].mapU, c.U16, (uint64_t)planes * c.Lpad, (uint64_t)c.Npad, TILE_M, BK)) { tc_plan_destroy(p); return LLOID_ECUDA; }
    const int nseg = tc_k_segments(c.Npad);
    const int kseg = ((c.Npad + nseg - 1) / nseg + BK - 1) / BK * BK;
    struct Sub { int det, c0, w; };
    std::vector<Sub> subs;
    for (int det = 0; det < n_det; ++det)
      for (int c0 = 0; c0 < c.ncols;) {                      // wide sub-tiles (<= 256 columns) while more than 128 remain
        const int w = (c.ncols - c0 > TILE_N) ? std::min(SUB_W, c.ncols - c0) : c.ncols - c0;
        subs.push_back({det, c0, w});
        c0 += w;
      }
    for (int r0 = 0; r0 < c.Lstack; r0 += TILE_M)
      for (int sg = 0; sg < nseg; ++sg) {
        const int k0 = sg * kseg, k1 = std::min(c.Npad, k0 + kseg);
        if (k0 >= k1) continue;
        for (size_t s0 = 0; s0 < subs.size();) {
          TcCorrUnit u; memset(&u, 0, sizeof(u));
          u.cls = (int)ci; u.row0 = r0; u.k0 = k0; u.k1 = k1; u.seg = sg;
          // pack up to MAX_SUB sub-tiles into the unit's UNIT_N accumulator columns (they share every U tile)
          int cols = 0, xo = 0;
          while (s0 < subs.size() && u.nsub < MAX_SUB) {
            const int nt = (subs[s0].w + 15) & ~15;
            if (cols + nt > UNIT_N) break;
            const int i = u.nsub++;
            u.det[i] = subs[s0].det; u.col0[i] = subs[s0].c0; u.nt[i] = nt;
            u.tcol[i] = cols; u.soff[i] = 16 * (cols + i * KS); u.xoff[i] = xo;
            cols += nt; xo += nt + (k1 - k0) + 8;
            ++s0;
          }
          cu.push_back(u);
        }
      }
  }
  p->n_cunits = (int)cu.size();
  p->n_phase = std::max(1, n_phase);
  // ---- a3: two tensor maps per bank.  Banks whose R tile fits the resident region (split mode, Kpad <= RES_KMAX) become
  //      items (bank, template tile, detector group, run of time tiles) of the resident-R kernel; the others are tiled
  //      (bank, template tile, detector, run of time tiles) for the streaming kernel
  std::vector<TcReconBank> rb(banks.size());
  std::vector<TcReconTile> rt, ri;
  std::vector<char> is_res(banks.size(), 0);
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  long long n_mu = 0, n_bm = 0;
  for (size_t b = 0; b < banks.size(); ++b) {
    const ReconBank &k = banks[b];
    memset(&rb[b], 0, sizeof(TcReconBank));
    const uint64_t Bp = (uint64_t)yup_pitch(B), yrows = (uint64_t)n_det * k.Kpad;
    const uint8_t *y8 = reinterpret_cast<const uint8_t *>(k.yup) + 2 * k.yup_plane_stride;      // the correction plane (bytes)
    if (!make_map(&rb[b].mapR, k.R16, (uint64_t)planes * 2 * k.Mpad, (uint64_t)k.Kpad, TILE_M, 16) ||
        !make_map(&rb[b].mapR64, k.R16, (uint64_t)planes * 2 * k.Mpad, (uint64_t)k.Kpad, TILE_M, RBK_STR) ||
        !make_map_y(&rb[b].mapY, k.yup, false, yrows, Bp, RBK_RES) || !make_map_y(&rb[b].mapY64, k.yup, false, yrows, Bp, RBK_STR)) {
      tc_plan_destroy(p); return LLOID_ECUDA;
    }
    if (planes == 2 && (!make_map_y(&rb[b].mapY8, y8, true, 2 * yrows, Bp, 2 * RBK_RES) || !make_map_y(&rb[b].mapY8_64, y8, true, 2 * yrows, Bp, 2 * RBK_STR))) {
      tc_plan_destroy(p); return LLOID_ECUDA;
    }
    rb[b].M = k.M; rb[b].Mpad = k.Mpad; rb[b].Kpad = k.Kpad; rb[b].tmpl_off = k.tmpl_off; rb[b].inv_scale = k.inv_scale;
    rb[b].acorr = k.acorr; rb[b].xi_delta = k.xi_delta;
    if (xi_delta > 0) {                                        // history ring: rows of 3 B samples, plane stride n_det * Kpad * 3 B
      const uint8_t *h8 = reinterpret_cast<const uint8_t *>(k.yhist) + 2 * yrows * 3 * (uint64_t)B;
      if (!make_map_y(&rb[b].mapYh, k.yhist, false, yrows, 3 * (uint64_t)B, RBK_STR) ||
          !make_map_y(&rb[b].mapYh8, h8, true, 2 * yrows, 3 * (uint64_t)B, 2 * RBK_STR)) { tc_plan_destroy(p); return LLOID_ECUDA; }
    }
    // resident R pays when the item reuses it over enough tiles (short buffers, config 4, stream R with Y instead)
    is_res[b] = (planes == 2 && k.Kpad <= RES_KMAX && (long long)n_det * ((B + TILE_N - 1) / TILE_N) >= 8) ? 1 : 0;
    const long long mt = (k.M + TILE_M - 1) / TILE_M;
    if (is_res[b]) n_bm += mt;
    else n_mu += mt * n_det;
  }
  const int nt = recon_run_tiles(B, n_mu), ntile = (B + TILE_N - 1) / TILE_N;
  p->n_tt = n_mu ? tc_time_splits(B, n_mu) : 4;
  // resident items: split by detector, then into runs of time tiles, until the persistent grid has a few items per SM
  const int det_split = (n_bm < 4LL * sms && n_det > 1) ? n_det : 1;
  int r_time = 1;
  while (n_bm * det_split * r_time < 2LL * sms && ntile / (r_time * 2) >= 2) r_time *= 2;
  const int nt_run = (ntile + r_time - 1) / r_time, n_runs = (ntile + nt_run - 1) / nt_run;
  if (n_bm) p->n_tt = std::max(p->n_tt, 4 * n_runs);
  for (size_t b = 0; b < banks.size(); ++b) {
    const ReconBank &k = banks[b];
    for (int m0 = 0; m0 < k.M; m0 += TILE_M) {
      if (is_res[b]) {
        const int nd = n_det / det_split;
        for (int dg = 0; dg < det_split; ++dg)
          for (int r = 0; r < n_runs; ++r)
            ri.push_back({(int)b, dg * nd, nd, m0, r * nt_run * TILE_N, std::min(nt_run, ntile - r * nt_run), r});
      } else {
        for (int det = 0; det < n_det; ++det)
          for (int i0 = 0; i0 < ntile; i0 += nt) rt.push_back({(int)b, det, 1, m0, i0 * TILE_N, std::min(nt, ntile - i0), i0 / nt});
      }
    }
  }
  // tail pass (trigger windows overlapped by `overlap` samples): one streaming item per (bank, template
  // tile, detector) over the tiles that hold the buffer's last `overlap` samples; its epilogue masks samples < B - overlap
  std::vector<TcReconTile> tail;
  p->tail_tmin = std::max(0, B - overlap);
  if (overlap > 0) {
    const int i0 = p->tail_tmin / TILE_N;
    for (size_t b = 0; b < banks.size(); ++b)
      for (int m0 = 0; m0 < banks[b].M; m0 += TILE_M)
        for (int det = 0; det < n_det; ++det) tail.push_back({(int)b, det, 1, m0, i0 * TILE_N, ntile - i0, 0});
  }
  // xi^2 pass: per (bank, template tile, detector) the 128-aligned tiles covering [-delta, B + delta) of the target buffer
  std::vector<TcReconTile> xit;
  if (xi_delta > 0) {
    const int t_first = -((xi_delta + TILE_N - 1) / TILE_N) * TILE_N, nt_xi = (B + xi_delta - t_first + TILE_N - 1) / TILE_N;
    for (size_t b = 0; b < banks.size(); ++b)
      for (int m0 = 0; m0 < banks[b].M; m0 += TILE_M)
        for (int det = 0; det < n_det; ++det) xit.push_back({(int)b, det, 1, m0, t_first, nt_xi, 0});
  }
  p->n_xi = (int)xit.size();
  p->xi_grid = std::max(1, std::min(p->n_xi, sms));
  p->n_tail = (int)tail.size();
  p->tail_grid = std::max(1, std::min(p->n_tail, sms));
  p->n_res_items = (int)ri.size();
  // classes by K blocks of the R tile: <= 2 (<= 64 KB resident, 8 stages), 3 (<= 96 KB, 7-8 stages), more (<= 144 KB, 4 stages);
  // a class too small to fill the persistent grid joins its neighbour
  std::vector<TcReconTile> rcls[3];
  int rk[3] = {0, 0, 0};
  for (const TcReconTile &t : ri) {
    const int nkb = (rb[t.bank].Kpad + RBK_RES - 1) / RBK_RES, c = nkb <= 2 ? 0 : (nkb == 3 ? 1 : 2);
    rcls[c].push_back(t); rk[c] = std::max(rk[c], rb[t.bank].Kpad);
  }
  for (int c = 0; c < 3; ++c) {
    if (rcls[c].empty() || (long long)rcls[c].size() >= 4LL * sms) continue;
    int d = -1;
    for (int j = c + 1; j < 3 && d < 0; ++j) if (!rcls[j].empty()) d = j;
    for (int j = c - 1; j >= 0 && d < 0; --j) if (!rcls[j].empty()) d = j;
    if (d < 0) continue;                                         // the only class
    rcls[d].insert(rcls[d].end(), rcls[c].begin(), rcls[c].end()); rk[d] = std::max(rk[d], rk[c]);
    rcls[c].clear(); rk[c] = 0;
  }
  p->n_res_classes = 0;
  std::vector<int> ibegin[3];
  for (int c = 0; c < 3; ++c) {
    if (rcls[c].empty()) continue;
    const int i = p->n_res_classes++;
    p->n_res[i] = (int)rcls[c].size();
    p->res_grid[i] = std::max(1, std::min(p->n_res[i], sms));
    p->res_ring_off[i] = (rk[c] / 16) * RSTEP_BYTES;
    p->res_stages[i] = std::min(RMAX_STAGES, (RECON_SMEM_BUDGET - REC_BYTES - p->res_ring_off[i]) / (2 * TILE_M * RBK_RES * 2));
    // cost in cycles: 4 MMAs of ~97 cycles per 16 of K per tile (at least the epilogue's ~600), plus the once-per-item R load
    lpt_assign(rcls[c], p->res_grid[i], [&](const TcReconTile &t) {
      const long long kp = rb[t.bank].Kpad;
      return (long long)t.ndet * t.nt * std::max<long long>(kp / 16 * 388, 600) + 3000 + kp * 8; }, ibegin[i]);
    if (!plan_upload(p, &p->res_items_dev[i], rcls[c]) || !plan_upload(p, &p->res_begin_dev[i], ibegin[i])) { tc_plan_destroy(p); return LLOID_ENOMEM; }
  }
  p->str_stages = std::min(RMAX_STAGES, (RECON_SMEM_BUDGET - REC_BYTES) / (3 * planes * TILE_M * RBK_STR * 2));
  p->n_rtiles = (int)rt.size();
  p->recon_grid = std::max(1, std::min(p->n_rtiles, sms));
  p->corr_grid = std::max(1, std::min(p->n_cunits, sms));
  std::vector<int> cbegin, rbegin;
  {
    // batch-ahead (a slice delayed by more than a second may be filtered ahead of need): list f holds the
    // units of the classes correlated every push plus those whose phase is f; the last list holds every class (first push)
    std::vector<TcCorrUnit> all;
    for (int li = 0; li <= p->n_phase; ++li) {
      std::vector<TcCorrUnit> lu;
      for (const TcCorrUnit &u : cu) { const int ph = classes[u.cls].phase; if (li == p->n_phase || ph < 0 || ph == li) lu.push_back(u); }
      std::vector<int> lb;
      lpt_assign(lu, p->corr_grid, [](const TcCorrUnit &u) { return (long long)(u.nt[0] + u.nt[1] + u.nt[2] + u.nt[3]) * (u.k1 - u.k0) / 128 + 128; }, lb);
      p->clist_off.push_back((int)all.size()); p->clist_n.push_back((int)lu.size());
      all.insert(all.end(), lu.begin(), lu.end());
      cbegin.insert(cbegin.end(), lb.begin(), lb.end());
    }
    cu.swap(all);
  }
  lpt_assign(rt, p->recon_grid, [&](const TcReconTile &t) { return (long long)t.nt * (rb[t.bank].Kpad / 16 + 2); }, rbegin);
  std::vector<int> tbegin, xbegin;
  lpt_assign(xit, p->xi_grid, [&](const TcReconTile &t) { return (long long)t.nt * (rb[t.bank].Kpad / 16 + 2); }, xbegin);
  lpt_assign(tail, p->tail_grid, [&](const TcReconTile &t) { return (long long)t.nt * (rb[t.bank].Kpad / 16 + 2); }, tbegin);
  if (!plan_upload(p, &p->cbegin_dev, cbegin) || !plan_upload(p, &p->rbegin_dev, rbegin) ||
      !plan_upload(p, &p->tail_dev, tail) || !plan_upload(p, &p->tail_begin_dev, tbegin) ||
      !plan_upload(p, &p->xi_dev, xit) || !plan_upload(p, &p->xi_begin_dev, xbegin)) { tc_plan_destroy(p); return LLOID_ENOMEM; }
  if (!plan_upload(p, &p->cmaps_dev, cm) || !plan_upload(p, &p->cunits_dev, cu) || !plan_upload(p, &p->rbanks_dev, rb) ||
      !plan_upload(p, &p->rtiles_dev, rt)) { tc_plan_destroy(p); return LLOID_ENOMEM; }
  p->recon_smem = RECON_SMEM_BUDGET + 1024 + 256;
  p->corr_smem = (planes == 2 ? 4 : 6) * planes * TILE_BYTES + 2 * planes * STRIP_PLANE + XWIN_TOTAL * 4 + 1024 + 256;
  cudaError_t e;
  if (planes == 2) {
    e = cudaFuncSetAttribute(recon_tc_kernel<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->recon_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(recon_tc_kernel<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->recon_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(recon_tc_kernel<2, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->recon_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(corr_tc_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->corr_smem);
  } else {
    e = cudaFuncSetAttribute(recon_tc_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->recon_smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(corr_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, p->corr_smem);
  }
  if (e != cudaSuccess) { set_error("stream_create: cudaFuncSetAttribute: %s", cudaGetErrorString(e)); tc_plan_destroy(p); return LLOID_ECUDA; }
  *out = p;
  return LLOID_OK;
}

cudaError_t tc_launch_corr(TcPlan *p, const long long *n0, cudaStream_t st, int list) {
  if (p->clist_n[list] == 0) return cudaSuccess;
  const TcCorrUnit *units = p->cunits_dev + p->clist_off[list];
  const int *begin = p->cbegin_dev + (size_t)list * (p->corr_grid + 1);
  if (p->planes == 2)
    corr_tc_kernel<2><<<p->corr_grid, CORR_THREADS, p->corr_smem, st>>>(p->classes_dev, p->cmaps_dev, units, begin, n0);
  else
    corr_tc_kernel<1><<<p->corr_grid, CORR_THREADS, p->corr_smem, st>>>(p->classes_dev, p->cmaps_dev, units, begin, n0);
  return cudaGetLastError();
}

int tc_plan_n_tt(const TcPlan *p) { return p->n_tt; }
int tc_plan_recon_launches(const TcPlan *p) { return (p->n_rtiles ? 1 : 0) + p->n_res_classes + (p->n_tail ? 1 : 0); }

cudaError_t tc_launch_xi2(TcPlan *p, const lloid_peak *peaks, float *xi_partial, int Mtot, int row_base, cudaStream_t st) {
  if (p->n_xi == 0 || p->planes != 2) return cudaErrorInvalidValue;
  XiArgs xa; xa.peaks = peaks; xa.partial = xi_partial; xa.row_base = row_base; xa.ring_rows = 3 * p->B;
  recon_tc_kernel<2, false, true><<<p->xi_grid, RECON_THREADS, p->recon_smem, st>>>(p->rbanks_dev, p->xi_dev, p->xi_begin_dev, p->n_det, p->B,
                                                                                  nullptr, Mtot, 4, nullptr, -1, 0, p->str_stages, 0, xa);
  return cudaGetLastError();
}

// tail pass: the peak of every template over the buffer's last `overlap` samples -> tail_partial [n_det][4][Mtot]
cudaError_t tc_launch_recon_tail(TcPlan *p, PeakPartial *tail_partial, int Mtot, cudaStream_t st) {
  if (p->n_tail == 0) return cudaSuccess;
  if (p->planes == 2)
    recon_tc_kernel<2, false><<<p->tail_grid, RECON_THREADS, p->recon_smem, st>>>(p->rbanks_dev, p->tail_dev, p->tail_begin_dev, p->n_det, p->B,
                                                                               tail_partial, Mtot, 4, nullptr, -1, 0, p->str_stages, p->tail_tmin);
  else
    recon_tc_kernel<1, false><<<p->tail_grid, RECON_THREADS, p->recon_smem, st>>>(p->rbanks_dev, p->tail_dev, p->tail_begin_dev, p->n_det, p->B,
                                                                               tail_partial, Mtot, 4, nullptr, -1, 0, p->str_stages, p->tail_tmin);
  return cudaGetLastError();
}

cudaError_t tc_launch_recon(TcPlan *p, PeakPartial *partial, int Mtot, float *snr_debug, int debug_bank, cudaStream_t st) {
  // launch k = 0 on the caller's stream, k >= 1 on side stream k - 1 (after the fork event); the caller's stream then waits for all
  const int n_launch = p->n_res_classes + (p->n_rtiles ? 1 : 0);
  cudaError_t e = cudaSuccess;
  if (n_launch > 1) e = cudaEventRecord(p->fork_ev, st);
  int k = 0;
  auto stream_of = [&](int i) -> cudaStream_t {
    if (i == 0) return st;
    cudaStreamWaitEvent(p->side[i - 1], p->fork_ev, 0);
    return p->side[i - 1];
  };
  for (int i = 0; i < p->n_res_classes && e == cudaSuccess; ++i, ++k) {
    recon_tc_kernel<2, true><<<p->res_grid[i], RECON_THREADS, p->recon_smem, stream_of(k)>>>(p->rbanks_dev, p->res_items_dev[i], p->res_begin_dev[i], p->n_det, p->B,
                                                                                         partial, Mtot, p->n_tt, snr_debug, debug_bank, p->res_ring_off[i], p->res_stages[i], 0);
    e = cudaGetLastError();
  }
  if (p->n_rtiles && e == cudaSuccess) {
    cudaStream_t s2 = stream_of(k++);
    if (p->planes == 2)
      recon_tc_kernel<2, false><<<p->recon_grid, RECON_THREADS, p->recon_smem, s2>>>(p->rbanks_dev, p->rtiles_dev, p->rbegin_dev, p->n_det, p->B,
                                                                                  partial, Mtot, p->n_tt, snr_debug, debug_bank, 0, p->str_stages, 0);
    else
      recon_tc_kernel<1, false><<<p->recon_grid, RECON_THREADS, p->recon_smem, s2>>>(p->rbanks_dev, p->rtiles_dev, p->rbegin_dev, p->n_det, p->B,
                                                                                  partial, Mtot, p->n_tt, snr_debug, debug_bank, 0, p->str_stages, 0);
    e = cudaGetLastError();
  }
  for (int i = 1; i < k; ++i) {                                   // join (also after a failed launch: nothing may be left dangling)
    cudaError_t e2 = cudaEventRecord(p->join_ev[i - 1], p->side[i - 1]);
    if (e2 == cudaSuccess) e2 = cudaStreamWaitEvent(st, p->join_ev[i - 1], 0);
    if (e == cudaSuccess) e = e2;
  }
  return e;
}

}  // namespace lloid
