// LLOID_PREC_FP32_FFMA contractions: a2 basis correlation (Eq. 5, with the slice delay of
// Eq. 9) and a3 reconstruction (Eq. 6) fused with the peak search
// (PAPER.md:199-201), both as shared-memory tiled fp32 FFMA kernels.  This is the 1e-4-gate path of
// BASELINE.json's north_star and the on-device cross-check of the tcgen05 kernels (kernels_tc.cu).
#include "lloid_internal.h"

namespace lloid {

// ------------------------------------------------------------------------------------------------
// a2: Y[j][l] = sum_{n<N} U[l][n] * x[j - delay - N + 1 + n] for the ncols new columns of a push,
// j in [n0/D + H, (n0+B)/D + H).  Tile: 64 basis rows x 64 columns, 256 threads, 4x4 per thread.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) corr_ffma_kernel(const CorrClass *__restrict__ classes,
                                                        const CorrTile *__restrict__ tiles,
                                                        const long long *__restrict__ n0_ptr) {
  constexpr int TK = 32;
  __shared__ float Us[TK][64 + 4];
  __shared__ float xs[64 + TK];
  const CorrTile tl = tiles[blockIdx.x];
  const CorrClass &c = classes[tl.cls];
  const int det = blockIdx.y;
  const long long n0 = *n0_ptr;
  const long long j0 = n0 / c.D + c.H + tl.col0;                 // first column of this tile
  // x[j0 - delay - N + 1 + i], i >= 0, is contiguous in the mirrored ring starting at slot p0
  long long first = j0 - c.delay - c.N + 1 + c.lag;
  int p0 = (int)(((first % c.rlen) + c.rlen) % c.rlen);
  const float *x = c.ring2 + (size_t)det * c.ring_det_stride + p0;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = 0.f;

  for (int k0 = 0; k0 < c.N; k0 += TK) {
    for (int i = threadIdx.x; i < 64 * TK; i += 256) {
      int r = i / TK, k = i % TK;
      int row = tl.row0 + r, n = k0 + k;
      Us[k][r] = (row < c.Lstack && n < c.N) ? c.U32[(size_t)row * c.Npad + n] : 0.f;
    }
    for (int i = threadIdx.x; i < 64 + TK; i += 256) xs[i] = x[k0 + i];   // window stays inside 2*rlen
    __syncthreads();
#pragma unroll 8
    for (int k = 0; k < TK; ++k) {
      float u[4], v[4];
#pragma unroll
      for (int a = 0; a < 4; ++a) u[a] = Us[k][ty * 4 + a];
#pragma unroll
      for (int b = 0; b < 4; ++b) v[b] = xs[k + tx * 4 + b];
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = fmaf(u[a], v[b], acc[a][b]);
    }
    __syncthreads();
  }
  float *yr = c.yring + (size_t)det * c.ydet_stride;
#pragma unroll
  for (int b = 0; b < 4; ++b) {
    int col = tl.col0 + tx * 4 + b;
    if (col >= c.ncols) continue;
    long long j = j0 + tx * 4 + b;
    int slot = (int)((j + 64) % c.ylen);
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      int row = tl.row0 + ty * 4 + a;
      if (row < c.Lstack) yr[(size_t)slot * c.Lpad + row] = acc[a][b];
    }
  }
}

cudaError_t launch_corr_ffma(const CorrClass *cls_dev, const CorrTile *tiles_dev, int n_tiles, int n_det,
                             const long long *n0, cudaStream_t st) {
  dim3 grid(n_tiles, n_det);
  corr_ffma_kernel<<<grid, 256, 0, st>>>(cls_dev, tiles_dev, n0);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a3 + a5: rho_re[m][k] = sum_K Rre[m][K] Yup[k][K], same for im, over the bank's concatenated basis axis
// (all slices, already at f0), then p = re^2 + im^2 and the first maximum over the tile's 64 samples.
// Tile: 64 templates x 64 samples; thread = 4 templates x 4 samples x (re, im).
// grid = (time tiles, template tiles (max over banks), bank*n_det + det).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) recon_ffma_kernel(const ReconBank *__restrict__ banks, int n_det, int B,
                                                         PeakPartial *__restrict__ partial, int Mtot,
                                                         float *__restrict__ snr_debug, int debug_bank) {
  constexpr int TK = 16;
  __shared__ float Ar[TK][64 + 4], Ai[TK][64 + 4], Ys[TK][64 + 4];
  __shared__ PeakPartial red[64][16];
  const int bank = blockIdx.z / n_det, det = blockIdx.z % n_det;
  const ReconBank &bk = banks[bank];
  const int m0 = blockIdx.y * 64, k0 = blockIdx.x * 64;
  if (m0 >= bk.M) return;
  const float *Rre = bk.R32, *Rim = bk.R32 + bk.r_part_stride;
  const float *Y = reinterpret_cast<const float *>(bk.yup) + (size_t)det * bk.yup_det_stride;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float are[4][4], aim[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) are[a][b] = aim[a][b] = 0.f;

  for (int kk = 0; kk < bk.Kpad; kk += TK) {
    for (int i = threadIdx.x; i < 64 * TK; i += 256) {
      int r = i / TK, k = i % TK;
      size_t o = (size_t)(m0 + r) * bk.Kpad + kk + k;          // rows < Mpad are allocated (zero padded)
      Ar[k][r] = Rre[o];
      Ai[k][r] = Rim[o];
      int t = k0 + r;
      Ys[k][r] = (t < B) ? Y[(size_t)t * bk.Kpad + kk + k] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < TK; ++k) {
      float ur[4], ui[4], v[4];
#pragma unroll
      for (int a = 0; a < 4; ++a) { ur[a] = Ar[k][ty * 4 + a]; ui[a] = Ai[k][ty * 4 + a]; }
#pragma unroll
      for (int b = 0; b < 4; ++b) v[b] = Ys[k][tx * 4 + b];
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          are[a][b] = fmaf(ur[a], v[b], are[a][b]);
          aim[a][b] = fmaf(ui[a], v[b], aim[a][b]);
        }
    }
    __syncthreads();
  }
  // optional full-SNR dump (parity tests only)
  if (snr_debug != nullptr && bank == debug_bank) {
    float *out = snr_debug + (size_t)det * 2 * bk.M * B;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      int m = m0 + ty * 4 + a;
      if (m >= bk.M) continue;
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        int t = k0 + tx * 4 + b;
        if (t >= B) continue;
        out[(size_t)(2 * m) * B + t] = are[a][b];
        out[(size_t)(2 * m + 1) * B + t] = aim[a][b];
      }
    }
  }
  // peak over the tile: per thread ascending in time with strict '>', then across the 16 time-threads
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    PeakPartial best;
    best.p = -1.f; best.idx = 0; best.re = 0.f; best.im = 0.f;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      int t = k0 + tx * 4 + b;
      float p = are[a][b] * are[a][b] + aim[a][b] * aim[a][b];
      if (t < B && p > best.p) { best.p = p; best.idx = t; best.re = are[a][b]; best.im = aim[a][b]; }
    }
    red[ty * 4 + a][tx] = best;
  }
  __syncthreads();
  if (threadIdx.x < 64) {
    int m = m0 + threadIdx.x;
    if (m < bk.M) {
      PeakPartial best = red[threadIdx.x][0];
      for (int i = 1; i < 16; ++i) {
        PeakPartial c = red[threadIdx.x][i];
        if (c.p > best.p) best = c;
      }
      const int n_tt = gridDim.x;
      partial[((size_t)det * n_tt + blockIdx.x) * Mtot + bk.tmpl_off + m] = best;   // [detector][slot][template]
    }
  }
}

cudaError_t launch_recon_ffma(const ReconBank *banks_dev, int n_banks, int max_mtiles, int n_det, int B,
                              PeakPartial *partial, int Mtot, float *snr_debug, int debug_bank, cudaStream_t st) {
  dim3 grid((B + 63) / 64, max_mtiles, n_banks * n_det);
  recon_ffma_kernel<<<grid, 256, 0, st>>>(banks_dev, n_det, B, partial, Mtot, snr_debug, debug_bank);
  return cudaGetLastError();
}

}  // namespace lloid
