// a1 decimator (Eq. 4), the basis-domain polyphase upsampler (Eqs. 7-9)
// and the peak finalisation.  FP32 CUDA-core kernels shared by every precision mode:
// they are latency/HBM-bound stages, not contractions.
#include "lloid_internal.h"

namespace lloid {

// ------------------------------------------------------------------------------------------------
// K1: append the pushed strain to the f0 ring and decimate it to every lower rate.
//   d_r[j] = sum_k taps[k] * d[j*D + c - k], taps = sqrt(D)*ghat (host, float64 -> fp32), zero phase.
//   New outputs of a push: j in [n0/D - n_down, (n0+B)/D - n_down)  (needs c future f0 samples).
//   One warp per output; lane t sums taps t, t+32, ... in a fixed order, then a shuffle tree: deterministic.
// ------------------------------------------------------------------------------------------------
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
  const int warp = ((blockIdx.x - P.copy_blocks) * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (warp >= P.total_out) return;
  int ri = 1;
  while (ri + 1 < P.n_rates && warp >= P.r[ri + 1].out_begin) ++ri;
  const RateDev &r = P.r[ri];
  const long long j = n0 / r.D - r.lag + (warp - r.out_begin);
  const long long top = j * r.D + r.c;            // f0 index read by tap k = 0
  float acc = 0.f;
  const int ntap = 2 * r.c + 1;
  for (int k = lane; k < ntap; k += 32) {
    long long i = top - k;
    float v;
    if (i >= n0) v = sd[i - n0];
    else if (i < 0) v = 0.f;
    else v = ring0[(int)(i % r0.rlen)];
    acc = fmaf(r.taps[k], v, acc);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) {
    int slot = (int)((j + r.lag) % r.rlen);
    float *ring = r.ring2 + (size_t)det * 2 * r.rlen;
    ring[slot] = acc;
    ring[slot + r.rlen] = acc;
  }
}

cudaError_t launch_decimate(const DecimParams &P, const float *strain, const long long *n0, cudaStream_t st) {
  int dec_blocks = (P.total_out + 7) / 8;
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
//   CTA = (time chunk of `chunk` f0 samples, item = 32 basis rows of one slice, detector).  lane = basis row.
// ------------------------------------------------------------------------------------------------
#define UP_MAXW 168   // widest staged level: chunk/2 + 2*8 + ... <= 256/2 + 33
template <int HALF_PLANES>
__global__ void __launch_bounds__(256) upsample_kernel(const UpItem *__restrict__ items, int B, int chunk,
                                                       const float *__restrict__ uptaps,
                                                       const int *__restrict__ uptap_off,
                                                       const long long *__restrict__ n0_ptr) {
  __shared__ float buf[2][UP_MAXW][32];
  const UpItem it = items[blockIdx.y];
  const int det = blockIdx.z;
  const long long n0 = *n0_ptr;
  const int ka = blockIdx.x * chunk;
  const int kb = min(ka + chunk, B);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const bool active = lane < it.nl;

  long long lo[LLOID_MAX_GROUPS + 1], hi[LLOID_MAX_GROUPS + 1];
  lo[0] = n0 + ka;
  hi[0] = n0 + kb;
  for (int h = 1; h <= it.g; ++h) {
    lo[h] = (lo[h - 1] >> it.log2f[h]) - LLOID_NUP;          // arithmetic shift = floor division
    hi[h] = ((hi[h - 1] - 1) >> it.log2f[h]) + LLOID_NUP + 1;
  }
  const float *yr = it.yring + (size_t)det * it.ydet_stride + it.row0 + lane;
  const size_t out_row0 = (size_t)det * it.yup_det_stride + (size_t)it.kcol + lane;

  auto store_out = [&](int k, float v) {   // k: sample within the buffer
    size_t o = out_row0 + (size_t)k * it.kpitch;
    if (HALF_PLANES == 0) {
      reinterpret_cast<float *>(it.yup)[o] = v;
    } else {
      __half hi16 = __float2half_rn(v);
      reinterpret_cast<__half *>(it.yup)[o] = hi16;
      if (HALF_PLANES == 2)
        reinterpret_cast<__half *>(it.yup)[o + it.yup_plane_stride] = __float2half_rn(v - __half2float(hi16));
    }
  };

  // level g from the Y ring (columns never computed at stream start are the ring's zeros)
  const int wg = (int)(hi[it.g] - lo[it.g]);
  if (it.g == 0) {
    for (int c = warp; c < wg; c += nwarp) {
      long long j = lo[0] + c;
      int slot = (int)((j + 64) % it.ylen);
      if (active) store_out(ka + c, yr[(size_t)slot * it.ypitch]);
    }
    return;
  }
  for (int c = warp; c < wg; c += nwarp) {
    long long j = lo[it.g] + c;
    int slot = (int)((j + 64) % it.ylen);
    buf[0][c][lane] = active ? yr[(size_t)slot * it.ypitch] : 0.f;
  }
  __syncthreads();
  int cur = 0;
  for (int h = it.g; h >= 1; --h) {
    const int lf = it.log2f[h], f = 1 << lf;
    const float *g = uptaps + uptap_off[lf];
    const int wout = (int)(hi[h - 1] - lo[h - 1]);
    for (int c = warp; c < wout; c += nwarp) {
      long long i = lo[h - 1] + c;
      long long q = i >> lf;
      int ph = (int)(i & (f - 1));
      int base = (int)(q - lo[h]);           // index of in[q]
      float v;
      if (ph == 0) {
        v = buf[cur][base][lane];
      } else {
        v = 0.f;
#pragma unroll
        for (int k = 0; k < 2 * LLOID_NUP; ++k) v = fmaf(buf[cur][base + LLOID_NUP - k][lane], g[k * f + ph], v);
      }
      if (h == 1) { if (active) store_out(ka + c, v); }
      else buf[cur ^ 1][c][lane] = v;
    }
    __syncthreads();
    cur ^= 1;
  }
}

cudaError_t launch_upsample(const UpItem *items_dev, int n_items, int n_det, int B, int chunk, const float *uptaps,
                            const int *uptap_off, const long long *n0, int out_half_planes, cudaStream_t st) {
  dim3 grid((B + chunk - 1) / chunk, n_items, n_det);
  if (out_half_planes == 0) upsample_kernel<0><<<grid, 256, 0, st>>>(items_dev, B, chunk, uptaps, uptap_off, n0);
  else if (out_half_planes == 1) upsample_kernel<1><<<grid, 256, 0, st>>>(items_dev, B, chunk, uptaps, uptap_off, n0);
  else upsample_kernel<2><<<grid, 256, 0, st>>>(items_dev, B, chunk, uptaps, uptap_off, n0);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a5 finalisation: reduce the per-time-tile partial peaks of every template in ascending time order
// (strict '>' keeps the first maximum), then snr = sqrt(p), phase = atan2(im, re).
// The last thread also advances the device-side stream clock n0 by B.
// ------------------------------------------------------------------------------------------------
__global__ void finalize_kernel(const PeakPartial *__restrict__ partial, int n_det, int Mtot, int n_tt,
                                float threshold, lloid_peak *__restrict__ peaks, long long *n0, int B) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t == 0) *n0 += B;
  if (t >= n_det * Mtot) return;
  const PeakPartial *pp = partial + (size_t)t * n_tt;
  PeakPartial best = pp[0];
  for (int i = 1; i < n_tt; ++i) {
    PeakPartial c = pp[i];
    if (c.p > best.p) best = c;
  }
  lloid_peak o;
  o.snr = sqrtf(best.p);
  o.sample = best.idx;
  o.phase = atan2f(best.im, best.re);
  if (threshold > 0.f && o.snr < threshold) { o.snr = 0.f; o.sample = -1; o.phase = 0.f; }
  peaks[t] = o;
}

cudaError_t launch_finalize(const PeakPartial *partial, int n_det, int Mtot, int n_tt, float threshold,
                            lloid_peak *peaks, long long *n0, int B, cudaStream_t st) {
  int n = n_det * Mtot;
  finalize_kernel<<<(n + 255) / 256, 256, 0, st>>>(partial, n_det, Mtot, n_tt, threshold, peaks, n0, B);
  return cudaGetLastError();
}

}  // namespace lloid
