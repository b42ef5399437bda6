// Event identification on the per-template triggers of one push (Sec. II.D.3-4):
// coincidence formation across detectors and clustering to one event per bank.  Small reductions over the peaks
// array (12 B per template and detector); one CTA per bank.
#include "lloid_internal.h"

namespace lloid {

struct CoincParams {
  int n_det;
  int dt[LLOID_MAX_DET][LLOID_MAX_DET];   // coincidence window of every detector pair, f0 samples, inclusive
};

// One CTA per bank.  Thread t looks at templates t, t + 256, ... of the bank: a trigger exists where the peak was
// reported (sample != LLOID_NO_TRIGGER).  Among the detector sets with >= 2 members whose triggers are pairwise within
// dt, the template's event is the one with the largest sum of snr^2 (ascending bit-mask order breaks ties); the
// bank's event is the template with the largest such sum (lowest template index breaks ties).
__global__ void __launch_bounds__(256) coinc_cluster_kernel(const lloid_peak *__restrict__ peaks, int Mtot,
                                                            const int *__restrict__ bank_off, CoincParams P,
                                                            lloid_event *__restrict__ events) {
  const int b = blockIdx.x, lo = bank_off[b], hi = bank_off[b + 1];
  double best_v = 0.0;
  int best_j = 0x7fffffff, best_mask = 0;
  for (int j = lo + threadIdx.x; j < hi; j += blockDim.x) {
    float snr[LLOID_MAX_DET];
    int smp[LLOID_MAX_DET];
    int have = 0;
#pragma unroll
    for (int a = 0; a < LLOID_MAX_DET; ++a) {
      snr[a] = 0.f; smp[a] = 0;
      if (a < P.n_det) {
        const lloid_peak pk = peaks[(size_t)a * Mtot + j];
        if (pk.sample != LLOID_NO_TRIGGER) { have |= 1 << a; snr[a] = pk.snr; smp[a] = pk.sample; }
      }
    }
    int pair_ok = 0;                                  // bit (a * 4 + c): triggers of a and c exist and are within dt
#pragma unroll
    for (int a = 0; a < LLOID_MAX_DET; ++a)
#pragma unroll
      for (int c = a + 1; c < LLOID_MAX_DET; ++c)
        if (((have >> a) & 1) && ((have >> c) & 1) && abs(smp[a] - smp[c]) <= P.dt[a][c]) pair_ok |= 1 << (a * 4 + c);
    double tv = 0.0;
    int tmask = 0;
    for (int m = 3; m < (1 << P.n_det); ++m) {
      if (__popc(m) < 2 || (m & have) != m) continue;
      bool ok = true;
      double v = 0.0;
#pragma unroll
      for (int a = 0; a < LLOID_MAX_DET; ++a) {
        if (!((m >> a) & 1)) continue;
        v += (double)snr[a] * (double)snr[a];
#pragma unroll
        for (int c = a + 1; c < LLOID_MAX_DET; ++c)
          if (((m >> c) & 1) && !((pair_ok >> (a * 4 + c)) & 1)) ok = false;
      }
      if (ok && v > tv) { tv = v; tmask = m; }
    }
    if (tmask != 0 && (tv > best_v || (tv == best_v && j < best_j))) { best_v = tv; best_j = j; best_mask = tmask; }
  }
  __shared__ double sv[256];
  __shared__ int sj[256], sm[256];
  sv[threadIdx.x] = best_v; sj[threadIdx.x] = best_j; sm[threadIdx.x] = best_mask;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) {
      const double v = sv[threadIdx.x + o];
      const int j = sj[threadIdx.x + o];
      if (sm[threadIdx.x + o] != 0 && (sm[threadIdx.x] == 0 || v > sv[threadIdx.x] || (v == sv[threadIdx.x] && j < sj[threadIdx.x]))) {
        sv[threadIdx.x] = v; sj[threadIdx.x] = j; sm[threadIdx.x] = sm[threadIdx.x + o];
      }
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    lloid_event e;
    e.template_index = sm[0] ? sj[0] : -1;
    e.det_mask = sm[0];
    e.net_snr = sm[0] ? (float)sqrt(sv[0]) : 0.f;
    e.reserved = 0;
    for (int a = 0; a < LLOID_MAX_DET; ++a) {
      e.snr[a] = 0.f; e.sample[a] = LLOID_NO_TRIGGER; e.phase[a] = 0.f;
      if ((sm[0] >> a) & 1) {
        const lloid_peak pk = peaks[(size_t)a * Mtot + sj[0]];
        e.snr[a] = pk.snr; e.sample[a] = pk.sample; e.phase[a] = pk.phase;
      }
    }
    events[b] = e;
  }
}

cudaError_t launch_coinc_cluster(const lloid_peak *peaks, int n_det, int Mtot, const int *bank_off_dev, int n_banks,
                                 const int32_t *dt_host, lloid_event *events, cudaStream_t st) {
  CoincParams P;
  P.n_det = n_det;
  for (int a = 0; a < LLOID_MAX_DET; ++a)
    for (int c = 0; c < LLOID_MAX_DET; ++c) P.dt[a][c] = (a < n_det && c < n_det) ? dt_host[a * n_det + c] : -1;
  coinc_cluster_kernel<<<n_banks, 256, 0, st>>>(peaks, Mtot, bank_off_dev, P, events);
  return cudaGetLastError();
}

}  // namespace lloid

// ------------------------------------------------------------------------------------------------
// Signal-based consistency test, Eq. 10, for the triggers of one bank whose SNR series is
// materialised (the snr_debug output of lloid_stream_push, consecutive buffers side by side):
//   xi2_j = sum_{t=-delta}^{delta} |z_j[k0 + t] - z_j[k0] R_j[t]|^2 / sum_t (2 - 2 |R_j[t]|^2)
// One warp per template; lane l takes t = -delta + l, -delta + l + 32, ...; fixed-order shuffle reduction
// (deterministic).  Samples outside [0, n) count as zero (stream start / the caller did not wait for the padding).
// ------------------------------------------------------------------------------------------------
namespace lloid {

__global__ void __launch_bounds__(256) xi2_series_kernel(const float *__restrict__ snr, int M, long long n,
                                                         const int *__restrict__ k0v, const float2 *__restrict__ acorr, int delta,
                                                         float *__restrict__ out) {
  const int j = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
  if (j >= M) return;
  const int k0 = k0v[j];
  if (k0 == LLOID_NO_TRIGGER || k0 < 0 || k0 >= n) { if (lane == 0) out[j] = -1.f; return; }
  const float *re = snr + (size_t)(2 * j) * n, *im = re + n;
  const float2 *R = acorr + (size_t)j * (2 * delta + 1);
  const float z0r = re[k0], z0i = im[k0];
  float num = 0.f, den = 0.f;
  for (int u = lane; u <= 2 * delta; u += 32) {
    const long long k = (long long)k0 - delta + u;
    const float2 a = R[u];
    float zr = 0.f, zi = 0.f;
    if (k >= 0 && k < n) { zr = re[k]; zi = im[k]; }
    const float dr = zr - (z0r * a.x - z0i * a.y), di = zi - (z0r * a.y + z0i * a.x);
    num += dr * dr + di * di;
    den += 2.f - 2.f * (a.x * a.x + a.y * a.y);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { num += __shfl_xor_sync(0xffffffffu, num, o); den += __shfl_xor_sync(0xffffffffu, den, o); }
  if (lane == 0) out[j] = num / den;
}

}  // namespace lloid

extern "C" int lloid_xi2_series(const float *snr, int32_t n_templates, int64_t n_samples, const int32_t *trigger_sample,
                                const float *acorr, int32_t delta, float *xi2_out, void *cuda_stream) {
  using namespace lloid;
  if (!snr || !trigger_sample || !acorr || !xi2_out || n_templates < 1 || n_samples < 1 || delta < 1) {
    set_error("xi2_series: NULL pointer or non-positive size"); return LLOID_EINVAL;
  }
  const long long threads = (long long)n_templates * 32;
  xi2_series_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(
      snr, n_templates, n_samples, trigger_sample, reinterpret_cast<const float2 *>(acorr), delta, xi2_out);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_error("xi2_series: launch failed: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  return LLOID_OK;
}
