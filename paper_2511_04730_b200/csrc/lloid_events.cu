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
