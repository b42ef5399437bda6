// PSD estimation + whitening front end (Sec. II.B.2, lines 63-81, Figs. 2-3): the step immediately before the
// LLOID path.  Per push of hop = N/2 - Z input samples per detector:
//   window + zero pad -> R2C FFT (length N) -> running median / geometric-mean PSD, whitening, frequency-domain
//   downsampling -> C2R FFT (length N_out) -> Tukey window, overlap-add, emit hop_out samples.
// The two FFTs are plain library transforms (cuFFT, loaded at run time so that liblloid.so itself does not depend on
// it); everything else is the three small kernels below.  Latency: N/2 input samples.
#include <cufft.h>
#include <dlfcn.h>

#include <cmath>
#include <vector>

#include "lloid_internal.h"

namespace lloid {

static const double kEulerGamma = 0.57721566490153286;

// ---- cuFFT through dlopen
struct CufftApi {
  void *lib = nullptr;
  cufftResult (*PlanMany)(cufftHandle *, int, int *, int *, int, int, int *, int, int, cufftType, int) = nullptr;
  cufftResult (*SetStream)(cufftHandle, cudaStream_t) = nullptr;
  cufftResult (*ExecR2C)(cufftHandle, cufftReal *, cufftComplex *) = nullptr;
  cufftResult (*ExecC2R)(cufftHandle, cufftComplex *, cufftReal *) = nullptr;
  cufftResult (*Destroy)(cufftHandle) = nullptr;
};
static CufftApi *cufft_api() {
  static CufftApi api;
  static bool tried = false;
  if (!tried) {
    tried = true;
    const char *names[] = {"libcufft.so.11", "/usr/local/cuda/lib64/libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so"};
    for (const char *n : names) { api.lib = dlopen(n, RTLD_NOW | RTLD_LOCAL); if (api.lib) break; }
    if (api.lib) {
      api.PlanMany = (decltype(api.PlanMany))dlsym(api.lib, "cufftPlanMany");
      api.SetStream = (decltype(api.SetStream))dlsym(api.lib, "cufftSetStream");
      api.ExecR2C = (decltype(api.ExecR2C))dlsym(api.lib, "cufftExecR2C");
      api.ExecC2R = (decltype(api.ExecC2R))dlsym(api.lib, "cufftExecC2R");
      api.Destroy = (decltype(api.Destroy))dlsym(api.lib, "cufftDestroy");
      if (!api.PlanMany || !api.SetStream || !api.ExecR2C || !api.ExecC2R || !api.Destroy) { dlclose(api.lib); api.lib = nullptr; }
    }
  }
  return api.lib ? &api : nullptr;
}

// c(m) = E log(median of m iid unit-mean exponential variates), m odd: trapezoid rule in u = log x over
// u f(e^u) e^u, f = density of the k-th order statistic, k = (m + 1) / 2 (c(1) = -gamma).
static double log_median_mean(int m) {
  const int k = (m + 1) / 2;
  double cst = 1.0;
  for (int i = 2; i <= m; ++i) cst *= i;
  for (int i = 2; i <= k - 1; ++i) cst /= i;
  for (int i = 2; i <= m - k; ++i) cst /= i;
  const double h = 1e-4;
  double s = 0.0;
  for (double u = -60.0; u <= 6.0; u += h) {
    const double x = std::exp(u);
    s += u * cst * std::pow(-std::expm1(-x), k - 1) * std::exp(-x * (m - k + 1)) * x;
  }
  return s * h;
}

// ---- kernels
// K1: slide the input segment by hop and build the windowed, zero-padded FFT block.
__global__ void whiten_window_kernel(const float *__restrict__ x, const float *__restrict__ seg_old, float *__restrict__ seg_new,
                                     const float *__restrict__ hann, float *__restrict__ block, int N, int Z, int hop) {
  const int det = blockIdx.y, L = N - 2 * Z;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
    float v = 0.f;
    if (i >= Z && i < N - Z) {
      const int j = i - Z;
      const float s = (j < L - hop) ? seg_old[(size_t)det * L + j + hop] : x[(size_t)det * hop + j - (L - hop)];
      seg_new[(size_t)det * L + j] = s;
      v = s * hann[j];
    }
    block[(size_t)det * N + i] = v;
  }
}

// K2: per kept frequency bin: instantaneous PSD into the history ring, median of the last m (odd), running mean of its
// log, PSD, whitened + band-limited spectrum.
__global__ void whiten_psd_kernel(const float2 *__restrict__ X, int xpitch, float *__restrict__ hist, float *__restrict__ logG,
                                  float2 *__restrict__ W, float *__restrict__ psd_out, int nb, int n_med, int slot, int m, int n_avg_eff,
                                  int first, float p_scale, float log_corr, float w_scale) {
  const int det = blockIdx.y;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nb) return;
  const float2 xv = X[(size_t)det * xpitch + k];
  const float P = p_scale * (xv.x * xv.x + xv.y * xv.y);
  float *h = hist + ((size_t)det * n_med) * nb + k;
  h[(size_t)slot * nb] = P;
  float v[7];
#pragma unroll
  for (int i = 0; i < 7; ++i) {
    int s = slot - i;
    if (s < 0) s += n_med;
    v[i] = (i < m) ? ((i == 0) ? P : h[(size_t)s * nb]) : 3.0e38f;
  }
#pragma unroll
  for (int i = 0; i < 6; ++i)                        // compare-exchange network on 7 registers (ascending)
#pragma unroll
    for (int j = 0; j < 6 - i; ++j) { const float a = fminf(v[j], v[j + 1]), b = fmaxf(v[j], v[j + 1]); v[j] = a; v[j + 1] = b; }
  float med = v[0];
#pragma unroll
  for (int i = 1; i < 7; ++i) if (i == m / 2) med = v[i];
  const float lg = logf(med) - log_corr;             // log of the single-block geometric-mean estimate
  const size_t gi = (size_t)det * nb + k;
  const float G = first ? lg : ((float)(n_avg_eff - 1) * logG[gi] + lg) / (float)n_avg_eff;
  logG[gi] = G;
  const float S = expf(G + (float)0.57721566490153286);
  if (psd_out) psd_out[gi] = S;
  float2 w = make_float2(0.f, 0.f);
  if (k > 0 && k < nb - 1 && S > 0.f) { const float a = w_scale * rsqrtf(S); w.x = xv.x * a; w.y = xv.y * a; }
  W[gi] = w;
}

// K3: Tukey window, overlap-add, emit the finished hop_out samples and slide the accumulator.
__global__ void whiten_ola_kernel(const float *__restrict__ w, const float *__restrict__ tukey, const float *__restrict__ acc_old,
                                  float *__restrict__ acc_new, float *__restrict__ out, int N_out, int hop_out, float scale) {
  const int det = blockIdx.y;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N_out; i += gridDim.x * blockDim.x) {
    const float v = acc_old[(size_t)det * N_out + i] + w[(size_t)det * N_out + i] * tukey[i] * scale;
    if (i < hop_out) { out[(size_t)det * hop_out + i] = v; acc_new[(size_t)det * N_out + N_out - hop_out + i] = 0.f; }
    else acc_new[(size_t)det * N_out + i - hop_out] = v;
  }
}

}  // namespace lloid

using namespace lloid;

struct lloid_whitener {
  int n_det, f_in, f_out, N, Z, L, hop, N_out, Z_out, hop_out, nb, n_med, n_avg;
  long long count;
  float p_scale, w_scale;
  cudaStream_t st;
  cufftHandle plan_fwd, plan_inv;
  bool have_fwd, have_inv;
  float *hann, *tukey, *seg[2], *block, *acc[2], *hist, *logG, *wt;
  float2 *X, *W;
  double c_m[8];
  std::vector<void *> allocs;
};

extern "C" void lloid_whitener_destroy(lloid_whitener *w) {
  if (!w) return;
  CufftApi *api = cufft_api();
  if (api && w->have_fwd) api->Destroy(w->plan_fwd);
  if (api && w->have_inv) api->Destroy(w->plan_inv);
  for (void *p : w->allocs) cudaFree(p);
  delete w;
}

template <typename T>
static bool wh_alloc(lloid_whitener *w, T **p, size_t n) {
  void *q = nullptr;
  if (cudaMalloc(&q, std::max<size_t>(n * sizeof(T), 16)) != cudaSuccess) return false;
  cudaMemset(q, 0, std::max<size_t>(n * sizeof(T), 16));
  w->allocs.push_back(q);
  *p = (T *)q;
  return true;
}

extern "C" int lloid_whitener_create(lloid_whitener **out, int32_t n_det, int32_t rate_in, int32_t rate_out, int32_t fft_len,
                                     int32_t zero_pad, int32_t n_median, int32_t n_average, void *cuda_stream) {
  if (!out) { set_error("whitener_create: out is NULL"); return LLOID_EINVAL; }
  *out = nullptr;
  if (n_det < 1 || rate_in < 1 || rate_out < 1 || rate_in % rate_out != 0 || fft_len < 8 || zero_pad < 0 || fft_len % 2 != 0 ||
      (fft_len - 2 * zero_pad) < 2 || (fft_len - 2 * zero_pad) % 2 != 0 || ((long long)fft_len * rate_out) % rate_in != 0 ||
      ((long long)zero_pad * rate_out) % rate_in != 0 || n_median < 1 || n_median > 7 || n_median % 2 != 1 || n_average < 1) {
    set_error("whitener_create: need rate_out | rate_in, even fft_len and fft_len - 2 zero_pad, lengths that stay integer at rate_out, "
              "odd n_median <= 7, n_average >= 1");
    return LLOID_EINVAL;
  }
  CufftApi *api = cufft_api();
  if (!api) { set_error("whitener_create: libcufft.so.11 could not be loaded (dlopen)"); return LLOID_ECUDA; }
  lloid_whitener *w = new lloid_whitener();
  w->n_det = n_det; w->f_in = rate_in; w->f_out = rate_out; w->N = fft_len; w->Z = zero_pad; w->L = fft_len - 2 * zero_pad;
  w->hop = fft_len / 2 - zero_pad;
  w->N_out = (int)((long long)fft_len * rate_out / rate_in); w->Z_out = (int)((long long)zero_pad * rate_out / rate_in);
  w->hop_out = w->N_out / 2 - w->Z_out; w->nb = w->N_out / 2 + 1; w->n_med = n_median; w->n_avg = n_average;
  w->count = 0; w->st = (cudaStream_t)cuda_stream; w->have_fwd = w->have_inv = false;
  for (int m = 1; m <= 7; m += 2) w->c_m[m] = log_median_mean(m);
  bool ok = wh_alloc(w, &w->hann, w->L) && wh_alloc(w, &w->tukey, w->N_out) && wh_alloc(w, &w->seg[0], (size_t)n_det * w->L) &&
            wh_alloc(w, &w->seg[1], (size_t)n_det * w->L) && wh_alloc(w, &w->block, (size_t)n_det * w->N) &&
            wh_alloc(w, &w->acc[0], (size_t)n_det * w->N_out) && wh_alloc(w, &w->acc[1], (size_t)n_det * w->N_out) &&
            wh_alloc(w, &w->hist, (size_t)n_det * n_median * w->nb) && wh_alloc(w, &w->logG, (size_t)n_det * w->nb) &&
            wh_alloc(w, &w->wt, (size_t)n_det * w->N_out) && wh_alloc(w, &w->X, (size_t)n_det * (w->N / 2 + 1)) &&
            wh_alloc(w, &w->W, (size_t)n_det * w->nb);
  if (!ok) { set_error("whitener_create: cudaMalloc failed"); lloid_whitener_destroy(w); return LLOID_ENOMEM; }
  std::vector<float> hann(w->L), tuk(w->N_out, 1.f);
  double hsum = 0;
  for (int i = 0; i < w->L; ++i) { const double h = 0.5 - 0.5 * std::cos(2.0 * M_PI * i / w->L); hann[i] = (float)h; hsum += h * h; }
  w->p_scale = (float)(2.0 / ((double)rate_in * hsum));                                     // one-sided PSD per Hz
  w->w_scale = (float)(std::sqrt(2.0 / (double)rate_in) * std::sqrt((double)rate_in / (double)rate_out));
  for (int i = 0; i < w->Z_out; ++i) {
    const float r = (float)(0.5 * (1.0 - std::cos(M_PI * (i + 0.5) / w->Z_out)));
    tuk[i] = r; tuk[w->N_out - 1 - i] = r;
  }
  cudaMemcpy(w->hann, hann.data(), hann.size() * 4, cudaMemcpyHostToDevice);
  cudaMemcpy(w->tukey, tuk.data(), tuk.size() * 4, cudaMemcpyHostToDevice);
  int n1 = w->N, n2 = w->N_out;
  if (api->PlanMany(&w->plan_fwd, 1, &n1, nullptr, 1, w->N, nullptr, 1, w->N / 2 + 1, CUFFT_R2C, n_det) != CUFFT_SUCCESS) {
    set_error("whitener_create: cufftPlanMany (R2C, %d) failed", n1); lloid_whitener_destroy(w); return LLOID_ECUDA;
  }
  w->have_fwd = true;
  if (api->PlanMany(&w->plan_inv, 1, &n2, nullptr, 1, w->nb, nullptr, 1, w->N_out, CUFFT_C2R, n_det) != CUFFT_SUCCESS) {
    set_error("whitener_create: cufftPlanMany (C2R, %d) failed", n2); lloid_whitener_destroy(w); return LLOID_ECUDA;
  }
  w->have_inv = true;
  api->SetStream(w->plan_fwd, w->st);
  api->SetStream(w->plan_inv, w->st);
  if (cudaDeviceSynchronize() != cudaSuccess) { set_error("whitener_create: CUDA error"); lloid_whitener_destroy(w); return LLOID_ECUDA; }
  *out = w;
  return LLOID_OK;
}

extern "C" int32_t lloid_whitener_hop_in(const lloid_whitener *w) { return w ? w->hop : -1; }
extern "C" int32_t lloid_whitener_hop_out(const lloid_whitener *w) { return w ? w->hop_out : -1; }
extern "C" int32_t lloid_whitener_psd_bins(const lloid_whitener *w) { return w ? w->nb : -1; }

extern "C" int lloid_whitener_push(lloid_whitener *w, const float *strain_in, float *white_out, float *psd_out) {
  if (!w || !strain_in || !white_out) { set_error("whitener_push: NULL argument"); return LLOID_EINVAL; }
  CufftApi *api = cufft_api();
  const int cur = (int)(w->count & 1), nxt = cur ^ 1;
  dim3 g1((w->N + 255) / 256 > 128 ? 128 : (w->N + 255) / 256, w->n_det);
  whiten_window_kernel<<<g1, 256, 0, w->st>>>(strain_in, w->seg[cur], w->seg[nxt], w->hann, w->block, w->N, w->Z, w->hop);
  if (api->ExecR2C(w->plan_fwd, w->block, (cufftComplex *)w->X) != CUFFT_SUCCESS) { set_error("whitener_push: cufftExecR2C failed"); return LLOID_ECUDA; }
  const long long cnt = w->count + 1;
  int m = (int)std::min<long long>(cnt, w->n_med);
  m -= 1 - m % 2;
  dim3 g2((w->nb + 255) / 256, w->n_det);
  whiten_psd_kernel<<<g2, 256, 0, w->st>>>(w->X, w->N / 2 + 1, w->hist, w->logG, w->W, psd_out, w->nb, w->n_med, (int)(w->count % w->n_med), m,
                                         (int)std::min<long long>(cnt, w->n_avg), w->count == 0 ? 1 : 0, w->p_scale,
                                         (float)(w->c_m[m] + kEulerGamma), w->w_scale);
  if (api->ExecC2R(w->plan_inv, (cufftComplex *)w->W, w->wt) != CUFFT_SUCCESS) { set_error("whitener_push: cufftExecC2R failed"); return LLOID_ECUDA; }
  dim3 g3((w->N_out + 255) / 256 > 128 ? 128 : (w->N_out + 255) / 256, w->n_det);
  whiten_ola_kernel<<<g3, 256, 0, w->st>>>(w->wt, w->tukey, w->acc[cur], w->acc[nxt], white_out, w->N_out, w->hop_out, 1.f / (float)w->N);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_error("whitener_push: launch failed: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  w->count = cnt;
  return LLOID_OK;
}

extern "C" int lloid_whitener_reset(lloid_whitener *w) {
  if (!w) { set_error("whitener_reset: NULL"); return LLOID_EINVAL; }
  cudaMemsetAsync(w->seg[0], 0, (size_t)w->n_det * w->L * 4, w->st); cudaMemsetAsync(w->seg[1], 0, (size_t)w->n_det * w->L * 4, w->st);
  cudaMemsetAsync(w->acc[0], 0, (size_t)w->n_det * w->N_out * 4, w->st); cudaMemsetAsync(w->acc[1], 0, (size_t)w->n_det * w->N_out * 4, w->st);
  w->count = 0;
  return LLOID_OK;
}
