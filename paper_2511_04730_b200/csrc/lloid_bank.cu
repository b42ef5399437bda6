// lloid_bank_create / destroy: validation of the slice table, the halo recursion of the upsample chain
// (PAPER.md:146-185), and conversion of the reconstruction matrices R^s = V diag(sigma) (Eq. 6,
// PAPER.md:140-144) into the device operand of the fused reconstruction kernel.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include <cuda_fp8.h>

#include "lloid_internal.h"

namespace lloid {
static thread_local char g_err[512] = "";
void set_error(const char *fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
static bool is_pow2(long long v) { return v > 0 && (v & (v - 1)) == 0; }
static long long floor_div(long long a, long long b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }
}  // namespace lloid

using namespace lloid;

extern "C" const char *lloid_last_error(void) { return g_err; }
extern "C" const char *lloid_version(void) { return "lloid-b200 0.1 (sm_100a)"; }

extern "C" void lloid_options_default(lloid_options *opt) {
  if (!opt) return;
  opt->n_down = 32;
  opt->n_up = LLOID_NUP;
  opt->precision = LLOID_PREC_F16_SPLIT;
  opt->threshold = 0.f;
  opt->trigger_overlap = 0;
}

extern "C" void lloid_bank_destroy(lloid_bank *b) {
  if (!b) return;
  if (b->dR32) cudaFree(b->dR32);
  if (b->dR16) cudaFree(b->dR16);
  if (b->dAcorr) cudaFree(b->dAcorr);
  if (b->dXiDen) cudaFree(b->dXiDen);
  delete b;
}

extern "C" int lloid_bank_create(lloid_bank **out, int32_t f0, int32_t M, int32_t S, const lloid_slice *sl,
                                 const lloid_options *opt_in) {
  if (!out) { set_error("bank_create: out is NULL"); return LLOID_EINVAL; }
  *out = nullptr;
  if (!sl || S < 1 || M < 1) { set_error("bank_create: need slices, n_slices >= 1, n_templates >= 1"); return LLOID_EINVAL; }
  if (!is_pow2(f0)) { set_error("bank_create: strain_rate_hz %d is not a power of two", f0); return LLOID_EINVAL; }
  lloid_options opt;
  lloid_options_default(&opt);
  if (opt_in) opt = *opt_in;
  if (opt.n_up != LLOID_NUP) { set_error("bank_create: only n_up = %d is supported", LLOID_NUP); return LLOID_EINVAL; }
  if (opt.trigger_overlap < 0 || (opt.trigger_overlap > 0 && opt.precision == LLOID_PREC_FP32_FFMA)) {
    set_error("bank_create: trigger_overlap must be >= 0 and needs a tensor-core precision"); return LLOID_EINVAL;
  }
  if (opt.n_down < 1 || opt.n_down > 64) { set_error("bank_create: n_down %d outside [1, 64]", opt.n_down); return LLOID_EINVAL; }
  if (opt.precision < LLOID_PREC_FP32_FFMA || opt.precision > LLOID_PREC_F16_SPLIT) {
    set_error("bank_create: unknown precision %d", opt.precision); return LLOID_EINVAL;
  }
  // ---- slice table (contiguous time slices with shared boundaries)
  for (int s = 0; s < S; ++s) {
    const lloid_slice &x = sl[s];
    if (x.rate_hz < 1 || x.rate_hz > f0 || f0 % x.rate_hz != 0 || !is_pow2(f0 / x.rate_hz)) {
      set_error("bank_create: slice %d rate %d is not f0 / 2^k", s, x.rate_hz); return LLOID_EINVAL;
    }
    if (x.n_taps < 1 || x.n_basis < 1 || !x.basis || !x.recon) {
      set_error("bank_create: slice %d needs n_taps, n_basis >= 1 and non-null arrays", s); return LLOID_EINVAL;
    }
    if (s == 0) {
      if (x.rate_hz != f0) { set_error("bank_create: slice 0 must run at the strain rate"); return LLOID_EINVAL; }
      if (x.delay != 0) { set_error("bank_create: delay[0] must be 0"); return LLOID_EINVAL; }
    } else {
      const lloid_slice &p = sl[s - 1];
      if (x.rate_hz > p.rate_hz) { set_error("bank_create: rates increase at slice %d", s); return LLOID_EINVAL; }
      long long end_prev = (p.delay + p.n_taps) * (long long)(f0 / p.rate_hz);
      long long beg = x.delay * (long long)(f0 / x.rate_hz);
      if (x.delay < 0 || end_prev != beg) {
        set_error("bank_create: slice %d does not abut slice %d (%lld vs %lld f0 samples)", s, s - 1, beg, end_prev);
        return LLOID_EINVAL;
      }
    }
  }
  lloid_bank *b = new (std::nothrow) lloid_bank();
  if (!b) { set_error("bank_create: out of host memory"); return LLOID_ENOMEM; }
  b->f0 = f0; b->M = M; b->Mpad = (M + 127) / 128 * 128; b->S = S; b->opt = opt;
  b->dR32 = nullptr; b->dR16 = nullptr; b->r_scale = 1.f; b->r_planes = 0;
  b->dAcorr = nullptr; b->dXiDen = nullptr; b->xi_delta = 0;
  // ---- groups = runs of equal rate; halo recursion of the zero-phase chain (oracle: upsample_input_range)
  int koff = 0;
  for (int s = 0; s < S; ++s) {
    SliceInfo si;
    si.rate = sl[s].rate_hz; si.D = f0 / si.rate; si.N = sl[s].n_taps; si.L = sl[s].n_basis;
    si.delay = sl[s].delay; si.koff = koff; koff += si.L;
    if (b->groups.empty() || b->groups.back().rate != si.rate) {
      GroupInfo g;
      g.rate = si.rate; g.D = si.D; g.first_slice = s; g.n_slices = 0;
      if (b->groups.empty()) { g.f = 1; g.A = 0; g.H = 0; }
      else {
        const GroupInfo &p = b->groups.back();
        g.f = g.D / p.D;
        if (g.f > (1 << LLOID_MAX_GROUPS)) {              // the upsampler's tap table covers stage factors up to 2^LLOID_MAX_GROUPS
          set_error("bank_create: slice %d: upsample stage factor %d exceeds %d", s, g.f, 1 << LLOID_MAX_GROUPS);
          delete b; return LLOID_EINVAL;
        }
        g.A = (p.A + g.f - 1) / g.f + LLOID_NUP;
        g.H = (int)floor_div(p.H - 1, g.f) + LLOID_NUP + 1;
      }
      b->groups.push_back(g);
    }
    b->groups.back().n_slices++;
    si.group = (int)b->groups.size() - 1;
    b->slices.push_back(std::move(si));
  }
  b->G = (int)b->groups.size();
  b->Ktot = koff; b->Kpad = (koff + 15) / 16 * 16;            // MMA K granularity; TMA zero-fills the rest of a 64-wide box
  if (b->G > LLOID_MAX_GROUPS) { set_error("bank_create: more than %d distinct rates", LLOID_MAX_GROUPS); delete b; return LLOID_EINVAL; }
  // ---- causality: the newest column a push needs, (n0+B)/D + H - 1, must only read
  //      decimated samples that exist, i.e. index <= (n0+B)/D - n_down - 1.
  for (int s = 0; s < S; ++s) {
    const SliceInfo &si = b->slices[s];
    if (si.D > 1 && si.delay < opt.n_down + b->groups[si.group].H) {
      set_error("bank_create: slice %d at %d Hz has delay %lld < n_down + halo = %d samples", s, si.rate, si.delay,
                opt.n_down + b->groups[si.group].H);
      delete b; return LLOID_ELATENCY;
    }
  }
  // ---- copy U (kept on the host for stacking at stream_create) and R
  std::vector<float> Rh;
  try {
    for (int s = 0; s < S; ++s) b->slices[s].U.resize((size_t)b->slices[s].L * b->slices[s].N);
    Rh.assign((size_t)2 * b->Mpad * b->Kpad, 0.f);
  } catch (const std::bad_alloc &) { set_error("bank_create: out of host memory"); delete b; return LLOID_ENOMEM; }
  std::vector<float> tmp;
  for (int s = 0; s < S; ++s) {
    SliceInfo &si = b->slices[s];
    cudaError_t e = cudaMemcpy(si.U.data(), sl[s].basis, si.U.size() * sizeof(float), cudaMemcpyDefault);
    if (e == cudaSuccess) {
      tmp.resize((size_t)2 * M * si.L);
      e = cudaMemcpy(tmp.data(), sl[s].recon, tmp.size() * sizeof(float), cudaMemcpyDefault);
    }
    if (e != cudaSuccess) { set_error("bank_create: copy of slice %d failed: %s", s, cudaGetErrorString(e)); lloid_bank_destroy(b); return LLOID_ECUDA; }
    // de-interleave rows: part 0 = real rows 2j, part 1 = imaginary rows 2j+1; column = koff_s + l
    for (int j = 0; j < M; ++j)
      for (int part = 0; part < 2; ++part) {
        const float *src = &tmp[(size_t)(2 * j + part) * si.L];
        float *dst = &Rh[((size_t)part * b->Mpad + j) * b->Kpad + si.koff];
        memcpy(dst, src, sizeof(float) * si.L);
      }
  }
  cudaError_t e;
  if (opt.precision == LLOID_PREC_FP32_FFMA) {
    e = cudaMalloc(&b->dR32, Rh.size() * sizeof(float));
    if (e != cudaSuccess) { set_error("bank_create: cudaMalloc R: %s", cudaGetErrorString(e)); lloid_bank_destroy(b); return LLOID_ENOMEM; }
    e = cudaMemcpy(b->dR32, Rh.data(), Rh.size() * sizeof(float), cudaMemcpyHostToDevice);
  } else {
    // fp16 operand(s): scale by a power of two so that the largest entry sits near 2^10, then hi (+ lo) planes
    float mx = 0.f;
    for (float v : Rh) mx = fmaxf(mx, fabsf(v));
    int ex = 0;
    if (mx > 0.f && std::isfinite(mx)) { frexpf(mx, &ex); ex = 10 - ex; }
    if (ex > 24) ex = 24;
    if (ex < -24) ex = -24;
    b->r_scale = ldexpf(1.f, ex);
    b->r_planes = (opt.precision == LLOID_PREC_F16_SPLIT) ? 2 : 1;
    std::vector<__half> R16;
    try { R16.resize(Rh.size() * b->r_planes); } catch (const std::bad_alloc &) { set_error("bank_create: out of host memory"); lloid_bank_destroy(b); return LLOID_ENOMEM; }
    for (size_t i = 0; i < Rh.size(); ++i) {
      float v = Rh[i] * b->r_scale;
      __half h = __float2half_rn(v);
      R16[i] = h;
      if (b->r_planes == 2) {
        // correction plane: 16 bits = { e4m3(R_hi / 4), e4m3(256 R_lo) }, the A operand of the one
        // fp8 MMA that adds R_hi Y_lo + R_lo Y_hi (its B operand is the matching { e5m2(4 Y_lo), e5m2(Y_hi / 256) })
        const float hf = __half2float(h);
        const unsigned lo8 = __nv_cvt_float_to_fp8(hf * 0.25f, __NV_SATFINITE, __NV_E4M3);
        const unsigned hi8 = __nv_cvt_float_to_fp8((v - hf) * 256.f, __NV_SATFINITE, __NV_E4M3);
        R16[Rh.size() + i] = __ushort_as_half((unsigned short)(lo8 | (hi8 << 8)));
      }
    }
    e = cudaMalloc(&b->dR16, R16.size() * sizeof(__half));
    if (e != cudaSuccess) { set_error("bank_create: cudaMalloc R: %s", cudaGetErrorString(e)); lloid_bank_destroy(b); return LLOID_ENOMEM; }
    e = cudaMemcpy(b->dR16, R16.data(), R16.size() * sizeof(__half), cudaMemcpyHostToDevice);
  }
  if (e != cudaSuccess) { set_error("bank_create: upload of R failed: %s", cudaGetErrorString(e)); lloid_bank_destroy(b); return LLOID_ECUDA; }
  *out = b;
  return LLOID_OK;
}

// Template autocorrelations for the xi^2 statistic of Eq. 10: R_j(t), t = -delta..delta.
extern "C" int lloid_bank_set_autocorrelation(lloid_bank *b, const float *acorr, int32_t delta) {
  if (!b || !acorr || delta < 1) { set_error("bank_set_autocorrelation: NULL pointer or delta < 1"); return LLOID_EINVAL; }
  const size_t n = (size_t)b->M * (2 * (size_t)delta + 1);
  std::vector<float> h(2 * n);
  cudaError_t e = cudaMemcpy(h.data(), acorr, h.size() * sizeof(float), cudaMemcpyDefault);
  if (e != cudaSuccess) { set_error("bank_set_autocorrelation: copy failed: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  std::vector<float> den(b->M);
  for (int j = 0; j < b->M; ++j) {
    double d = 0;
    for (int u = 0; u <= 2 * delta; ++u) {
      const double re = h[2 * ((size_t)j * (2 * delta + 1) + u)], im = h[2 * ((size_t)j * (2 * delta + 1) + u) + 1];
      d += 2.0 - 2.0 * (re * re + im * im);
    }
    den[j] = (float)d;
  }
  if (b->dAcorr) { cudaFree(b->dAcorr); b->dAcorr = nullptr; }
  if (b->dXiDen) { cudaFree(b->dXiDen); b->dXiDen = nullptr; }
  if (cudaMalloc(&b->dAcorr, n * sizeof(float2)) != cudaSuccess || cudaMalloc(&b->dXiDen, b->M * sizeof(float)) != cudaSuccess) {
    set_error("bank_set_autocorrelation: cudaMalloc failed"); return LLOID_ENOMEM;
  }
  e = cudaMemcpy(b->dAcorr, h.data(), n * sizeof(float2), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(b->dXiDen, den.data(), b->M * sizeof(float), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { set_error("bank_set_autocorrelation: upload failed: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  b->xi_delta = delta;
  return LLOID_OK;
}
