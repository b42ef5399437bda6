// lloid_stream_*: device-resident streaming state (per-rate strain rings, per-class Y rings), the stacking of
// equal-geometry slices across banks ("multidimensional filtering"), and the per-push launch
// sequence  K1 decimate -> a2 correlate -> K_up upsample -> a3 reconstruct+peaks -> finalize.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <new>
#include <tuple>

#include <cuda_fp8.h>

#include "lloid_internal.h"

using namespace lloid;

struct lloid_stream {
  std::vector<const lloid_bank *> banks;
  int n_det, B, f0, precision, n_down, Mtot, n_tt, max_mtiles, overlap;
  int *bank_off_dev;                               // [n_banks + 1] template offsets (coincidence / clustering)
  int xi_delta;                                    // > 0: xi^2 enabled (every bank carries autocorrelations of this half width)
  YupCopy *ycopy_dev; int n_ycopy;                 // xi^2: pieces of the per-push copy of upsampled Y into the history ring
  lloid_peak *peaks_hist[2];                       // xi^2: triggers of the last two pushes
  float *xi_partial_dev, *xi_den_dev;              // xi^2: [n_det][Mtot][4] numerators; [Mtot] denominators
  long long n_pushes;
  int n_phase;                                     // batch-ahead: pushes per batch of the deep classes (1 = off)
  PeakPartial *tail_dev, *tail_partial_dev;        // overlapped trigger windows: previous buffer's tail peak, this buffer's partials
  float threshold;
  cudaStream_t st;
  long long n0_host;
  long long *n0_dev;
  DecimParams dec;
  std::vector<CorrClass> classes;
  CorrClass *classes_dev;
  CorrTile *tiles_dev; int n_tiles;
  UpItem *items_dev; UpRow *uprows_dev; int n_items;
  float *uptaps_dev; int *uptap_off_dev;
  ReconBank *rbanks_dev;
  std::vector<ReconBank> rbanks;
  PeakPartial *partial_dev;                        // [n_det][n_tt][Mtot] partial peaks (slot-major)
  float *strain_dev; lloid_peak *peaks_dev;       // staging for push_host
  // push_host_async: two pushes in flight.  Two device peak buffers (the first is peaks_dev), a copy stream that drains
  // buffer b while the next push computes, and per buffer the events "kernels done" / "D2H done"
  lloid_peak *peaks_async[2]; cudaStream_t copy_st; cudaEvent_t ev_done[2], ev_copied[2]; long long n_async; bool async_ready;
  std::vector<void *> allocs;                      // every cudaMalloc of this stream
  std::vector<std::pair<void *, size_t>> state;    // (ptr, bytes) zeroed by reset
  int up_planes, up_chunk;
  UpTaps2 taps2;                                   // x2 interpolation taps (kernel parameter of the upsampler)
  bool failed;                                     // a launch of an earlier push failed: state is inconsistent until reset
  double work[8];
  bool stage_timing;
  std::vector<cudaEvent_t> ev_pool;               // free events
  std::vector<std::vector<cudaEvent_t>> ev_rec;    // per timed push: LLOID_N_STAGES + 1 events
  TcPlan *tc;                                      // tensor-core launch plan (kernels_tc.cu), nullptr for FFMA
};

static double sinc_pi(double x) { return x == 0.0 ? 1.0 : std::sin(M_PI * x) / (M_PI * x); }
// Eq. 4: g[k] = sinc((k-c)/f) sinc((k-c)/c), c = f*half_len, k = 0..2c
static std::vector<double> eq4_kernel(int f, int half_len) {
  int c = f * half_len;
  std::vector<double> g(2 * c + 1);
  for (int k = 0; k <= 2 * c; ++k) g[k] = sinc_pi((double)(k - c) / f) * sinc_pi((double)(k - c) / c);
  return g;
}

template <typename T>
static cudaError_t dev_alloc(lloid_stream *s, T **p, size_t count, bool is_state = false) {
  void *q = nullptr;
  size_t bytes = std::max<size_t>(count * sizeof(T), 16);
  cudaError_t e = cudaMalloc(&q, bytes);
  if (e != cudaSuccess) return e;
  e = cudaMemset(q, 0, bytes);
  s->allocs.push_back(q);
  if (is_state) s->state.push_back({q, bytes});
  *p = (T *)q;
  return e;
}
template <typename T>
static cudaError_t dev_upload(lloid_stream *s, T **p, const std::vector<T> &h) {
  cudaError_t e = dev_alloc(s, p, h.size());
  if (e != cudaSuccess || h.empty()) return e;
  return cudaMemcpy(*p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
}

extern "C" void lloid_stream_destroy(lloid_stream *s) {
  if (!s) return;
  if (s->tc) tc_plan_destroy(s->tc);
  for (auto &v : s->ev_rec) for (cudaEvent_t e : v) cudaEventDestroy(e);
  for (cudaEvent_t e : s->ev_pool) cudaEventDestroy(e);
  if (s->async_ready) {
    cudaStreamSynchronize(s->copy_st);
    for (int i = 0; i < 2; ++i) { cudaEventDestroy(s->ev_done[i]); cudaEventDestroy(s->ev_copied[i]); }
    cudaStreamDestroy(s->copy_st);
  }
  for (void *p : s->allocs) cudaFree(p);
  delete s;
}

#define CK(expr)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (expr);                                                                       \
    if (e_ != cudaSuccess) {                                                                       \
      set_error("stream_create: %s: %s", #expr, cudaGetErrorString(e_));                           \
      lloid_stream_destroy(s);                                                                     \
      return (e_ == cudaErrorMemoryAllocation) ? LLOID_ENOMEM : LLOID_ECUDA;                       \
    }                                                                                              \
  } while (0)

extern "C" int lloid_stream_create(lloid_stream **out, const lloid_bank *const *banks, int32_t n_banks,
                                   int32_t n_det, int32_t B, void *cuda_stream) {
  if (!out) { set_error("stream_create: out is NULL"); return LLOID_EINVAL; }
  *out = nullptr;
  if (!banks || n_banks < 1 || n_det < 1 || B < 1) { set_error("stream_create: need banks, n_banks, n_detectors, buffer_len >= 1"); return LLOID_EINVAL; }
  int Dmax = 1;
  for (int b = 0; b < n_banks; ++b) {
    if (!banks[b]) { set_error("stream_create: bank %d is NULL", b); return LLOID_EINVAL; }
    if (banks[b]->f0 != banks[0]->f0 || banks[b]->opt.precision != banks[0]->opt.precision ||
        banks[b]->opt.n_down != banks[0]->opt.n_down || banks[b]->opt.threshold != banks[0]->opt.threshold ||
        banks[b]->opt.trigger_overlap != banks[0]->opt.trigger_overlap) {
      set_error("stream_create: bank %d differs from bank 0 in strain rate, precision, n_down, threshold or trigger_overlap", b); return LLOID_EINVAL;
    }
    for (const SliceInfo &si : banks[b]->slices) Dmax = std::max(Dmax, si.D);
  }
  if (banks[0]->opt.trigger_overlap >= B) { set_error("stream_create: trigger_overlap %d must be smaller than buffer_len %d", banks[0]->opt.trigger_overlap, B); return LLOID_EINVAL; }
  if (B % Dmax != 0) { set_error("stream_create: buffer_len %d is not a multiple of the largest decimation factor %d", B, Dmax); return LLOID_EINVAL; }
  lloid_stream *s = new (std::nothrow) lloid_stream();
  if (!s) { set_error("stream_create: out of host memory"); return LLOID_ENOMEM; }
  s->banks.assign(banks, banks + n_banks);
  s->n_det = n_det; s->B = B; s->f0 = banks[0]->f0; s->precision = banks[0]->opt.precision;
  s->n_down = banks[0]->opt.n_down; s->threshold = banks[0]->opt.threshold; s->overlap = banks[0]->opt.trigger_overlap;
  s->tail_dev = nullptr; s->tail_partial_dev = nullptr;
  s->n_pushes = 0; s->n_ycopy = 0; s->ycopy_dev = nullptr; s->peaks_hist[0] = s->peaks_hist[1] = nullptr;
  s->xi_partial_dev = s->xi_den_dev = nullptr;
  // xi^2 (Eq. 10) runs when EVERY bank carries autocorrelations of one half width; it needs the split tensor mode and
  // 128-sample-aligned buffers longer than the half width (the history ring is addressed in whole tiles)
  s->xi_delta = banks[0]->xi_delta;
  for (int b = 0; b < n_banks; ++b) if (banks[b]->xi_delta != s->xi_delta) s->xi_delta = 0;
  if (s->precision != LLOID_PREC_F16_SPLIT || B % 128 != 0 || s->xi_delta >= B) s->xi_delta = 0;
  s->async_ready = false; s->n_async = 0; s->peaks_async[0] = s->peaks_async[1] = nullptr;
  s->st = (cudaStream_t)cuda_stream; s->n0_host = 0; s->tc = nullptr; s->stage_timing = false; s->failed = false;
  s->up_planes = s->precision == LLOID_PREC_FP32_FFMA ? 0 : (s->precision == LLOID_PREC_F16 ? 1 : 2);
  const int planes = std::max(1, s->up_planes);
  s->up_chunk = std::min(B, 512);                   // = UP_CHUNK of kernels_stream.cu
  memset(s->work, 0, sizeof(s->work));
  s->n_phase = (s->precision != LLOID_PREC_FP32_FFMA && B < s->f0 && s->f0 % B == 0) ? std::min(64, s->f0 / B) : 1;
  int dev = 0; cudaDeviceProp prop;
  CK(cudaGetDevice(&dev));
  CK(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) { set_error("stream_create: device %s is sm_%d%d, this library is sm_100a only", prop.name, prop.major, prop.minor); lloid_stream_destroy(s); return LLOID_ECUDA; }
  CK(dev_alloc(s, &s->n0_dev, 1, true));
  CK(upsample_configure(&s->taps2));                  // per-device kernel attributes: set on every create

  // ---- rates and their rings
  std::map<int, long long> span;                       // D -> max(delay + N) over slices at that rate
  for (const lloid_bank *bk : s->banks)
    for (const SliceInfo &si : bk->slices) span[si.D] = std::max(span[si.D], si.delay + si.N);
  if ((int)span.size() > LLOID_MAX_RATES) { set_error("stream_create: more than %d distinct rates", LLOID_MAX_RATES); lloid_stream_destroy(s); return LLOID_EINVAL; }
  std::map<int, int> rate_index;
  DecimParams &dp = s->dec;
  memset(&dp, 0, sizeof(dp));
  dp.n_det = n_det; dp.B = B; dp.copy_blocks = std::max(1, std::min(8, B / 256));
  int out_begin = 0;
  for (auto &kv : span) {
    int D = kv.first, ri = dp.n_rates++;
    rate_index[D] = ri;
    RateDev &r = dp.r[ri];
    r.D = D; r.lag = (D == 1) ? 0 : s->n_down; r.c = s->n_down * D; r.n_out = B / D;
    long long need = B / D + kv.second + 256;
    if (D == 1) need = std::max<long long>(need, B + 2LL * s->n_down * Dmax + 256);
    r.rlen = (int)need;
    CK(dev_alloc(s, &r.ring2, (size_t)n_det * 2 * r.rlen, true));
    r.taps = nullptr; r.out_begin = 0;
    if (D > 1) {
      std::vector<double> g = eq4_kernel(D, s->n_down);
      double sum = 0; for (double v : g) sum += v;
      std::vector<float> t(g.size());
      for (size_t k = 0; k < g.size(); ++k) t[k] = (float)(std::sqrt((double)D) * g[k] / sum);
      float *td; CK(dev_upload(s, &td, t)); r.taps = td;
      r.out_begin = out_begin; out_begin += (r.n_out + 7) / 8 * 8;   // groups of 8 outputs never straddle rates
    }
  }
  dp.total_out = out_begin;

  // ---- geometry classes (slices of equal rate stacked across banks).  Slices at one rate with the same
  //      upsample halo H whose tap windows [delay, delay + N) nearly coincide share ONE Hankel operand: the class window
  //      is the union [dmin, emax), every member's U is placed at column emax - (delay_i + N_i) and zero padded, as long
  //      as the union stays within 1.25x of the shortest member (so no member's contraction grows by more than 25 %).
  struct Member { int b, i, L; long long d, e; };
  std::map<std::pair<int, int>, std::vector<Member>> by_rate;   // (D, H) -> slices
  for (int b = 0; b < n_banks; ++b) {
    const lloid_bank *bk = s->banks[b];
    for (int i = 0; i < bk->S; ++i) {
      const SliceInfo &si = bk->slices[i];
      by_rate[{si.D, bk->groups[si.group].H}].push_back({b, i, si.L, si.delay, si.delay + si.N});
    }
  }
  std::vector<std::vector<Member>> members;                      // class -> members
  std::vector<std::vector<int>> row_off(n_banks), cls_of(n_banks);
  for (int b = 0; b < n_banks; ++b) { row_off[b].resize(s->banks[b]->S); cls_of[b].resize(s->banks[b]->S); }
  for (auto &kv : by_rate) {
    std::vector<Member> &v = kv.second;
    std::stable_sort(v.begin(), v.end(), [](const Member &x, const Member &y) { return x.d != y.d ? x.d < y.d : x.e < y.e; });
    size_t i0 = 0;
    while (i0 < v.size()) {
      long long dmin = v[i0].d, emax = v[i0].e, nmin = v[i0].e - v[i0].d;
      size_t i1 = i0 + 1;
      for (; i1 < v.size(); ++i1) {
        const long long d2 = std::min(dmin, v[i1].d), e2 = std::max(emax, v[i1].e), n2 = std::min(nmin, v[i1].e - v[i1].d);
        if ((e2 - d2) * 4 > n2 * 5) break;
        dmin = d2; emax = e2; nmin = n2;
      }
      const int c = (int)s->classes.size();
      CorrClass cc; memset(&cc, 0, sizeof(cc));
      const int D = kv.first.first;
      const RateDev &r = dp.r[rate_index[D]];
      cc.ring2 = r.ring2; cc.ring_det_stride = 2LL * r.rlen; cc.rlen = r.rlen; cc.lag = r.lag; cc.D = D;
      cc.N = (int)(emax - dmin); cc.Npad = (cc.N + 63) / 64 * 64; cc.H = kv.first.second; cc.delay = dmin;
      cc.ncols = B / D; cc.ylen = B / D + 32; cc.u_scale_inv = 1.f; cc.phase = -1;
      // batch-ahead: with short buffers a class whose newest tap lies more than a batch (one second) in the
      // past is correlated once per n_phase pushes for all of them; the phases are staggered over the classes
      if (s->n_phase > 1 && cc.delay >= (long long)(s->n_phase - 1) * (B / D) + cc.H + s->n_down + 8) {
        cc.phase = c % s->n_phase; cc.ncols = s->n_phase * (B / D); cc.ylen = cc.ncols + B / D + 64;
      }
      members.emplace_back();
      // keep bank order inside the class (deterministic row layout)
      std::vector<Member> mm(v.begin() + i0, v.begin() + i1);
      std::stable_sort(mm.begin(), mm.end(), [](const Member &x, const Member &y) { return x.b != y.b ? x.b < y.b : x.i < y.i; });
      for (const Member &m : mm) {
        row_off[m.b][m.i] = cc.Lstack; cls_of[m.b][m.i] = c;
        cc.Lstack += m.L;
        members.back().push_back(m);
      }
      s->classes.push_back(cc);
      i0 = i1;
    }
  }
  std::vector<CorrTile> tiles;
  for (size_t c = 0; c < s->classes.size(); ++c) {
    CorrClass &cc = s->classes[c];
    cc.Lpad = (cc.Lstack + 127) / 128 * 128;
    std::vector<float> U((size_t)cc.Lpad * cc.Npad, 0.f);
    int row = 0;
    double alg = 0;
    for (const Member &m : members[c]) {
      const SliceInfo &si = s->banks[m.b]->slices[m.i];
      const long long off = (cc.delay + cc.N) - m.e;            // class column of the member's oldest tap
      for (int l = 0; l < si.L; ++l, ++row) memcpy(&U[(size_t)row * cc.Npad + off], &si.U[(size_t)l * si.N], sizeof(float) * si.N);
      alg += (double)si.L * si.N;
    }
    if (s->precision == LLOID_PREC_FP32_FFMA) {
      float *p; CK(dev_upload(s, &p, U)); cc.U32 = p;
    } else {
      // fp16 operand planes; orthonormal rows have entries ~1/sqrt(N): scale by 2^ceil(log2 sqrt(N)) first
      int ex = (int)std::ceil(0.5 * std::log2((double)cc.N)) + 2;
      float sc = std::ldexp(1.f, ex);
      cc.u_scale_inv = 1.f / sc;
      std::vector<__half> U16(U.size() * planes);
      for (size_t i = 0; i < U.size(); ++i) {
        float v = U[i] * sc; __half h = __float2half_rn(v);
        U16[i] = h;
        if (planes == 2) {
          // correction plane: per tap 16 bits = { e4m3(U_hi / 4), e4m3(256 U_lo) }
          const float hf = __half2float(h);
          const unsigned lo8 = __nv_cvt_float_to_fp8(hf * 0.25f, __NV_SATFINITE, __NV_E4M3);
          const unsigned hi8 = __nv_cvt_float_to_fp8((v - hf) * 256.f, __NV_SATFINITE, __NV_E4M3);
          U16[U.size() + i] = __ushort_as_half((unsigned short)(lo8 | (hi8 << 8)));
        }
      }
      __half *p; CK(dev_upload(s, &p, U16)); cc.U16 = p;
    }
    cc.nseg = (s->precision == LLOID_PREC_FP32_FFMA) ? 1 : tc_k_segments(cc.Npad);
    if ((size_t)cc.ylen * cc.Lpad >= ((size_t)1 << 31)) {       // the upsampler addresses a ring with 32-bit element offsets
      set_error("stream_create: a basis-output ring of %d columns x %d rows exceeds 2^31 elements; use fewer banks per stream", cc.ylen, cc.Lpad);
      lloid_stream_destroy(s); return LLOID_EINVAL;
    }
    CK(dev_alloc(s, &cc.yring, (size_t)cc.nseg * n_det * cc.ylen * cc.Lpad, true));
    cc.ydet_stride = (long long)cc.ylen * cc.Lpad;
    cc.yseg_stride = (long long)n_det * cc.ydet_stride;
    for (int r0 = 0; r0 < cc.Lstack; r0 += 64)
      for (int c0 = 0; c0 < cc.ncols; c0 += 64) tiles.push_back({(int)c, r0, c0});
    s->work[0] += 2.0 * cc.Lpad * cc.Npad * (B / cc.D) * n_det;             // executed (padded) flop, one pass, per push
    s->work[2] += 2.0 * alg * (B / cc.D) * n_det;
    s->work[5] += (double)cc.Lpad * cc.Npad * (s->precision == LLOID_PREC_FP32_FFMA ? 4 : 2 * planes);
    s->work[6] += 2.0 * 4.0 * cc.Lstack * (B / cc.D) * n_det;
  }
  CK(dev_upload(s, &s->classes_dev, s->classes));
  s->n_tiles = (int)tiles.size();
  CK(dev_upload(s, &s->tiles_dev, tiles));

  // ---- upsampler taps (Eq. 4 with c = 8 f, not normalised) for f = 2 .. 2^11
  {
    std::vector<float> taps; std::vector<int> off(LLOID_MAX_GROUPS + 1, 0);
    for (int lf = 1; lf <= LLOID_MAX_GROUPS; ++lf) {
      if ((1 << lf) > Dmax) { off[lf] = 0; continue; }
      off[lf] = (int)taps.size();
      std::vector<double> g = eq4_kernel(1 << lf, LLOID_NUP);
      for (double v : g) taps.push_back((float)v);
    }
    if (taps.empty()) taps.push_back(0.f);
    CK(dev_upload(s, &s->uptaps_dev, taps));
    CK(dev_upload(s, &s->uptap_off_dev, off));
  }

  // ---- per-bank Yup buffers, upsample items, reconstruction descriptors
  // rows are grouped by upsample chain (stage factors) so that a warp's 32 lanes are 32 rows of ANY slices / banks
  // sharing the chain; within a chain they are ordered by (bank, column) to keep the stores contiguous
  std::map<std::vector<int>, std::vector<UpRow>> chains;
  std::vector<YupCopy> ycopies;
  s->Mtot = 0; s->max_mtiles = 0;
  for (int b = 0; b < n_banks; ++b) {
    const lloid_bank *bk = s->banks[b];
    ReconBank rb; memset(&rb, 0, sizeof(rb));
    // FFMA: fp32 [n_det][B][Kpad]; tensor-core modes: [planes][n_det][Kpad][Bp] 16-bit units, sample-contiguous rows
    const int Bp = s->up_planes == 0 ? B : yup_pitch(B);
    size_t plane_elems = (size_t)n_det * Bp * bk->Kpad;
    void *yup = nullptr;
    if (s->up_planes == 0) { float *p; CK(dev_alloc(s, &p, plane_elems)); yup = p; }
    else { __half *p; CK(dev_alloc(s, &p, plane_elems * planes)); yup = p; }
    if (s->xi_delta > 0) {
      __half *h; CK(dev_alloc(s, &h, plane_elems * planes * 3, true));        // zero = "before the stream started"
      rb.yhist = h; rb.acorr = bk->dAcorr; rb.xi_delta = bk->xi_delta;
      for (int pd = 0; pd < planes * n_det; ++pd) {             // B % 128 == 0 here, so Bp == B: the rows of a piece are contiguous
        YupCopy c;
        c.src = reinterpret_cast<const uint4 *>((const __half *)yup + (size_t)pd * B * bk->Kpad);
        c.dst = reinterpret_cast<uint4 *>(h + (size_t)pd * 3 * B * bk->Kpad);
        const bool byte_rows = pd >= n_det;                     // plane 1: two rows of B bytes per basis row
        c.n_rows = byte_rows ? 2 * bk->Kpad : bk->Kpad;
        c.row16 = (byte_rows ? B : 2 * B) / 16; c.dst_pitch16 = 3 * c.row16;
        ycopies.push_back(c);
      }
    }
    rb.R32 = bk->dR32; rb.R16 = bk->dR16;
    rb.r_part_stride = (long long)bk->Mpad * bk->Kpad; rb.r_plane_stride = 2 * rb.r_part_stride;
    rb.yup = yup; rb.yup_det_stride = (long long)Bp * bk->Kpad; rb.yup_plane_stride = (long long)plane_elems;
    rb.M = bk->M; rb.Mpad = bk->Mpad; rb.Kpad = bk->Kpad; rb.tmpl_off = s->Mtot;
    rb.inv_scale = 1.f / bk->r_scale; rb.inv_scale2 = rb.inv_scale * rb.inv_scale;
    s->rbanks.push_back(rb);
    s->Mtot += bk->M;
    s->max_mtiles = std::max(s->max_mtiles, (bk->M + 63) / 64);
    double rate_sum = 0, up_out = 0;
    for (int g = 0; g < bk->G; ++g) { if (g > 0) up_out += bk->groups[g - 1].rate; }
    for (int i = 0; i < bk->S; ++i) {
      const SliceInfo &si = bk->slices[i];
      const CorrClass &cc = s->classes[cls_of[b][i]];
      std::vector<int> key;
      key.push_back(si.D);
      key.push_back(cc.ylen);                        // rows of batch-ahead classes live in longer Y rings: never in one item with others
      for (int h = 1; h <= si.group; ++h) key.push_back((int)std::lround(std::log2((double)bk->groups[h].f)));
      std::vector<UpRow> &dst = chains[key];
      for (int l = 0; l < si.L; ++l) {
        UpRow r; memset(&r, 0, sizeof(r));
        r.ysrc = cc.yring + row_off[b][i] + l; r.ydet_stride = cc.ydet_stride; r.yseg_stride = cc.yseg_stride;
        r.nseg = cc.nseg; r.ypitch = cc.Lpad;
        r.yup = yup; r.yup_det_stride = rb.yup_det_stride; r.yup_plane_stride = rb.yup_plane_stride;
        if (s->up_planes == 0) { r.dst0 = si.koff + l; r.kpitch = bk->Kpad; }
        else { r.dst0 = (long long)(si.koff + l) * Bp; r.kpitch = Bp; }
        r.bank = b;
        dst.push_back(r);
      }
      rate_sum += (double)si.L * si.rate;
    }
    double secs = (double)B / s->f0;
    s->work[1] += 2.0 * 2 * bk->Mpad * (double)bk->Kpad * B * n_det;
    s->work[3] += 2.0 * 2 * bk->M * rate_sum * secs * n_det;
    s->work[4] += 16.0 * 2 * bk->M * up_out * secs * n_det;
    s->work[5] += 2.0 * bk->Mpad * bk->Kpad * (s->precision == LLOID_PREC_FP32_FFMA ? 4 : 2 * planes);
    s->work[6] += 2.0 * plane_elems * (s->up_planes == 0 ? 4 : 2 * planes);
  }
  std::vector<UpItem> items;
  std::vector<UpRow> uprows;
  for (auto &kv : chains) {
    const std::vector<int> &key = kv.first;
    for (size_t r0 = 0; r0 < kv.second.size(); r0 += 32) {
      UpItem it; memset(&it, 0, sizeof(it));
      it.row0 = (int)(uprows.size() + r0); it.nl = (int)std::min<size_t>(32, kv.second.size() - r0);
      it.g = (int)key.size() - 2; it.ylen = key[1];
      for (int h = 1; h <= it.g; ++h) it.log2f[h] = key[h + 1];
      items.push_back(it);
    }
    uprows.insert(uprows.end(), kv.second.begin(), kv.second.end());
  }
  // Items that write the same Yup lines (the same banks, other chains) should run close together in time: a warp of a
  // small slice fills only part of a 32-byte sector and the rest comes from another item; if that item runs much later
  // the line has left the L2 and DRAM sees a read-modify-write.  Order the items by the bank of their first row.
  // Only needed when the upsampled-Y arrays of all banks do not fit the L2 (126 MB); below that the chain-major order
  // (shallow chains first) measured faster (config 2: 45 us against 49.5 us bank-major, 52.8 us deepest-first).
  if (s->work[6] / 2 > 100e6)
    std::stable_sort(items.begin(), items.end(), [&](const UpItem &x, const UpItem &y) { return uprows[x.row0].bank < uprows[y.row0].bank; });
  s->n_items = (int)items.size();
  CK(dev_upload(s, &s->items_dev, items));
  CK(dev_upload(s, &s->uprows_dev, uprows));
  CK(dev_upload(s, &s->rbanks_dev, s->rbanks));
  {
    std::vector<int> off;
    for (const ReconBank &rb : s->rbanks) off.push_back(rb.tmpl_off);
    off.push_back(s->Mtot);
    CK(dev_upload(s, &s->bank_off_dev, off));
  }
  s->n_tt = (B + 63) / 64;
  CK(dev_alloc(s, &s->strain_dev, (size_t)n_det * B));
  CK(dev_alloc(s, &s->peaks_dev, (size_t)n_det * s->Mtot));
  s->peaks_async[0] = s->peaks_dev;
  CK(dev_alloc(s, &s->peaks_async[1], (size_t)n_det * s->Mtot));
  CK(cudaStreamCreateWithFlags(&s->copy_st, cudaStreamNonBlocking));
  for (int i = 0; i < 2; ++i) {
    CK(cudaEventCreateWithFlags(&s->ev_done[i], cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&s->ev_copied[i], cudaEventDisableTiming));
  }
  s->async_ready = true;
  if (s->precision != LLOID_PREC_FP32_FFMA) {
    int rc = tc_plan_create(&s->tc, s->classes, s->classes_dev, s->rbanks, s->rbanks_dev, n_det, B, planes, s->overlap, s->xi_delta, s->n_phase);
    if (rc != LLOID_OK) { lloid_stream_destroy(s); return rc; }
    s->n_tt = tc_plan_n_tt(s->tc);                 // partial peaks per template: the larger of the two a3 kernels' splits
    s->work[0] *= (planes == 2 ? 2 : 1);           // split mode: two MMAs per product in a2 (U_hi x, U_lo x) and in a3
    s->work[1] *= (planes == 2 ? 2 : 1);           // (fp16 R_hi Y_hi + one fp8 MMA carrying both cross terms)
  }
  // partial-peak slots a kernel never writes hold p = -3 (below every real partial, finalize ignores them)
  CK(dev_alloc(s, &s->partial_dev, (size_t)n_det * s->Mtot * s->n_tt));
  CK(launch_fill_partial(s->partial_dev, (size_t)n_det * s->Mtot * s->n_tt, s->st));
  if (s->overlap > 0) {
    // zeroed tail state = "no tail peak" (index 0 lies outside the overlap): reset restores it
    CK(dev_alloc(s, &s->tail_dev, (size_t)n_det * s->Mtot, true));
    CK(dev_alloc(s, &s->tail_partial_dev, (size_t)n_det * s->Mtot * 4));
    CK(launch_fill_partial(s->tail_partial_dev, (size_t)n_det * s->Mtot * 4, s->st));
  }
  if (s->xi_delta > 0) {
    s->n_ycopy = (int)ycopies.size();
    CK(dev_upload(s, &s->ycopy_dev, ycopies));
    CK(dev_alloc(s, &s->peaks_hist[0], (size_t)n_det * s->Mtot));
    CK(dev_alloc(s, &s->peaks_hist[1], (size_t)n_det * s->Mtot));
    CK(dev_alloc(s, &s->xi_partial_dev, (size_t)n_det * s->Mtot * 4));
    CK(dev_alloc(s, &s->xi_den_dev, (size_t)s->Mtot));
    for (size_t b = 0; b < s->banks.size(); ++b)
      CK(cudaMemcpy(s->xi_den_dev + s->rbanks[b].tmpl_off, s->banks[b]->dXiDen, sizeof(float) * s->banks[b]->M, cudaMemcpyDeviceToDevice));
  }
  CK(cudaDeviceSynchronize());
  *out = s;
  return LLOID_OK;
}
#undef CK

extern "C" int lloid_stream_push(lloid_stream *s, const float *strain, lloid_peak *peaks, float *snr_debug,
                                 int32_t debug_bank) {
  if (!s || !strain || !peaks) { set_error("stream_push: stream, strain and peaks must be non-NULL"); return LLOID_EINVAL; }
  if (snr_debug && (debug_bank < 0 || debug_bank >= (int)s->banks.size())) { set_error("stream_push: debug_bank %d out of range", debug_bank); return LLOID_ESTATE; }
  if (s->failed) { set_error("stream_push: an earlier push failed part-way; call lloid_state_reset first"); return LLOID_ESTATE; }
  std::vector<cudaEvent_t> ev;
  if (s->stage_timing) {
    for (int i = 0; i <= LLOID_N_STAGES; ++i) {
      cudaEvent_t x;
      if (!s->ev_pool.empty()) { x = s->ev_pool.back(); s->ev_pool.pop_back(); }
      else if (cudaEventCreate(&x) != cudaSuccess) { set_error("stream_push: cudaEventCreate failed"); return LLOID_ECUDA; }
      ev.push_back(x);
    }
  }
  auto mark = [&](int i) { if (s->stage_timing) cudaEventRecord(ev[i], s->st); };
  mark(0);
  const char *where = "a1 decimate";
  cudaError_t e = launch_decimate(s->dec, strain, s->n0_dev, s->st);
  mark(1);
  if (e == cudaSuccess) {
    where = "a2 correlate";
    if (s->tc) e = tc_launch_corr(s->tc, s->n0_dev, s->st, s->n_pushes == 0 ? s->n_phase : (int)(s->n_pushes % s->n_phase));
    else e = launch_corr_ffma(s->classes_dev, s->tiles_dev, s->n_tiles, s->n_det, s->n0_dev, s->st);
  }
  mark(2);
  if (e == cudaSuccess) where = "a4 upsample";
  if (e == cudaSuccess)
    e = launch_upsample(s->items_dev, s->uprows_dev, s->n_items, s->n_det, s->B, s->up_chunk, s->uptaps_dev, s->uptap_off_dev,
                        s->n0_dev, s->up_planes, s->taps2, s->st);
  if (e == cudaSuccess && s->xi_delta > 0) e = launch_yup_copy(s->ycopy_dev, s->n_ycopy, (int)(s->n_pushes % 3), s->st);
  mark(3);
  if (e == cudaSuccess) {
    where = "a3 reconstruct";
    if (s->tc) e = tc_launch_recon(s->tc, s->partial_dev, s->Mtot, snr_debug, snr_debug ? debug_bank : -1, s->st);
    else e = launch_recon_ffma(s->rbanks_dev, (int)s->banks.size(), s->max_mtiles, s->n_det, s->B, s->partial_dev,
                               s->Mtot, snr_debug, snr_debug ? debug_bank : -1, s->st);
  }
  if (e == cudaSuccess && s->overlap > 0) e = tc_launch_recon_tail(s->tc, s->tail_partial_dev, s->Mtot, s->st);
  mark(4);
  if (e == cudaSuccess) where = "a5 finalize";
  if (e == cudaSuccess)
    e = launch_finalize(s->partial_dev, s->n_det, s->Mtot, s->n_tt, s->threshold, peaks, s->n0_dev, s->B, s->tail_dev,
                        s->tail_partial_dev, s->overlap, s->st);
  if (e == cudaSuccess && s->xi_delta > 0)
    e = cudaMemcpyAsync(s->peaks_hist[s->n_pushes & 1], peaks, sizeof(lloid_peak) * s->n_det * s->Mtot, cudaMemcpyDeviceToDevice, s->st);
  mark(5);
  if (s->stage_timing) s->ev_rec.push_back(std::move(ev));
  if (e != cudaSuccess) {
    // kernels already enqueued have appended to the rings while the stream clock did not advance: the state is
    // inconsistent, so the stream refuses further pushes (LLOID_ESTATE) until lloid_state_reset
    s->failed = true;
    set_error("stream_push: launch of %s failed: %s (stream needs lloid_state_reset)", where, cudaGetErrorString(e)); return LLOID_ECUDA;
  }
  s->n0_host += s->B;
  s->n_pushes += 1;
  return LLOID_OK;
}

// xi^2 (Eq. 10) of the triggers of the push BEFORE the last one: their +-delta windows reach into the last push.
extern "C" int lloid_stream_xi2(lloid_stream *s, float *xi2_out) {
  if (!s || !xi2_out) { set_error("stream_xi2: NULL argument"); return LLOID_EINVAL; }
  if (s->xi_delta <= 0) { set_error("stream_xi2: not enabled (every bank needs lloid_bank_set_autocorrelation with one half width, "
                                    "LLOID_PREC_F16_SPLIT, buffer_len a multiple of 128 and longer than the half width)"); return LLOID_ESTATE; }
  if (s->failed || s->n_pushes < 2) { set_error("stream_xi2: needs two pushes (the statistic lags by one buffer)"); return LLOID_ESTATE; }
  const long long b = s->n_pushes - 2;                              // the target buffer
  cudaError_t e = tc_launch_xi2(s->tc, s->peaks_hist[b & 1], s->xi_partial_dev, s->Mtot, (int)(b % 3) * s->B, s->st);
  if (e == cudaSuccess) e = launch_xi2_finalize(s->xi_partial_dev, s->peaks_hist[b & 1], s->xi_den_dev, s->n_det, s->Mtot, xi2_out, s->st);
  if (e != cudaSuccess) { set_error("stream_xi2: launch failed: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  return LLOID_OK;
}

extern "C" int lloid_stream_events(lloid_stream *s, const lloid_peak *peaks, const int32_t *dt_samples, lloid_event *events) {
  if (!s || !peaks || !dt_samples || !events) { set_error("stream_events: NULL argument"); return LLOID_EINVAL; }
  if (s->n_det > LLOID_MAX_DET) { set_error("stream_events: at most %d detectors", LLOID_MAX_DET); return LLOID_EINVAL; }
  for (int a = 0; a < s->n_det; ++a)
    for (int c = 0; c < s->n_det; ++c)
      if (dt_samples[a * s->n_det + c] < 0 || dt_samples[a * s->n_det + c] != dt_samples[c * s->n_det + a]) {
        set_error("stream_events: dt_samples must be symmetric and non-negative"); return LLOID_EINVAL;
      }
  cudaError_t e = launch_coinc_cluster(peaks, s->n_det, s->Mtot, s->bank_off_dev, (int)s->banks.size(), dt_samples, events, s->st);
  if (e != cudaSuccess) { set_error("stream_events: launch failed: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  return LLOID_OK;
}

extern "C" int lloid_stream_push_host(lloid_stream *s, const float *strain_host, lloid_peak *peaks_host) {
  if (!s || !strain_host || !peaks_host) { set_error("stream_push_host: NULL argument"); return LLOID_EINVAL; }
  cudaError_t e = cudaMemcpyAsync(s->strain_dev, strain_host, sizeof(float) * s->n_det * s->B, cudaMemcpyHostToDevice, s->st);
  if (e != cudaSuccess) { set_error("stream_push_host: H2D copy: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  int rc = lloid_stream_push(s, s->strain_dev, s->peaks_dev, nullptr, -1);
  if (rc != LLOID_OK) return rc;
  e = cudaMemcpyAsync(peaks_host, s->peaks_dev, sizeof(lloid_peak) * s->n_det * s->Mtot, cudaMemcpyDeviceToHost, s->st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->st);
  if (e != cudaSuccess) { set_error("stream_push_host: D2H copy / sync: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  return LLOID_OK;
}

// Pipelined variant: returns as soon as the work is queued.  Call n computes into device peak buffer n & 1; a separate copy
// stream moves it to peaks_host while call n + 1 computes.  Before reusing buffer n & 1, call n + 2 waits for that copy.
extern "C" int lloid_stream_push_host_async(lloid_stream *s, const float *strain_host, lloid_peak *peaks_host) {
  if (!s || !strain_host || !peaks_host) { set_error("stream_push_host_async: NULL argument"); return LLOID_EINVAL; }
  const int b = (int)(s->n_async & 1);
  cudaError_t e = cudaSuccess;
  if (s->n_async >= 2) e = cudaEventSynchronize(s->ev_copied[b]);          // the D2H of call n - 2 has left this buffer
  if (e == cudaSuccess) e = cudaMemcpyAsync(s->strain_dev, strain_host, sizeof(float) * s->n_det * s->B, cudaMemcpyHostToDevice, s->st);
  if (e != cudaSuccess) { set_error("stream_push_host_async: wait / H2D copy: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  int rc = lloid_stream_push(s, s->strain_dev, s->peaks_async[b], nullptr, -1);
  if (rc != LLOID_OK) return rc;
  e = cudaEventRecord(s->ev_done[b], s->st);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(s->copy_st, s->ev_done[b], 0);
  if (e == cudaSuccess) e = cudaMemcpyAsync(peaks_host, s->peaks_async[b], sizeof(lloid_peak) * s->n_det * s->Mtot, cudaMemcpyDeviceToHost, s->copy_st);
  if (e == cudaSuccess) e = cudaEventRecord(s->ev_copied[b], s->copy_st);
  if (e != cudaSuccess) { set_error("stream_push_host_async: D2H copy: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  ++s->n_async;
  return LLOID_OK;
}

extern "C" int lloid_stream_host_sync(lloid_stream *s) {
  if (!s) { set_error("stream_host_sync: stream is NULL"); return LLOID_EINVAL; }
  cudaError_t e = cudaStreamSynchronize(s->st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->copy_st);
  if (e != cudaSuccess) { set_error("stream_host_sync: %s", cudaGetErrorString(e)); s->failed = true; return LLOID_ECUDA; }
  return LLOID_OK;
}

extern "C" int lloid_state_reset(lloid_stream *s) {
  if (!s) { set_error("state_reset: stream is NULL"); return LLOID_EINVAL; }
  for (auto &p : s->state) {
    cudaError_t e = cudaMemsetAsync(p.first, 0, p.second, s->st);
    if (e != cudaSuccess) { set_error("state_reset: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  }
  if (s->async_ready) cudaStreamSynchronize(s->copy_st);     // peaks still on their way to the host are delivered first
  s->n_async = 0;
  s->n0_host = 0;
  s->n_pushes = 0;
  s->failed = false;
  return LLOID_OK;
}

extern "C" int64_t lloid_stream_samples_pushed(const lloid_stream *s) { return s ? s->n0_host : -1; }
extern "C" int32_t lloid_stream_total_templates(const lloid_stream *s) { return s ? s->Mtot : -1; }
extern "C" int32_t lloid_stream_launches_per_push(const lloid_stream *s) { return s ? 4 + (s->tc ? tc_plan_recon_launches(s->tc) : 1) : -1; }
extern "C" int lloid_stream_work_per_push(const lloid_stream *s, double out[8]) {
  if (!s || !out) { set_error("work_per_push: NULL argument"); return LLOID_EINVAL; }
  for (int i = 0; i < 8; ++i) out[i] = s->work[i];
  return LLOID_OK;
}

extern "C" int lloid_stream_set_stage_timing(lloid_stream *s, int32_t enable) {
  if (!s) { set_error("set_stage_timing: stream is NULL"); return LLOID_EINVAL; }
  s->stage_timing = enable != 0;
  return LLOID_OK;
}

extern "C" int lloid_stream_stage_times(lloid_stream *s, float ms[LLOID_N_STAGES]) {
  if (!s || !ms) { set_error("stage_times: NULL argument"); return LLOID_EINVAL; }
  cudaError_t e = cudaStreamSynchronize(s->st);
  if (e != cudaSuccess) { set_error("stage_times: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  for (int i = 0; i < LLOID_N_STAGES; ++i) ms[i] = 0.f;
  int n = 0;
  for (auto &v : s->ev_rec) {
    for (int i = 0; i < LLOID_N_STAGES; ++i) {
      float t = 0.f;
      if (cudaEventElapsedTime(&t, v[i], v[i + 1]) == cudaSuccess) ms[i] += t;
    }
    for (cudaEvent_t x : v) s->ev_pool.push_back(x);
    ++n;
  }
  s->ev_rec.clear();
  return n;
}

extern "C" const char *lloid_stage_name(int32_t i) {
  static const char *names[LLOID_N_STAGES] = {"a1_decimate", "a2_correlate", "a4_upsample_basis", "a3_reconstruct_a5_peaks",
                                              "a5_finalize"};
  return (i >= 0 && i < LLOID_N_STAGES) ? names[i] : "";
}
