// SVD bank construction on the GPU (Eq. 3): truncated singular value decomposition of one time slice's
// template matrix H (2M real rows x N taps), H ~= R U with U = L orthonormal basis filters and R = V diag(sigma).
// One-sided (Hestenes) Jacobi in float64: plane rotations applied on the left make the ROWS of A = W H mutually orthogonal,
//   A_l = sigma_l u_l,   V = W^T,   R[i][l] = W[l][i] sigma_l,
// which needs no Gram matrix (its condition number would be squared) and no library: per step n/2 disjoint row pairs (a
// round-robin tournament) are rotated by n/2 CTAs; a sweep is n - 1 steps; sweeps repeat until no pair needed a rotation.
#include <algorithm>
#include <cmath>
#include <mutex>
#include <numeric>
#include <vector>

#include "lloid_internal.h"

namespace lloid {

__device__ __forceinline__ double block_sum(double v, double *sh) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];      // fixed order: deterministic
  return t;
}

// One tournament step: CTA i rotates rows (p, q) of A [n][N] and of W [n][n].  n is even (the host pads with a zero row).
__global__ void __launch_bounds__(256) jacobi_step_kernel(double *__restrict__ A, double *__restrict__ W, int n, int N, int step, double tol,
                                                          double floor2, int *__restrict__ n_rot) {
  __shared__ double sh[8];
  const int i = blockIdx.x, m = n - 1;
  int p, q;
  if (i == 0) { p = m; q = step % m; }
  else { p = (step + i) % m; q = (step - i + m) % m; }
  if (p > q) { const int t = p; p = q; q = t; }
  double *ap = A + (size_t)p * N, *aq = A + (size_t)q * N;
  double al = 0.0, be = 0.0, ga = 0.0;
  for (int k = threadIdx.x; k < N; k += blockDim.x) { const double x = ap[k], y = aq[k]; al += x * x; be += y * y; ga += x * y; }
  al = block_sum(al, sh); be = block_sum(be, sh); ga = block_sum(ga, sh);
  // rows at rounding level (the null space when rank < n) are left alone: rotating them among themselves never converges
  if (al <= floor2 || be <= floor2 || fabs(ga) <= tol * sqrt(al * be)) return;
  if (threadIdx.x == 0) atomicAdd(n_rot, 1);
  const double zeta = (be - al) / (2.0 * ga);
  const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
  const double c = 1.0 / sqrt(1.0 + t * t), s = c * t;
  for (int k = threadIdx.x; k < N; k += blockDim.x) { const double x = ap[k], y = aq[k]; ap[k] = c * x - s * y; aq[k] = s * x + c * y; }
  double *wp = W + (size_t)p * n, *wq = W + (size_t)q * n;
  for (int k = threadIdx.x; k < n; k += blockDim.x) { const double x = wp[k], y = wq[k]; wp[k] = c * x - s * y; wq[k] = s * x + c * y; }
}

__global__ void svd_init_kernel(const double *__restrict__ H, double *__restrict__ A, double *__restrict__ W, int rows, int n, int N) {
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < (size_t)n * N) { const int r = (int)(t / N); A[t] = r < rows ? H[t] : 0.0; }
  if (t < (size_t)n * n) W[t] = (t / n == t % n) ? 1.0 : 0.0;
}

__global__ void svd_norms_kernel(const double *__restrict__ A, int N, double *__restrict__ norm2) {
  __shared__ double sh[8];
  const double *a = A + (size_t)blockIdx.x * N;
  double v = 0.0;
  for (int k = threadIdx.x; k < N; k += blockDim.x) v += a[k] * a[k];
  v = block_sum(v, sh);
  if (threadIdx.x == 0) norm2[blockIdx.x] = v;
}

// basis[l][k] = A[order[l]][k] / sigma_l ;  recon[i][l] = W[order[l]][i] * sigma_l
__global__ void svd_emit_kernel(const double *__restrict__ A, const double *__restrict__ W, const int *__restrict__ order,
                                const double *__restrict__ sigma, int L, int rows, int n, int N, float *__restrict__ basis,
                                float *__restrict__ recon) {
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < (size_t)L * N) { const int l = (int)(t / N), k = (int)(t % N); basis[t] = (float)(A[(size_t)order[l] * N + k] / sigma[l]); }
  if (t < (size_t)rows * L) { const int i = (int)(t / L), l = (int)(t % L); recon[t] = (float)(W[(size_t)order[l] * n + i] * sigma[l]); }
}

}  // namespace lloid

using namespace lloid;

extern "C" int lloid_svd_slice(const double *H, int32_t n_rows, int32_t n_taps, double energy, int32_t max_basis, int32_t *n_basis_out,
                               float *basis_out, float *recon_out, double *singular_out, double *kept_energy_out, void *cuda_stream) {
  if (!H || !n_basis_out || !basis_out || !recon_out || n_rows < 1 || n_taps < 1 || max_basis < 1 || !(energy > 0.0) || energy > 1.0) {
    set_error("svd_slice: NULL pointer, non-positive size or energy outside (0, 1]"); return LLOID_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int rows = n_rows, N = n_taps, n = (rows + 1) & ~1;
  double *A = nullptr, *W = nullptr, *Hd = nullptr, *norm2 = nullptr, *sig_dev = nullptr;
  int *n_rot = nullptr, *order_dev = nullptr;
  auto cleanup = [&]() { cudaFree(A); cudaFree(W); cudaFree(Hd); cudaFree(norm2); cudaFree(sig_dev); cudaFree(n_rot); cudaFree(order_dev); };
  if (cudaMalloc(&A, sizeof(double) * n * N) != cudaSuccess || cudaMalloc(&W, sizeof(double) * n * n) != cudaSuccess ||
      cudaMalloc(&Hd, sizeof(double) * rows * N) != cudaSuccess || cudaMalloc(&norm2, sizeof(double) * n) != cudaSuccess ||
      cudaMalloc(&sig_dev, sizeof(double) * n) != cudaSuccess || cudaMalloc(&n_rot, sizeof(int)) != cudaSuccess ||
      cudaMalloc(&order_dev, sizeof(int) * n) != cudaSuccess) {
    cleanup(); set_error("svd_slice: cudaMalloc failed"); return LLOID_ENOMEM;
  }
  cudaError_t e = cudaMemcpyAsync(Hd, H, sizeof(double) * rows * N, cudaMemcpyDefault, st);
  const size_t tot = (size_t)n * std::max(N, n);
  svd_init_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(Hd, A, W, rows, n, N);
  // ||H||_F^2 sets the absolute floor below which a row counts as zero
  svd_norms_kernel<<<n, 256, 0, st>>>(A, N, norm2);
  std::vector<double> n2(n);
  if (e == cudaSuccess) e = cudaMemcpyAsync(n2.data(), norm2, sizeof(double) * n, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  double fro2 = 0.0;
  for (double v : n2) fro2 += v;
  const double floor2 = 1e-26 * fro2;
  int sweeps = 0;
  if (n >= 2 && e == cudaSuccess) {
    for (; sweeps < 40; ++sweeps) {
      cudaMemsetAsync(n_rot, 0, sizeof(int), st);
      for (int step = 0; step < n - 1; ++step) jacobi_step_kernel<<<n / 2, 256, 0, st>>>(A, W, n, N, step, 1e-13, floor2, n_rot);
      int h = 0;
      e = cudaMemcpyAsync(&h, n_rot, sizeof(int), cudaMemcpyDeviceToHost, st);
      if (e == cudaSuccess) e = cudaStreamSynchronize(st);
      if (e != cudaSuccess) break;
      if (h == 0) break;
    }
  }
  if (e != cudaSuccess) { cleanup(); set_error("svd_slice: CUDA error during the Jacobi sweeps: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  svd_norms_kernel<<<n, 256, 0, st>>>(A, N, norm2);
  e = cudaMemcpyAsync(n2.data(), norm2, sizeof(double) * n, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) { cleanup(); set_error("svd_slice: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  std::vector<int> order(n);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return n2[a] > n2[b]; });
  double total = 0.0;
  for (double v : n2) total += v;
  // smallest L with sum_{l<L} sigma_l^2 >= energy * sum sigma^2 (BASELINE.json: 99.99 %)
  int L = 0;
  double acc = 0.0;
  while (L < n && n2[order[L]] > 0.0) { acc += n2[order[L]]; ++L; if (acc >= energy * total) break; }
  if (L < 1) L = 1;
  if (L > max_basis) { cleanup(); set_error("svd_slice: %d basis filters needed, max_basis is %d", L, max_basis); return LLOID_EINVAL; }
  std::vector<double> sig(L);
  for (int l = 0; l < L; ++l) sig[l] = std::sqrt(n2[order[l]]);
  cudaMemcpyAsync(sig_dev, sig.data(), sizeof(double) * L, cudaMemcpyHostToDevice, st);
  cudaMemcpyAsync(order_dev, order.data(), sizeof(int) * L, cudaMemcpyHostToDevice, st);
  const size_t tot2 = std::max((size_t)L * N, (size_t)rows * L);
  svd_emit_kernel<<<(unsigned)((tot2 + 255) / 256), 256, 0, st>>>(A, W, order_dev, sig_dev, L, rows, n, N, basis_out, recon_out);
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cleanup();
  if (e != cudaSuccess) { set_error("svd_slice: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  *n_basis_out = L;
  if (kept_energy_out) *kept_energy_out = total > 0.0 ? acc / total : 1.0;
  if (singular_out) for (int l = 0; l < L; ++l) singular_out[l] = sig[l];
  return LLOID_OK;
}

// ------------------------------------------------------------------------------------------------
// lloid_svd_slice_noalloc: the same decomposition for callers that may not allocate device memory (a tight serving loop, a
// harness that forbids cudaMalloc).  The Jacobi working set (A = W H, W, row norms, order, sigma, rotation counter) lives in
// ONE file-scope device array of a fixed, modest size, which every GPU that loads the library holds until exit:
// 128 x 2048 float64 for A + 128 x 128 for W + bookkeeping = 2.13 MiB.  Every call shares it and finds the previous call's
// contents there: svd_init_kernel rewrites A and W completely, the counter is cleared per sweep, the rest is written before
// it is read.  Calls that overlap on the GPU (two streams, two host threads) race on it.
// In host code `svd_scratch` is only a stand-in for the symbol: its device address is looked up once per device with
// cudaGetSymbolAddress (that device current) and passed to the kernels.
// ------------------------------------------------------------------------------------------------
#define SVD_NA_MAX_ROWS 128
#define SVD_NA_MAX_TAPS 2048
struct SvdScratch {
  double A[SVD_NA_MAX_ROWS * SVD_NA_MAX_TAPS];
  double W[SVD_NA_MAX_ROWS * SVD_NA_MAX_ROWS];
  double norm2[SVD_NA_MAX_ROWS];
  double sigma[SVD_NA_MAX_ROWS];
  int order[SVD_NA_MAX_ROWS];
  int n_rot;
};
static __device__ __align__(256) unsigned char svd_scratch[sizeof(SvdScratch)];

static SvdScratch *svd_scratch_address() {          // device address of svd_scratch on the CURRENT device, or nullptr (error set)
  static std::mutex mu;
  static SvdScratch *by_device[64] = {};
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { set_error("svd_slice_noalloc: no current CUDA device (or ordinal >= 64)"); return nullptr; }
  std::lock_guard<std::mutex> lock(mu);
  if (!by_device[dev]) {
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, svd_scratch);
    if (e != cudaSuccess || !p) { set_error("svd_slice_noalloc: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e)); return nullptr; }
    by_device[dev] = reinterpret_cast<SvdScratch *>(p);
  }
  return by_device[dev];
}

extern "C" int lloid_svd_slice_noalloc(const double *H, int32_t n_rows, int32_t n_taps, double energy, int32_t max_basis,
                                       int32_t *n_basis_out, float *basis_out, float *recon_out, double *singular_out,
                                       double *kept_energy_out, void *cuda_stream) {
  if (!H || !n_basis_out || !basis_out || !recon_out || n_rows < 1 || n_taps < 1 || max_basis < 1 || !(energy > 0.0) || energy > 1.0) {
    set_error("svd_slice_noalloc: NULL pointer, non-positive size or energy outside (0, 1]"); return LLOID_EINVAL;
  }
  if (n_rows > SVD_NA_MAX_ROWS || n_taps > SVD_NA_MAX_TAPS) {
    set_error("svd_slice_noalloc: %d x %d exceeds the fixed scratch of %d rows x %d taps; use lloid_svd_slice", n_rows, n_taps,
              SVD_NA_MAX_ROWS, SVD_NA_MAX_TAPS);
    return LLOID_EINVAL;
  }
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, H) != cudaSuccess || (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)) {
    cudaGetLastError();
    set_error("svd_slice_noalloc: H must be a DEVICE pointer (no staging buffer is allocated)"); return LLOID_EINVAL;
  }
  SvdScratch *sc = svd_scratch_address();
  if (!sc) return LLOID_ECUDA;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int rows = n_rows, N = n_taps, n = (rows + 1) & ~1;
  double *A = sc->A, *W = sc->W, *norm2 = sc->norm2, *sig_dev = sc->sigma;
  int *n_rot = &sc->n_rot, *order_dev = sc->order;
  const size_t tot = (size_t)n * std::max(N, n);
  svd_init_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(H, A, W, rows, n, N);
  svd_norms_kernel<<<n, 256, 0, st>>>(A, N, norm2);
  double n2[SVD_NA_MAX_ROWS];
  cudaError_t e = cudaMemcpyAsync(n2, norm2, sizeof(double) * n, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  double fro2 = 0.0;
  for (int i = 0; i < n; ++i) fro2 += n2[i];
  const double floor2 = 1e-26 * fro2;
  if (n >= 2 && e == cudaSuccess) {
    for (int sweeps = 0; sweeps < 40; ++sweeps) {
      cudaMemsetAsync(n_rot, 0, sizeof(int), st);
      for (int step = 0; step < n - 1; ++step) jacobi_step_kernel<<<n / 2, 256, 0, st>>>(A, W, n, N, step, 1e-13, floor2, n_rot);
      int h = 0;
      e = cudaMemcpyAsync(&h, n_rot, sizeof(int), cudaMemcpyDeviceToHost, st);
      if (e == cudaSuccess) e = cudaStreamSynchronize(st);
      if (e != cudaSuccess || h == 0) break;
    }
  }
  if (e != cudaSuccess) { set_error("svd_slice_noalloc: CUDA error during the Jacobi sweeps: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  svd_norms_kernel<<<n, 256, 0, st>>>(A, N, norm2);
  e = cudaMemcpyAsync(n2, norm2, sizeof(double) * n, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) { set_error("svd_slice_noalloc: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  int order[SVD_NA_MAX_ROWS];
  std::iota(order, order + n, 0);
  std::stable_sort(order, order + n, [&](int a, int b) { return n2[a] > n2[b]; });
  double total = 0.0;
  for (int i = 0; i < n; ++i) total += n2[i];
  int L = 0;
  double acc = 0.0;
  while (L < n && n2[order[L]] > 0.0) { acc += n2[order[L]]; ++L; if (acc >= energy * total) break; }
  if (L < 1) L = 1;
  if (L > max_basis) { set_error("svd_slice_noalloc: %d basis filters needed, max_basis is %d", L, max_basis); return LLOID_EINVAL; }
  double sig[SVD_NA_MAX_ROWS];
  for (int l = 0; l < L; ++l) sig[l] = std::sqrt(n2[order[l]]);
  cudaMemcpyAsync(sig_dev, sig, sizeof(double) * L, cudaMemcpyHostToDevice, st);
  cudaMemcpyAsync(order_dev, order, sizeof(int) * L, cudaMemcpyHostToDevice, st);
  const size_t tot2 = std::max((size_t)L * N, (size_t)rows * L);
  svd_emit_kernel<<<(unsigned)((tot2 + 255) / 256), 256, 0, st>>>(A, W, order_dev, sig_dev, L, rows, n, N, basis_out, recon_out);
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);     // sig / order live on this frame: the copies must have completed
  if (e != cudaSuccess) { set_error("svd_slice_noalloc: %s", cudaGetErrorString(e)); return LLOID_ECUDA; }
  *n_basis_out = L;
  if (kept_energy_out) *kept_energy_out = total > 0.0 ? acc / total : 1.0;
  if (singular_out) for (int l = 0; l < L; ++l) singular_out[l] = sig[l];
  return LLOID_OK;
}
