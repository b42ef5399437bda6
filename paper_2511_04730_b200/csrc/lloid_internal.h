// Internal declarations shared by the host code and the kernels of liblloid (not part of the C ABI).
// Notation follows include/lloid.h and DESIGN.md: f0, D = f0/rate, N taps, L bases, delay, group g =
// run of slices at one rate, A_g/H_g = low/high halo (in samples at the group's rate) of the zero-phase
// upsample chain above the group (Eqs. 7-9).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/lloid.h"

#define LLOID_MAX_GROUPS 12   // distinct rates in one bank (2048 .. 1 Hz)
#define LLOID_MAX_RATES 12    // distinct rates in one stream
#define LLOID_NUP 8

namespace lloid {

void set_error(const char *fmt, ...);

// ---------------------------------------------------------------------------------------------- bank
struct SliceInfo {
  int rate, D, N, L, group, koff;   // koff: first column of this slice in the bank's concatenated K axis
  long long delay;
  std::vector<float> U;              // host copy [L][N]; stacked per geometry class at stream_create
};
struct GroupInfo {
  int rate, D, f;                    // f = rate_{g-1}/rate_g (1 for g = 0)
  int A, H;                          // columns [n0/D - A, (n0+B)/D + H) of this group feed one push
  int first_slice, n_slices;
};
}  // namespace lloid

struct lloid_bank {
  int f0, M, Mpad, S, G;
  lloid_options opt;
  std::vector<lloid::SliceInfo> slices;
  std::vector<lloid::GroupInfo> groups;
  int Ktot, Kpad;                    // sum_s L^s and its round-up to 16
  float r_scale;                     // power of two applied to R before the fp16 cast (1 for fp32)
  float *dR32;                       // FFMA:   [2 (re,im)][Mpad][Kpad] fp32
  __half *dR16;                      // tensor: [planes (hi,lo)][2 (re,im)][Mpad][Kpad] fp16, scaled by r_scale
  int r_planes;
  float2 *dAcorr;                    // [M][2 xi_delta + 1] template autocorrelations R_j(t) (Eq. 10), nullptr = none
  float *dXiDen;                     // [M] sum_t (2 - 2 |R_j(t)|^2)
  int xi_delta;
};

// ---------------------------------------------------------------------------------------------- device tables
namespace lloid {

struct RateDev {                     // one per distinct rate in the stream (index 0 = f0)
  float *ring2;                      // [n_det][2*rlen] mirrored ring of the strain decimated to this rate
  const float *taps;                 // sqrt(D)*ghat_D[k], k = 0..2c  (Eq. 4), nullptr for D = 1
  int D, rlen, lag, c;               // ring slot of sample j is (j + lag) mod rlen; lag = n_down (0 for D = 1)
  int out_begin;                     // first flattened decimator output index of this rate in a push
  int n_out;                         // B / D
};

struct DecimParams {
  RateDev r[LLOID_MAX_RATES];
  int n_rates, n_det, B, total_out, copy_blocks;
};

struct CorrClass {                   // slices (across banks) with identical (rate, N, delay, H): stacked U
  const float *ring2;                // rate ring, detector 0
  long long ring_det_stride;
  int rlen, lag, D, N, Npad, H;
  long long delay;
  int Lstack, Lpad;                  // stacked basis rows and their round-up to 128
  const float *U32;                  // [Lpad][Npad] fp32 (FFMA path)
  const __half *U16;                 // [planes][Lpad][Npad] fp16 scaled by u_scale (tensor path)
  float *yring;                      // [nseg][n_det][ylen][Lpad] fp32 ring of Y columns; slot of column j = (j + 64) mod ylen;
                                     // Y = sum over the nseg tap segments (split-K partial sums, added by the reader in order)
  long long ydet_stride, yseg_stride;
  int nseg;
  int ylen, ncols;                   // ncols = B / D new columns per push: [n0/D + H, (n0+B)/D + H)
  float u_scale_inv;
  int phase;                         // batch-ahead (short buffers): -1 = correlated every push; else the push index mod
                                     // n_phase at which this class is correlated for the next n_phase pushes at once
};

struct CorrTile { int cls, row0, col0; };   // FFMA a2 work item: 64 rows x 64 columns

struct UpRow {                       // one basis row of one slice of one bank: where it comes from and where it goes
  const float *ysrc;                 // class Y ring + stacked row index (detector 0, segment 0)
  long long ydet_stride, yseg_stride;
  void *yup;                         // bank's upsampled-Y array (plane 0)
  long long dst0;                    // element offset of (detector 0, sample 0) of this row: its column (FFMA) / column * yup_pitch(B)
  long long yup_det_stride, yup_plane_stride;
  int nseg, ypitch, kpitch, bank;    // kpitch: Kpad (FFMA, sample pitch) / yup_pitch(B) (tensor-core layouts, row pitch);
                                     // bank: index of the owning bank (items are ordered by it for L2 locality)
};
struct UpItem {                      // <= 32 rows (lanes) that share one upsample chain: (rate, stage factors)
  int row0, nl;                      // rows [row0, row0 + nl) of the UpRow table
  int g;                             // number of upsample stages
  int log2f[LLOID_MAX_GROUPS];       // log2 f_h of stage h -> h-1, h = 1..g
  int ylen;                          // Y ring length at this rate (B/D + 32)
};

// Tensor-core modes: the upsampled-Y planes hold one row of yup_pitch(B) samples per (detector, basis row) -- sample-contiguous,
// so that the upsampler stores whole 32-byte sectors and a3 reads them as an MN-major operand
inline int yup_pitch(int B) { return (B + 63) & ~63; }

struct ReconBank {                   // a3 work description of one bank
  const float *R32; const __half *R16; long long r_part_stride, r_plane_stride;
  const void *yup; long long yup_det_stride, yup_plane_stride;
  int M, Mpad, Kpad, tmpl_off;       // tmpl_off: first template of this bank in the stream's peak array
  const void *yhist;                 // xi^2: [planes][n_det][Kpad (x2 byte rows in plane 1)][3 B] ring of the last three pushes' upsampled Y (or nullptr)
  const float2 *acorr; int xi_delta; // xi^2: the bank's autocorrelations
  float inv_scale2;                  // 1/(r_scale^2): applied to |z|^2
  float inv_scale;
};

struct PeakPartial { float p; int idx; float re, im; };

// ---------------------------------------------------------------------------------------------- launchers (kernels_*.cu)
cudaError_t launch_decimate(const DecimParams &P, const float *strain, const long long *n0, cudaStream_t st);
cudaError_t launch_corr_ffma(const CorrClass *cls_dev, const CorrTile *tiles_dev, int n_tiles, int n_det,
                             const long long *n0, cudaStream_t st);
struct UpTaps2 { float t[16]; };     // g_2[2k+1], k = 0..15: the 16 non-zero taps of the x2 interpolation phase (Eq. 7)
cudaError_t upsample_configure(UpTaps2 *t2);
cudaError_t launch_upsample(const UpItem *items_dev, const UpRow *rows_dev, int n_items, int n_det, int B, int chunk, const float *uptaps,
                            const int *uptap_off, const long long *n0, int out_half_planes, const UpTaps2 &t2, cudaStream_t st);
cudaError_t launch_recon_ffma(const ReconBank *banks_dev, int n_banks, int max_mtiles, int n_det, int B,
                              PeakPartial *partial, int Mtot, float *snr_debug, int debug_bank, cudaStream_t st);
// one (bank, plane, detector) piece: n_rows rows of row16 16-byte units (B samples), contiguous in the source, dst_pitch16 apart in the ring
struct YupCopy { const uint4 *src; uint4 *dst; long long n_rows, row16, dst_pitch16; };
cudaError_t launch_yup_copy(const YupCopy *table_dev, int n_pieces, int slot, cudaStream_t st);
cudaError_t launch_xi2_finalize(const float *xi_partial, const lloid_peak *peaks, const float *den, int n_det, int Mtot, float *xi2_out,
                                cudaStream_t st);
cudaError_t launch_fill_partial(PeakPartial *partial, size_t n, cudaStream_t st);
cudaError_t launch_finalize(const PeakPartial *partial, int n_det, int Mtot, int n_tt, float threshold,
                            lloid_peak *peaks, long long *n0, int B, PeakPartial *tail, const PeakPartial *tail_partial, int overlap,
                            cudaStream_t st);

cudaError_t launch_coinc_cluster(const lloid_peak *peaks, int n_det, int Mtot, const int *bank_off_dev, int n_banks,
                                 const int32_t *dt_host, lloid_event *events, cudaStream_t st);   // lloid_events.cu

// ---------------------------------------------------------------------------------------------- tcgen05 path (kernels_tc.cu)
struct TcPlan;
int tc_time_splits(int B, long long n_mtile_units);   // n_mtile_units = sum_banks ceil(M/128) * n_det
int tc_k_segments(int Npad);  // split-K segments of the tensor-core a2 kernel for a slice of Npad taps   // partial peaks per template written by the tensor-core a3 kernel
int tc_plan_create(TcPlan **out, const std::vector<CorrClass> &classes, const CorrClass *classes_dev,
                   const std::vector<ReconBank> &banks, const ReconBank *banks_dev, int n_det, int B, int planes, int overlap,
                   int xi_delta, int n_phase);
void tc_plan_destroy(TcPlan *p);
int tc_plan_n_tt(const TcPlan *p);              // partial peaks per template and detector the a3 kernels write
int tc_plan_recon_launches(const TcPlan *p);    // 1 or 2: streaming kernel and / or resident-R kernel
cudaError_t tc_launch_corr(TcPlan *p, const long long *n0, cudaStream_t st, int list);   // list: phase, or n_phase = every class
cudaError_t tc_launch_recon(TcPlan *p, PeakPartial *partial, int Mtot, float *snr_debug, int debug_bank,
                            cudaStream_t st);
cudaError_t tc_launch_recon_tail(TcPlan *p, PeakPartial *tail_partial, int Mtot, cudaStream_t st);
// xi^2 pass over [-delta, B + delta) of the buffer whose upsampled Y sits at ring rows [row_base, row_base + B) (mod 3 B)
cudaError_t tc_launch_xi2(TcPlan *p, const lloid_peak *peaks, float *xi_partial, int Mtot, int row_base, cudaStream_t st);

}  // namespace lloid
