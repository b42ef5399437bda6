// tcgen05 path -- placeholder until the tensor-core kernels land (next commit).
#include "lloid_internal.h"
namespace lloid {
struct TcPlan { int dummy; };
int tc_time_splits(int B) { return (B + 127) / 128; }
int tc_plan_create(TcPlan **out, const std::vector<CorrClass> &, const CorrClass *, const std::vector<ReconBank> &,
                   const ReconBank *, int, int, int) {
  *out = nullptr;
  set_error("stream_create: the tcgen05 path is not built in this revision; use LLOID_PREC_FP32_FFMA");
  return LLOID_ECUDA;
}
void tc_plan_destroy(TcPlan *p) { delete p; }
cudaError_t tc_launch_corr(TcPlan *, const long long *, cudaStream_t) { return cudaErrorNotSupported; }
cudaError_t tc_launch_recon(TcPlan *, PeakPartial *, int, float *, int, cudaStream_t) { return cudaErrorNotSupported; }
}  // namespace lloid
