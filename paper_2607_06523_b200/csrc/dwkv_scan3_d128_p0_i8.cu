// instance of the fused decode kernel: head dim 128, FULL mode (4 < G <= 8), 8-bit coefficient planes
#include "dwkv_scan3_kernel.cuh"
namespace dwkv {
bool launch_scan3_d128_p0_i8(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err) {
  return s3::launch_by_rank_i8<128, false>(p, n_sms, s, err);
}
}  // namespace dwkv
