// instance of the fused decode kernel: head dim 64, PAIR mode (G <= 4)
#include "dwkv_scan3_kernel.cuh"
namespace dwkv {
bool launch_scan3_d64_p1(const Scan3Params& p, int n_sms, cudaStream_t s, cudaError_t* err) {
  return s3::launch_by_rank<64, true>(p, n_sms, s, err);
}
}  // namespace dwkv
