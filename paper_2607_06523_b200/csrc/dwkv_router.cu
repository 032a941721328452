// dwkv_router.cu -- token-conditional router of PAPER.md:58-63 Eq. (2) (reading A26).
// Host-only integer / fp32 logic: the router "operates only on cache metadata" and its output is the host tier / flag
// arrays dwkv_append_compress takes. No device work, no handle, no global state.
//
//   z_t    = ((u0*phi_t0 + u1*phi_t1) + u2*phi_t2) + u3*phi_t3      fp32, one rounding per operation, no FMA contraction
//   tier_t = #{ k : z_t > tau_logit[k] }                             sigma(z) > tau  <=>  z > logit(tau): thresholds in logit space
//   flag_t = z_t > tau_flag_logit
//   thresholds for a memory budget given as the fractions of tokens per tier (low -> high) and the flagged fraction:
//   tau_logit[k-1] = the largest z that is NOT among the ceil(n * sum_{j>=k} frac_j) highest ones (-inf if all are, +inf if none)
#include <algorithm>
#include <cmath>
#include <limits>
#include <vector>

#include "../../include/dwkv.h"

namespace {

#if defined(__GNUC__) && !defined(__clang__)
__attribute__((optimize("fp-contract=off")))
#endif
inline float router_logit(const float* phi, const float* u) {
  const float p0 = u[0] * phi[0], p1 = u[1] * phi[1], p2 = u[2] * phi[2], p3 = u[3] * phi[3];
  const float s01 = p0 + p1;
  const float s012 = s01 + p2;
  return s012 + p3;
}

float threshold_for_count(const std::vector<float>& z_sorted, int64_t m) {   // m tokens shall lie strictly above
  const int64_t n = (int64_t)z_sorted.size();
  if (m <= 0) return std::numeric_limits<float>::infinity();
  if (m >= n) return -std::numeric_limits<float>::infinity();
  return z_sorted[n - m - 1];
}

}  // namespace

extern "C" int dwkv_route_tokens(int64_t n, const float* phi, const float* u, int32_t n_tiers, const float* tau_logit,
                                 float tau_flag_logit, uint8_t* tier, uint8_t* flag) {
  if (n < 0 || n_tiers < 1 || n_tiers > DWKV_MAX_TIERS) return DWKV_E_INVALID;
  if (n == 0) return DWKV_OK;
  if (!phi || !u || !tier || !flag || (n_tiers > 1 && !tau_logit)) return DWKV_E_INVALID;
  for (int k = 0; k + 2 < n_tiers; ++k)
    if (!(tau_logit[k] <= tau_logit[k + 1])) return DWKV_E_INVALID;         // ascending (NaN refused)
  for (int64_t t = 0; t < n; ++t) {
    const float z = router_logit(phi + 4 * t, u);
    int k = 0;
    for (int j = 0; j + 1 < n_tiers; ++j) k += z > tau_logit[j];
    tier[t] = (uint8_t)k;
    flag[t] = (uint8_t)(z > tau_flag_logit);
  }
  return DWKV_OK;
}

extern "C" int dwkv_router_thresholds(int64_t n, const float* phi, const float* u, int32_t n_tiers, const float* tier_frac,
                                      float flag_frac, float* tau_logit, float* tau_flag_logit) {
  if (n <= 0 || n_tiers < 1 || n_tiers > DWKV_MAX_TIERS || !phi || !u || !tier_frac || !tau_flag_logit) return DWKV_E_INVALID;
  if (n_tiers > 1 && !tau_logit) return DWKV_E_INVALID;
  if (!(flag_frac >= 0.f && flag_frac <= 1.f)) return DWKV_E_INVALID;
  for (int k = 0; k < n_tiers; ++k)
    if (!(tier_frac[k] >= 0.f && tier_frac[k] <= 1.f)) return DWKV_E_INVALID;
  std::vector<float> z((size_t)n);
  for (int64_t t = 0; t < n; ++t) z[(size_t)t] = router_logit(phi + 4 * t, u);
  std::sort(z.begin(), z.end());
  for (int k = 1; k < n_tiers; ++k) {
    double above = 0.0;
    for (int j = k; j < n_tiers; ++j) above += (double)tier_frac[j];
    tau_logit[k - 1] = threshold_for_count(z, (int64_t)std::ceil((double)n * above));
  }
  *tau_flag_logit = threshold_for_count(z, (int64_t)std::ceil((double)n * (double)flag_frac));
  return DWKV_OK;
}
