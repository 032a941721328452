// dwkv_controller.cu -- probe-driven threshold controller of PAPER.md:72 (reading A28).
// Host-only state machine, one (delta_m, quiet_m) per depth window; thresholds live in logit space (reading A26), tau_m = base + delta_m.
//   one probe interval (dwkv_controller_step): e_m = max of the reported Eq. (3) errors of window m
//     e_m > tol_m  ->  delta_m = max(delta_m - step_down, delta_min), quiet_m = 0                       "the router lowers tau_m"
//     else quiet_m += 1; quiet_m == patience -> delta_m = min(delta_m + step_up, delta_max), quiet_m = 0   "below tolerance for several
//                                                                                                        probe intervals, tau_m is increased"
//   fp32, one rounding per operation. A token's (tier, flag) is shared by all layers and heads (reading A4), so the thresholds for new
//   tokens are base + min_m delta_m (dwkv_controller_thresholds). Stored tokens are never re-tiered.
#include <cmath>
#include <limits>
#include <new>
#include <vector>

#include "../../include/dwkv.h"

struct dwkv_controller {
  dwkv_controller_config cfg;
  std::vector<float> tol, delta, emax;
  std::vector<int32_t> quiet;
  std::vector<uint8_t> seen;
};

extern "C" int dwkv_controller_create(const dwkv_controller_config* cfg, dwkv_controller** out) {
  if (!cfg || !out) return DWKV_E_INVALID;
  *out = nullptr;
  if (cfg->n_windows <= 0 || cfg->patience <= 0) return DWKV_E_INVALID;
  if (!(cfg->step_down >= 0.f) || !(cfg->step_up >= 0.f) || !(cfg->delta_min <= 0.f) || !(cfg->delta_max >= 0.f)) return DWKV_E_INVALID;
  if (!(cfg->tol_default >= 0.f)) return DWKV_E_INVALID;
  dwkv_controller* c = new (std::nothrow) dwkv_controller();
  if (!c) return DWKV_E_INVALID;
  c->cfg = *cfg;
  c->tol.assign(cfg->n_windows, cfg->tol_default);
  if (cfg->tol)
    for (int m = 0; m < cfg->n_windows; ++m) {
      if (!(cfg->tol[m] >= 0.f)) { delete c; return DWKV_E_INVALID; }
      c->tol[m] = cfg->tol[m];
    }
  c->cfg.tol = nullptr;       // the caller's array is copied, not kept
  c->delta.assign(cfg->n_windows, 0.f);
  c->quiet.assign(cfg->n_windows, 0);
  c->emax.assign(cfg->n_windows, 0.f);
  c->seen.assign(cfg->n_windows, 0);
  *out = c;
  return DWKV_OK;
}

extern "C" void dwkv_controller_destroy(dwkv_controller* c) { delete c; }

extern "C" int dwkv_controller_step(dwkv_controller* c, int32_t n_probes, const int32_t* window, const float* e) {
  if (!c || n_probes < 0 || (n_probes > 0 && (!window || !e))) return DWKV_E_INVALID;
  for (int i = 0; i < n_probes; ++i)
    if (window[i] < 0 || window[i] >= c->cfg.n_windows || std::isnan(e[i])) return DWKV_E_INVALID;     // state untouched on error
  for (int m = 0; m < c->cfg.n_windows; ++m) c->seen[m] = 0;
  for (int i = 0; i < n_probes; ++i) {
    const int m = window[i];
    if (!c->seen[m] || e[i] > c->emax[m]) c->emax[m] = e[i];
    c->seen[m] = 1;
  }
  for (int m = 0; m < c->cfg.n_windows; ++m) {
    if (!c->seen[m]) continue;
    if (c->emax[m] > c->tol[m]) {
      const volatile float d = c->delta[m] - c->cfg.step_down;        // one fp32 rounding (no wider intermediate)
      c->delta[m] = d > c->cfg.delta_min ? d : c->cfg.delta_min;
      c->quiet[m] = 0;
    } else if (++c->quiet[m] == c->cfg.patience) {
      const volatile float d = c->delta[m] + c->cfg.step_up;
      c->delta[m] = d < c->cfg.delta_max ? d : c->cfg.delta_max;
      c->quiet[m] = 0;
    }
  }
  return DWKV_OK;
}

extern "C" int dwkv_controller_state(const dwkv_controller* c, float* delta, int32_t* quiet) {
  if (!c) return DWKV_E_INVALID;
  for (int m = 0; m < c->cfg.n_windows; ++m) {
    if (delta) delta[m] = c->delta[m];
    if (quiet) quiet[m] = c->quiet[m];
  }
  return DWKV_OK;
}

extern "C" int dwkv_controller_thresholds(const dwkv_controller* c, int32_t n_tiers, const float* base_tau_logit, float base_flag_logit,
                                          float* tau_logit, float* tau_flag_logit) {
  if (!c || n_tiers < 1 || n_tiers > DWKV_MAX_TIERS || !tau_flag_logit || (n_tiers > 1 && (!base_tau_logit || !tau_logit))) return DWKV_E_INVALID;
  float dmin = c->delta[0];
  for (int m = 1; m < c->cfg.n_windows; ++m) dmin = c->delta[m] < dmin ? c->delta[m] : dmin;
  for (int k = 0; k + 1 < n_tiers; ++k) { const volatile float t = base_tau_logit[k] + dmin; tau_logit[k] = t; }
  const volatile float tf = base_flag_logit + dmin;
  *tau_flag_logit = tf;
  return DWKV_OK;
}
