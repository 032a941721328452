"""CPU oracle for the probe-driven controller and the router's attention features.  TEST INFRASTRUCTURE ONLY (only `tests/` may
import it; the product never does and shares no code with it).

PAPER.md:58 "the router computes a score from four online features: accumulated attention mass, maximum attention spike, ..."
PAPER.md:72 "If e_{l,h} exceeds a window-specific tolerance, the router lowers tau_m and assigns more tokens in that window to
higher residual rank. If the error remains below tolerance for several probe intervals, tau_m is increased and residual storage
is reduced."  The paper gives neither the step sizes nor the exact statistics; reading A28 fixes them:

  token statistics of one probed (layer, sequence, query vector):  p[hq, t] = softmax_t(q[hq] . K-hat[t] * scale)   (all T tokens)
      mass[t]  = sum_hq p[hq, t]            -> ACCUMULATED over probe steps      (feature phi_0 of Eq. 2)
      spike[t] = max_hq p[hq, t]            -> running MAXIMUM over probe steps  (feature phi_1)
  controller, one state (delta_m, quiet_m) per depth window m; thresholds live in logit space (reading A26) and tau_m = base + delta_m:
      one probe interval: e_m = max of the probe errors e_{l,h} (Eq. 3) reported for window m (windows without a probe keep their state)
        e_m > tol_m          ->  delta_m = max(delta_m - step_down, delta_min); quiet_m = 0          ("lowers tau_m")
        else quiet_m += 1; quiet_m == patience  ->  delta_m = min(delta_m + step_up, delta_max); quiet_m = 0   ("several probe intervals")
      all arithmetic in float32, one rounding per operation; comparisons strict as written.
  a token's (tier, flag) is shared by all layers and heads (reading A4), so the thresholds the router uses for NEW tokens are
      tau_k = base_k + min_m delta_m        (the most conservative window governs; stored tokens are never re-tiered: their
                                             original vectors no longer exist, promotion is impossible)
"""
from __future__ import annotations

import numpy as np


def attention_probs(q, K, scale: float) -> np.ndarray:
    """p[g, t] = softmax_t(q[g] . K[t] * scale); q [G, d], K [T, d]; float64, max-subtracted."""
    q = np.asarray(q, np.float64); K = np.asarray(K, np.float64)
    p = np.zeros((q.shape[0], K.shape[0]))
    for g in range(q.shape[0]):
        s = (K @ q[g]) * scale
        s = s - np.max(s)
        e = np.exp(s)
        p[g] = e / np.sum(e)
    return p


def token_stats(p):
    """p [H_q, T] (all query heads of a layer) -> (mass [T] = sum over heads, spike [T] = max over heads)."""
    p = np.asarray(p, np.float64)
    return p.sum(axis=0), p.max(axis=0)


class Controller:
    def __init__(self, n_windows, tol, step_down, step_up, patience, delta_min, delta_max):
        f = np.float32
        self.M = int(n_windows)
        self.tol = np.broadcast_to(np.asarray(tol, np.float32), (self.M,)).copy()
        self.step_down, self.step_up = f(step_down), f(step_up)
        self.patience = int(patience)
        self.delta_min, self.delta_max = f(delta_min), f(delta_max)
        self.delta = np.zeros(self.M, np.float32)
        self.quiet = np.zeros(self.M, np.int32)

    def step(self, window, e):
        """One probe interval: parallel lists window[i] (depth-window index) and e[i] (Eq. 3 error of a probed (layer, head))."""
        emax = {}
        for w, x in zip(window, e):
            x = np.float32(x)
            if int(w) not in emax or x > emax[int(w)]:
                emax[int(w)] = x
        for m, x in emax.items():
            if x > self.tol[m]:
                d = np.float32(self.delta[m] - self.step_down)
                self.delta[m] = d if d > self.delta_min else self.delta_min
                self.quiet[m] = 0
            else:
                self.quiet[m] += 1
                if self.quiet[m] == self.patience:
                    d = np.float32(self.delta[m] + self.step_up)
                    self.delta[m] = d if d < self.delta_max else self.delta_max
                    self.quiet[m] = 0

    def thresholds(self, base_tau_logit, base_flag_logit):
        dmin = np.float32(np.min(self.delta))
        tau = np.asarray([np.float32(np.float32(t) + dmin) for t in base_tau_logit], np.float32)
        return tau, np.float32(np.float32(base_flag_logit) + dmin)
