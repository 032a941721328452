"""CPU oracle for the token-conditional router of DepthWeave-KV.  TEST INFRASTRUCTURE ONLY (only `tests/` may import it).

PAPER.md:58-63, Eq. (2):  rho = rho_min + (rho_max - rho_min) * 1[ sigma(u^T phi) > tau_m ],  "In practice, we use three rank levels
rather than a binary decision", tau_m "an adaptive threshold chosen to satisfy the current memory budget". DESIGN.md reading A26:
  * the routed quantity is BASELINE.json's (tier, residual flag) pair of a token (readings A3-A5), shared by all layers and heads;
  * several levels = several thresholds tau_1 <= tau_2 <= ... on the same score; one more threshold for the residual flag;
  * sigma is monotone, so sigma(z) > tau <=> z > logit(tau): thresholds live in logit space and no exponential is evaluated;
  * z = ((u0*phi0 + u1*phi1) + u2*phi2) + u3*phi3 in float32, one rounding per operation (the precision the decision is taken in);
  * budget: the fraction of tokens per tier / flagged is given; the threshold is the order statistic that leaves exactly
    ceil(n * fraction above) tokens strictly above it.
Written as plain loops over tokens; numpy only for float32 scalars and the sort."""
from __future__ import annotations

import math

import numpy as np


def logits(phi, u) -> np.ndarray:
    phi = np.asarray(phi, np.float32); u = np.asarray(u, np.float32)
    z = np.zeros(phi.shape[0], np.float32)
    for t in range(phi.shape[0]):
        p0 = np.float32(u[0] * phi[t, 0]); p1 = np.float32(u[1] * phi[t, 1])
        p2 = np.float32(u[2] * phi[t, 2]); p3 = np.float32(u[3] * phi[t, 3])
        z[t] = np.float32(np.float32(np.float32(p0 + p1) + p2) + p3)
    return z


def route(phi, u, tau_logit, tau_flag_logit):
    z = logits(phi, u)
    tau = [np.float32(x) for x in tau_logit]
    tier = np.zeros(len(z), np.uint8); flag = np.zeros(len(z), np.uint8)
    for t in range(len(z)):
        k = 0
        for x in tau:
            if z[t] > x:
                k += 1
        tier[t] = k
        flag[t] = 1 if z[t] > np.float32(tau_flag_logit) else 0
    return tier, flag


def _threshold(z_sorted, m: int) -> np.float32:
    n = len(z_sorted)
    if m <= 0:
        return np.float32(np.inf)
    if m >= n:
        return np.float32(-np.inf)
    return z_sorted[n - m - 1]


def thresholds(phi, u, tier_frac, flag_frac):
    z = np.sort(logits(phi, u))
    n = len(z)
    frac = [float(np.float32(f)) for f in tier_frac]
    tau = []
    for k in range(1, len(frac)):
        above = 0.0
        for j in range(k, len(frac)):
            above += frac[j]
        tau.append(_threshold(z, int(math.ceil(n * above))))
    return np.asarray(tau, np.float32), _threshold(z, int(math.ceil(n * float(np.float32(flag_frac)))))
