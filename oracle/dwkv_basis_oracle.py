"""CPU oracle for the basis construction of DepthWeave-KV (prefill side).  TEST INFRASTRUCTURE ONLY.

Only `tests/` may import this module; the product never does and shares no code with it.

PAPER.md:56: "The shared bases are initialized online from the first compressed prefix block. For each depth window, we compute
a small randomized low-rank sketch of the cached keys and values after prefill ... The update is performed independently per
head and separately for keys and values". The paper gives no formula; reading A24 fixes one (the randomized range
finder of Halko, Martinsson and Tropp applied to the row space, without power iteration):

  for window m, kv head h, Z in {K, V}:
      X    = rows  x[l,h,t,:] / gate[l,h,:]   for l in window m (w layers), t < n          ((w*n) x d, gate-normalised: reading A13)
      S    = Omega^T X = sum_{l in window} Omega_l^T X_l                                     (k x d sketch, Omega_l is k x n ... see below)
      S    = U diag(sigma) W^T   (singular value decomposition, sigma descending)
      B[m,h] = first r rows of W^T, each with the sign that makes its largest-magnitude entry positive, rounded to bf16

  Omega is an INPUT (the random numbers the method draws): omega[j, i, t] for layer j of the window (the same for every window,
  head and Z), sketch row i < k, token t < n.  S[i,:] = sum_j sum_t omega[j,i,t] * x[m*w+j, h, t, :] / gate[m*w+j, h, :].

Everything is fp64 here (inputs are bf16 values held exactly); the SVD is numpy's (LAPACK gesdd). The rows are orthonormal and
ordered by the energy the sketch sees along them, which is what "leading r_t coefficients" (north_star) needs.
Pins: tests/test_basis_oracle_pins.py.
"""
from __future__ import annotations

import numpy as np


def sketch(x, gate, omega, w: int) -> np.ndarray:
    """S[m, h] = sum over the w layers of window m and the n tokens of omega[j, :, t] (x) x[l, h, t, :] / gate[l, h, :].

    x: [n, L, H, d]; gate: [L, H, d]; omega: [w, k, n]. Returns [M, H, k, d] (fp64)."""
    x = np.asarray(x, np.float64); gate = np.asarray(gate, np.float64); omega = np.asarray(omega, np.float64)
    n, L, H, d = x.shape
    k = omega.shape[1]
    M = L // w
    S = np.zeros((M, H, k, d))
    for m in range(M):
        for j in range(w):
            l = m * w + j
            for h in range(H):
                S[m, h] += omega[j] @ (x[:, l, h, :] / gate[l, h][None, :])
    return S


def basis_from_sketch(S, r: int) -> np.ndarray:
    """First r right singular vectors of each sketch S[m, h] (k x d), sign-normalised; fp64, not yet rounded. [M, H, r, d]."""
    M, H, k, d = S.shape
    B = np.zeros((M, H, r, d))
    for m in range(M):
        for h in range(H):
            _, _, Wt = np.linalg.svd(S[m, h], full_matrices=False)      # singular values descending
            rows = Wt[:r].copy()
            for i in range(r):
                j = int(np.argmax(np.abs(rows[i])))
                if rows[i, j] < 0:
                    rows[i] = -rows[i]
            B[m, h] = rows
    return B


def build_basis(x, gate, omega, w: int, r: int) -> np.ndarray:
    """The whole construction for one Z: sketch, SVD, first r rows (fp64, unrounded). Round with the decode oracle's round_to_bf16."""
    return basis_from_sketch(sketch(x, gate, omega, w), r)
