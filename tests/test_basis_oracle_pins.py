"""Pins of the basis-construction oracle (oracle/dwkv_basis_oracle.py, reading A24). CPU only.

The paper prints no number for this step, so the pins are what the mathematics fixes: exact recovery of a planted subspace,
gate normalisation, the index structure of the sketch on one-hot inputs, energy ordering, and agreement with a different
library route (symmetric eigendecomposition instead of the SVD)."""
import numpy as np

from oracle import dwkv_basis_oracle as bo


def _orthonormal_rows(rng, r, d):
    q, _ = np.linalg.qr(rng.standard_normal((d, r)))
    return q.T


def _projector(B):
    return B.T @ B


def test_planted_subspace_is_recovered_exactly():
    rng = np.random.default_rng(1)
    n, L, w, H, d, r, k = 96, 4, 2, 2, 32, 6, 16
    B0 = np.stack([[_orthonormal_rows(rng, r, d) for _ in range(H)] for _ in range(L // w)])        # [M, H, r, d]
    x = np.zeros((n, L, H, d))
    for l in range(L):
        for h in range(H):
            x[:, l, h] = rng.standard_normal((n, r)) @ B0[l // w, h]
    B = bo.build_basis(x, np.ones((L, H, d)), rng.standard_normal((w, k, n)), w, r)
    for m in range(L // w):
        for h in range(H):
            assert np.allclose(_projector(B[m, h]), _projector(B0[m, h]), atol=1e-10)
            assert np.allclose(B[m, h] @ B[m, h].T, np.eye(r), atol=1e-12)


def test_gate_divides_the_rows():
    """x = (c . B0) * gate must give the subspace of B0 (projection happens in gate-normalised space, reading A13)."""
    rng = np.random.default_rng(2)
    n, L, w, H, d, r, k = 64, 2, 2, 1, 32, 4, 16
    B0 = _orthonormal_rows(rng, r, d)
    gate = rng.uniform(0.5, 1.5, (L, H, d))
    x = np.zeros((n, L, H, d))
    for l in range(L):
        x[:, l, 0] = (rng.standard_normal((n, r)) @ B0) * gate[l, 0]
    B = bo.build_basis(x, gate, rng.standard_normal((w, k, n)), w, r)
    assert np.allclose(_projector(B[0, 0]), _projector(B0), atol=1e-10)
    wrong = bo.build_basis(x, 1.0 / gate, rng.standard_normal((w, k, n)), w, r)           # multiplying instead: a different subspace
    assert not np.allclose(_projector(wrong[0, 0]), _projector(B0), atol=1e-3)


def test_sketch_indices_on_one_hot_inputs():
    rng = np.random.default_rng(3)
    n, L, w, H, d, k = 10, 4, 2, 3, 16, 16
    x = rng.standard_normal((n, L, H, d))
    gate = rng.uniform(0.5, 1.5, (L, H, d))
    omega = np.zeros((w, k, n))
    omega[1, 5, 7] = 2.0                         # sketch row 5 = 2 * (token 7 of the SECOND layer of every window)
    S = bo.sketch(x, gate, omega, w)
    assert S.shape == (L // w, H, k, d)
    for m in range(L // w):
        for h in range(H):
            want = np.zeros((k, d)); want[5] = 2.0 * x[7, m * w + 1, h] / gate[m * w + 1, h]
            assert np.allclose(S[m, h], want, atol=1e-14)


def test_window_sums_its_layers_only():
    rng = np.random.default_rng(4)
    n, L, w, H, d, k = 12, 4, 2, 1, 16, 16
    x = np.zeros((n, L, H, d)); x[:, 1] = rng.standard_normal((n, H, d))          # only layer 1 (window 0) holds data
    omega = rng.standard_normal((w, k, n))
    S = bo.sketch(x, np.ones((L, H, d)), omega, w)
    assert np.allclose(S[1], 0.0) and np.allclose(S[0, 0], omega[1] @ x[:, 1, 0])


def test_rows_are_ordered_by_energy_and_signed():
    rng = np.random.default_rng(5)
    n, L, w, H, d, r, k = 256, 2, 2, 1, 32, 8, 16
    u = np.zeros(d); u[3] = 1.0
    x = rng.standard_normal((n, L, H, d)) * 0.1
    x[:, :, 0, :] += 10.0 * rng.standard_normal((n, L, 1)) * u                  # one dominant direction
    omega = rng.standard_normal((w, k, n))
    S = bo.sketch(x, np.ones((L, H, d)), omega, w)
    B = bo.basis_from_sketch(S, r)[0, 0]
    energy = np.linalg.norm(S[0, 0] @ B.T, axis=0)
    assert np.all(np.diff(energy) <= 1e-9)
    assert abs(B[0] @ u) > 0.999
    for i in range(r):
        assert B[i, np.argmax(np.abs(B[i]))] > 0


def test_against_symmetric_eigendecomposition():
    """Different library route: the leading eigenvectors of S^T S span the same subspaces as the leading right singular vectors."""
    rng = np.random.default_rng(6)
    n, L, w, H, d, r, k = 128, 2, 2, 2, 32, 8, 16
    x = rng.standard_normal((n, L, H, d)) * (1.0 / np.sqrt(1.0 + np.arange(d)))[None, None, None, :]
    S = bo.sketch(x, np.ones((L, H, d)), rng.standard_normal((w, k, n)), w)
    B = bo.basis_from_sketch(S, r)
    for h in range(H):
        lam, V = np.linalg.eigh(S[0, h].T @ S[0, h])
        lead = V[:, np.argsort(lam)[::-1][:r]].T
        for rr in (1, 4, 8):
            assert np.allclose(_projector(B[0, h][:rr]), _projector(lead[:rr]), atol=1e-8)
