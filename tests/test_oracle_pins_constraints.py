"""Pins for oracle.constraint_tightening (eq.(12d)) against things other than
itself: identity constraint rows reduce it to the (separately pinned) row-wise two-norm tube, A = I and rotations give
closed forms, brute-force scalar loops, and the worst-case disturbance: for ||d_j||_2 <= 1 the constraint value
c^T sum_j Phi(k,j) E_j d_j never exceeds sigma_k[i] and reaches it for the aligned disturbance."""
import numpy as np

from oracle import ltv_oracle as O
from workloads import dense_random


def _inputs(T, n, nc, seed):
    W = dense_random(1, T, n, 1, seed, 0.6)
    rng = np.random.default_rng(seed + 99)
    Hc = rng.normal(0.0, 1.0, (T, nc, n)).astype(np.float32)
    return W.A[0].astype(np.float64), W.w[0].astype(np.float64), Hc.astype(np.float64)


def test_identity_rows_give_the_row2norm_tube():
    A, w, _ = _inputs(6, 5, 5, 1)
    Hc = np.broadcast_to(np.eye(5), (6, 5, 5))
    np.testing.assert_allclose(O.constraint_tightening_item(A, w, Hc), O.tube_row2norm_item(A, w), rtol=1e-13, atol=0)


def test_identity_dynamics_closed_form():
    T, n, nc = 5, 4, 3
    _, w, Hc = _inputs(T, n, nc, 2)
    sig = O.constraint_tightening_item(np.broadcast_to(np.eye(n), (T, n, n)), w, Hc)
    assert np.all(sig[0] == 0.0)
    for k in range(1, T):
        ref = sum(np.linalg.norm(Hc[k] * w[j][None, :], axis=1) for j in range(k))
        np.testing.assert_allclose(sig[k], ref, rtol=1e-13)


def test_rotation_closed_form():
    """A_t = R(theta_t), w_j = omega_j (1,1): ||c^T R E|| = omega ||c|| whatever the angle."""
    th = np.array([0.3, -1.1, 0.7, 2.0, 0.4])
    R = np.stack([[[np.cos(t), -np.sin(t)], [np.sin(t), np.cos(t)]] for t in th])
    om = np.array([0.5, 2.0, 1.5, 0.25, 3.0])
    Hc = np.random.default_rng(0).normal(size=(5, 2, 2))
    sig = O.constraint_tightening_item(R, om[:, None] * np.ones((5, 2)), Hc)
    for k in range(1, 5):
        np.testing.assert_allclose(sig[k], np.linalg.norm(Hc[k], axis=1) * om[:k].sum(), rtol=1e-13)


def test_brute_force_scalar_loops():
    T, n, nc = 4, 3, 2
    A, w, Hc = _inputs(T, n, nc, 3)
    sig = O.constraint_tightening_item(A, w, Hc)
    for k in range(1, T):
        for i in range(nc):
            tot = 0.0
            for j in range(k):
                P = np.eye(n)
                for t in range(j, k):          # Phi(k,j) = A_{k-1} ... A_j, explicit left products
                    P = A[t] @ P
                sq = 0.0
                for col in range(n):
                    v = 0.0
                    for row in range(n):
                        v += Hc[k, i, row] * P[row, col]
                    sq += (v * w[j, col]) ** 2
                tot += sq ** 0.5
            assert abs(sig[k, i] - tot) <= 1e-12 * max(1.0, abs(tot))


def test_worst_case_disturbance_containment_and_tightness():
    T, n, nc = 6, 5, 3
    A, w, Hc = _inputs(T, n, nc, 4)
    sig = O.constraint_tightening_item(A, w, Hc)
    Phi = O.system_response_item(A)
    rng = np.random.default_rng(5)
    for k in range(1, T):
        for i in range(nc):
            rows = [Hc[k, i] @ Phi[O.packed_index(k, j)] @ np.diag(w[j]) for j in range(k)]
            worst = sum(r @ (r / np.linalg.norm(r)) for r in rows)          # aligned unit disturbances
            assert abs(worst - sig[k, i]) <= 1e-12 * sig[k, i]
            for _ in range(5):
                d = rng.normal(size=(k, n))
                d /= np.maximum(1.0, np.linalg.norm(d, axis=1, keepdims=True))
                val = sum(r @ d[j] for j, r in enumerate(rows))
                assert abs(val) <= sig[k, i] * (1 + 1e-12)


def test_homogeneity_and_batch_wrapper():
    T, n, nc = 5, 4, 2
    A, w, Hc = _inputs(T, n, nc, 6)
    sig = O.constraint_tightening_item(A, w, Hc)
    np.testing.assert_allclose(O.constraint_tightening_item(A, 2.0 * w, -3.0 * Hc), 6.0 * sig, rtol=1e-13)
    np.testing.assert_array_equal(O.constraint_tightening(A[None], w[None], Hc[None])[0], sig)
