"""Pins for the Kalman recursion (13) and the Riccati scan (16)(17) of oracle/ltv_oracle.py
against things OTHER than the oracle: brute-force Gaussian conditioning of the stacked linear-Gaussian model (the
definition of what the recursion computes), the information form of the measurement update, scipy's DARE solver for
the fixed point, the Lyapunov sum through Phi for C = 0, a scalar case, Joseph form + gain optimality, and the
scan = recursion / associativity invariants.  A dropped term, a wrong sign or a transposed operand in (13) or (16)
fails at least one of them."""
import numpy as np
import pytest
import scipy.linalg

from oracle import ltv_oracle as O
from workloads import dense_random, observation_model


def _inputs(T, n, p, seed, kind="dense", scale=0.5):
    W = dense_random(1, T, n, 1, seed, scale)
    M = observation_model(1, T, n, p, seed + 1, kind)
    return [a[0].astype(np.float64) for a in (W.A, M["C"], M["e"], M["f"], M["Pi0"])]


def _close(a, b, tol=1e-10):
    assert a.shape == b.shape
    assert np.max(np.abs(a - b)) <= tol * max(np.max(np.abs(b)), 1e-300), np.max(np.abs(a - b)) / np.max(np.abs(b))


def _joint(A, C, e, f, Pi0):
    """Covariances of the stacked model x_{k+1} = A_k x_k + E_k w_k, y_k = C_k x_k + F_k v_k, x_0 ~ N(0, Pi_0) with
    unit-covariance w, v: returns Sxx [(T+1)n, (T+1)n], Sxy [(T+1)n, Tp], Syy [Tp, Tp], built from the explicit map
    (x_0, w_0 .. w_{T-1}) -> (x_0 .. x_T), not from any recursion on covariances."""
    T, n, _ = A.shape
    p = C.shape[1]
    M = np.zeros(((T + 1) * n, (T + 1) * n))   # x = M xi, xi = (x_0, w_0, .., w_{T-1})
    M[:n, :n] = np.eye(n)
    for k in range(T):
        M[(k + 1) * n:(k + 2) * n] = A[k] @ M[k * n:(k + 1) * n]
        M[(k + 1) * n:(k + 2) * n, (k + 1) * n:(k + 2) * n] += np.diag(e[k])
    Sxi = np.eye((T + 1) * n)
    Sxi[:n, :n] = Pi0
    Sxx = M @ Sxi @ M.T
    H = np.zeros((T * p, (T + 1) * n))
    for k in range(T):
        H[k * p:(k + 1) * p, k * n:(k + 1) * n] = C[k]
    Syy = H @ Sxx @ H.T + np.diag(np.concatenate([f[k] ** 2 for k in range(T)]))
    return Sxx, Sxx @ H.T, Syy


@pytest.mark.parametrize("kind", ["dense", "track"])
def test_kalman_is_gaussian_conditioning(kind):
    """Pi_j = Cov(x_j | y_0 .. y_{j-1}) and -L_{j+1}^T = coefficient of y_j in E[x_{j+1} | y_0 .. y_j]."""
    T, n, p = 5, 6, 2
    A, C, e, f, Pi0 = _inputs(T, n, p, 3, kind)
    Pi, Lt = O.kalman_recursion_item(A, C, e, f, Pi0)
    Sxx, Sxy, Syy = _joint(A, C, e, f, Pi0)
    for j in range(T + 1):
        xs = slice(j * n, (j + 1) * n)
        cond = Sxx[xs, xs] - (Sxy[xs, :j * p] @ np.linalg.solve(Syy[:j * p, :j * p], Sxy[xs, :j * p].T) if j else 0.0)
        _close(Pi[j], cond, 1e-9)
    for j in range(T):
        xs = slice((j + 1) * n, (j + 2) * n)
        W = np.linalg.solve(Syy[:(j + 1) * p, :(j + 1) * p], Sxy[xs, :(j + 1) * p].T).T   # regression of x_{j+1} on y_{<=j}
        _close(-Lt[j], W[:, j * p:], 1e-8)


def test_kalman_information_form():
    """Measurement update in information form (textbook): Pi+ = (Pi^-1 + C^T R^-1 C)^-1, Pi' = A Pi+ A^T + E E^T."""
    T, n, p = 6, 7, 3
    A, C, e, f, Pi0 = _inputs(T, n, p, 5)
    Pi, Lt = O.kalman_recursion_item(A, C, e, f, Pi0)
    for j in range(T):
        post = np.linalg.inv(np.linalg.inv(Pi[j]) + C[j].T @ np.diag(1.0 / f[j] ** 2) @ C[j])
        _close(Pi[j + 1], A[j] @ post @ A[j].T + np.diag(e[j] ** 2), 1e-9)
        _close(Lt[j], -A[j] @ post @ C[j].T @ np.diag(1.0 / f[j] ** 2), 1e-8)   # K = Pi+ C^T R^-1


def test_kalman_scalar():
    a, c, e, f = 0.9, 2.0, 0.3, 0.5
    T = 8
    Pi, Lt = O.kalman_recursion_item(np.full((T, 1, 1), a), np.full((T, 1, 1), c), np.full((T, 1), e),
                                     np.full((T, 1), f), np.array([[2.0]]))
    pj = 2.0
    for j in range(T):
        post = 1.0 / (1.0 / pj + c * c / (f * f))   # posterior precision = prior precision + c^2 / f^2
        assert abs(Lt[j, 0, 0] + a * post * c / (f * f)) < 1e-13
        pj = a * a * post + e * e
        assert abs(Pi[j + 1, 0, 0] - pj) < 1e-13


def test_kalman_no_observation_is_lyapunov_sum_through_phi():
    """C = 0: L = 0 and Pi_t = Phi(t,0) Pi_0 Phi(t,0)^T + sum_s Phi(t,s+1) E_s E_s^T Phi(t,s+1)^T with Phi(t,t) = I:
    ties the recursion to the system-response oracle (pinned in test_oracle_pins.py)."""
    T, n, p = 6, 5, 2
    A, C, e, f, Pi0 = _inputs(T, n, p, 7)
    Pi, Lt = O.kalman_recursion_item(A, 0.0 * C, e, f, Pi0)
    assert np.all(Lt == 0.0)
    Phi = O.system_response_item(np.concatenate([A, A[:1]]))   # T+1 nodes: blocks (t,s), 0 <= s < t <= T
    blk = lambda t, s: np.eye(n) if t == s else Phi[O.packed_index(t, s)]
    for t in range(T + 1):
        ref = blk(t, 0) @ Pi0 @ blk(t, 0).T
        for s in range(t):
            ref = ref + blk(t, s + 1) @ np.diag(e[s] ** 2) @ blk(t, s + 1).T
        _close(Pi[t], ref)


def test_kalman_fixed_point_is_scipy_dare():
    n, p, T = 5, 2, 400
    A, C, e, f, Pi0 = _inputs(1, n, p, 11, scale=0.8)
    rep = lambda a: np.broadcast_to(a[0], (T,) + a.shape[1:])
    Pi, Lt = O.kalman_recursion_item(rep(A), rep(C), rep(e), rep(f), Pi0)
    X = scipy.linalg.solve_discrete_are(A[0].T, C[0].T, np.diag(e[0] ** 2), np.diag(f[0] ** 2))
    _close(Pi[-1], X, 1e-8)
    Kss = A[0] @ X @ C[0].T @ np.linalg.inv(np.diag(f[0] ** 2) + C[0] @ X @ C[0].T)
    _close(-Lt[-1], Kss, 1e-7)


def test_kalman_joseph_form_and_gain_optimality():
    """With Abar = A + L^T C the covariance obeys the Joseph form for ANY gain; the Kalman gain minimises it."""
    T, n, p = 4, 6, 3
    A, C, e, f, Pi0 = _inputs(T, n, p, 13)
    Pi, Lt = O.kalman_recursion_item(A, C, e, f, Pi0)
    rng = np.random.default_rng(0)

    def joseph(j, G):
        Ab = A[j] + G @ C[j]
        return Ab @ Pi[j] @ Ab.T + np.diag(e[j] ** 2) + G @ np.diag(f[j] ** 2) @ G.T

    for j in range(T):
        _close(Pi[j + 1], joseph(j, Lt[j]), 1e-9)
        _close(Pi[j + 1], A[j] @ Pi[j] @ (A[j] + Lt[j] @ C[j]).T + np.diag(e[j] ** 2), 1e-9)
        for _ in range(3):
            d = 1e-2 * rng.normal(size=Lt[j].shape) * np.max(np.abs(Lt[j]))
            gap = joseph(j, Lt[j] + d) - Pi[j + 1]
            assert np.min(np.linalg.eigvalsh(0.5 * (gap + gap.T))) >= -1e-12 * np.max(np.abs(Pi[j + 1]))
            assert np.trace(gap) > 0.0
        assert np.allclose(Pi[j + 1], Pi[j + 1].T, rtol=0, atol=1e-12 * np.max(np.abs(Pi[j + 1])))
        assert np.min(np.linalg.eigvalsh(0.5 * (Pi[j + 1] + Pi[j + 1].T))) > 0.0


@pytest.mark.parametrize("kind", ["dense", "track"])
def test_riccati_scan_equals_recursion(kind):
    T, n, p = 9, 8, 3
    A, C, e, f, Pi0 = _inputs(T, n, p, 17, kind)
    Pi, _ = O.kalman_recursion_item(A, C, e, f, Pi0)
    _close(O.riccati_scan_item(A, C, e, f, Pi0), Pi, 1e-9)


def test_riccati_combine_is_associative_and_tree_fold_matches():
    """(x (x) y) (x) z = x (x) (y (x) z) on general elements, and a balanced-tree fold of e_{T-1} .. e_0, e_init gives
    Pi_T: the property the parallel scan of PAPER.md:177 rests on."""
    T, n, p = 8, 6, 2
    A, C, e, f, Pi0 = _inputs(T, n, p, 19)
    elems = [(A[i].T, C[i].T @ np.diag(1.0 / f[i] ** 2) @ C[i], np.diag(e[i] ** 2)) for i in range(T)]
    x, y, z = elems[2], elems[1], elems[0]
    lhs = O.riccati_combine(O.riccati_combine(x, y), z)
    rhs = O.riccati_combine(x, O.riccati_combine(y, z))
    for a, b in zip(lhs, rhs):
        _close(a, b, 1e-9)
    seq = [e_ for e_ in reversed(elems)] + [(np.zeros((n, n)), np.zeros((n, n)), Pi0)]   # newest first
    while len(seq) > 1:
        seq = [O.riccati_combine(seq[i], seq[i + 1]) if i + 1 < len(seq) else seq[i] for i in range(0, len(seq), 2)]
    Pi, _ = O.kalman_recursion_item(A, C, e, f, Pi0)
    _close(seq[0][2], Pi[T], 1e-9)
    assert np.max(np.abs(seq[0][0])) == 0.0 and np.max(np.abs(seq[0][1])) == 0.0


def test_kalman_gains_close_the_observer_loop():
    """Lt[j] is the array observer_response consumes: with it, Pi_{j+1} = PhiX(j+1,j) Pi_j A_j^T + E E^T where
    PhiX(j+1,j) = A_j + Lt[j] C_j is the sub-diagonal block of eq.(14)."""
    T, n, p = 5, 6, 2
    A, C, e, f, Pi0 = _inputs(T, n, p, 23)
    Pi, Lt = O.kalman_recursion_item(A, C, e, f, Pi0)
    PhiX, _ = O.observer_response_item(A, Lt, C)
    for j in range(T - 1):
        _close(Pi[j + 1], PhiX[O.packed_index(j + 1, j)] @ Pi[j] @ A[j].T + np.diag(e[j] ** 2), 1e-9)


def test_kalman_hand_example_exact():
    """One and two steps by hand (all values dyadic or small rationals).  A = [[1,1],[0,1]], C = [1 0], E = diag(0,1),
    F = 1, Pi_0 = I:
      step 0: S = 1 + 1 = 2; C Pi A^T = [1 0]; L_1 = -[1/2 0]; A Pi C^T = [1 0]^T
              Pi_1 = diag(0,1) + A A^T + [1 0]^T L_1 = [[0,0],[0,1]] + [[2,1],[1,1]] + [[-1/2,0],[0,0]] = [[3/2,1],[1,2]]
      step 1: S = 1 + 3/2 = 5/2; C Pi_1 A^T = [3/2 1] A^T = [5/2 1]; L_2 = -[1 2/5];
              A Pi_1 A^T = [[11/2,3],[3,2]]; A Pi_1 C^T = [5/2 1]^T; [5/2 1]^T L_2 = -[[5/2,1],[1,2/5]]
              Pi_2 = [[0,0],[0,1]] + [[11/2,3],[3,2]] - [[5/2,1],[1,2/5]] = [[3,2],[2,13/5]]"""
    A = np.broadcast_to(np.array([[1.0, 1.0], [0.0, 1.0]]), (2, 2, 2))
    C = np.broadcast_to(np.array([[1.0, 0.0]]), (2, 1, 2))
    e = np.broadcast_to(np.array([0.0, 1.0]), (2, 2))
    f = np.ones((2, 1))
    Pi, Lt = O.kalman_recursion_item(A, C, e, f, np.eye(2))
    assert np.array_equal(Pi[1], np.array([[1.5, 1.0], [1.0, 2.0]]))
    assert np.array_equal(Lt[0], np.array([[-0.5], [0.0]]))
    np.testing.assert_allclose(Lt[1], np.array([[-1.0], [-0.4]]), rtol=1e-15)
    np.testing.assert_allclose(Pi[2], np.array([[3.0, 2.0], [2.0, 2.6]]), rtol=1e-15)
    np.testing.assert_allclose(O.riccati_scan_item(A, C, e, f, np.eye(2))[2], np.array([[3.0, 2.0], [2.0, 2.6]]), rtol=1e-14)
