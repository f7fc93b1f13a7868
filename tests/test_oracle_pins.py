"""Pins for oracle/ltv_oracle.py against things OTHER than itself: closed forms, the defining identity
(12c), brute force, a hand-computed example (tests/golden/hand_example.txt), the
tube-containment invariant and the adjoint dot-product identity ((10)).
Each is chosen so that a dropped term, a wrong sign/index or a transposed operand fails at least one."""
import numpy as np
import pytest

from oracle import ltv_oracle as O
from workloads import config, dense_random, generate

RT = 1e-12


def _rand(T, n, m=2, seed=0, scale=0.6):
    W = dense_random(1, T, n, m, seed, scale)
    return [a[0].astype(np.float64) for a in (W.A, W.B, W.c, W.x0, W.u, W.w, W.g)]


def _close(a, b, tol=RT):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    assert a.shape == b.shape
    assert np.max(np.abs(a - b)) <= tol * max(1.0, np.max(np.abs(b)))


# ------------------------------------------------------------------ golden (hand arithmetic)
def test_golden_hand_example(golden_hand):
    G = golden_hand
    Phi, r = O.system_response_tube_item(G["A"], G["w"])
    assert np.array_equal(Phi, G["Phi"])
    assert np.array_equal(r, G["r"])
    assert np.array_equal(O.system_response_item(G["A"]), G["Phi"])
    assert np.array_equal(O.tube_item(G["A"], G["w"]), G["r"])
    assert np.array_equal(O.rollout_item(G["A"], G["B"], G["c"], G["x0"], G["u"]), G["X"])
    lam, gu, gx0 = O.adjoint_item(G["A"], G["B"], G["g"])
    assert np.array_equal(lam, G["lam"])
    assert np.array_equal(gu, G["grad_u"])
    assert np.array_equal(gx0, G["grad_x0"])
    for t in range(1, 4):
        for s in range(t):
            assert np.array_equal(O.phi_block(G["A"], t, s), G["Phi"][O.packed_index(t, s)])


# ------------------------------------------------------------------ Phi
def test_phi_constant_A_is_matrix_power():
    A0 = _rand(1, 5, seed=1)[0][0]
    T = 7
    Phi = O.system_response_item(np.broadcast_to(A0, (T, 5, 5)))
    for t in range(1, T):
        for s in range(t):
            _close(Phi[O.packed_index(t, s)], np.linalg.matrix_power(A0, t - s))


def test_phi_identity_and_scalar():
    T, n = 6, 4
    Phi = O.system_response_item(np.broadcast_to(np.eye(n), (T, n, n)))
    assert np.array_equal(Phi, np.broadcast_to(np.eye(n), Phi.shape))
    a = np.array([0.5, -2.0, 3.0, 0.25, 1.5, 7.0])
    Phi = O.system_response_item(a[:, None, None] * np.eye(n))
    for t in range(1, T):
        for s in range(t):
            _close(Phi[O.packed_index(t, s)], np.prod(a[s:t]) * np.eye(n))


def test_phi_rotations_compose_to_angle_sum():
    th = np.array([0.3, -1.1, 0.7, 2.0, 0.05])
    R = lambda x: np.array([[np.cos(x), -np.sin(x)], [np.sin(x), np.cos(x)]])
    A = np.stack([R(x) for x in th])
    Phi = O.system_response_item(A)
    for t in range(1, 5):
        for s in range(t):
            _close(Phi[O.packed_index(t, s)], R(th[s:t].sum()))


def test_phi_order_of_factors_noncommuting():
    # Phi(2,0) = A_1 A_0, not A_0 A_1 (would pass the rotation pin, which commutes)
    A0 = np.array([[1.0, 1.0], [0.0, 1.0]])
    A1 = np.array([[1.0, 0.0], [1.0, 1.0]])
    Phi = O.system_response_item(np.stack([A0, A1, A0]))
    assert np.array_equal(Phi[O.packed_index(2, 0)], np.array([[1.0, 1.0], [1.0, 2.0]]))


@pytest.mark.parametrize("T,n", [(2, 3), (5, 3), (6, 4)])
def test_phi_defining_identity_12c(T, n):
    """(12c) without feedback: (I - Z blkdiag(A_0..A_{T-2}, *)) Phi_full = I, Phi_full unit block-lower-
    triangular with strictly-lower blocks Phi(t,s).  Checked with numpy.linalg.inv on the T*n system."""
    A = _rand(T, n, seed=3)[0]
    M = np.eye(T * n)
    for t in range(1, T):                     # Z shifts block-row t-1 of blkdiag(A) down to block-row t
        M[t * n:(t + 1) * n, (t - 1) * n:t * n] -= A[t - 1]
    Minv = np.linalg.inv(M)
    Phi = O.system_response_item(A)
    for t in range(T):
        for s in range(T):
            blk = Minv[t * n:(t + 1) * n, s * n:(s + 1) * n]
            if s < t:
                _close(Phi[O.packed_index(t, s)], blk, 1e-10)
            elif s == t:
                _close(blk, np.eye(n), 1e-10)
            else:
                assert np.max(np.abs(blk)) < 1e-10


def test_phi_bruteforce_python_loops():
    T, n = 5, 3
    A = _rand(T, n, seed=4)[0]
    Phi = O.system_response_item(A)
    for t in range(1, T):
        for s in range(t):
            P = [[float(i == j) for j in range(n)] for i in range(n)]
            for k in range(s, t):             # left-multiply by A_k, k = s..t-1
                P = [[sum(A[k][i][l] * P[l][j] for l in range(n)) for j in range(n)] for i in range(n)]
            _close(Phi[O.packed_index(t, s)], np.array(P))
            _close(O.phi_block(A, t, s), np.array(P))


def test_phi_scan_equals_recursion():
    """'obtain the solution ... by a forward parallel associative scan': an independent
    divide-and-conquer composition Phi(t,s) = Phi(t,mid) Phi(mid,s) and the semigroup property for every
    split point reproduce the sequential recursion."""
    T, n = 11, 4
    A = _rand(T, n, seed=5)[0]
    Phi = O.system_response_item(A)
    blocks = {}

    def solve(lo, hi):
        if hi - lo == 1:
            blocks[(hi, lo)] = A[lo]
            return
        mid = (lo + hi) // 2
        solve(lo, mid)
        solve(mid, hi)
        for t in range(mid + 1, hi + 1):
            for s in range(lo, mid):
                blocks[(t, s)] = blocks[(t, mid)] @ blocks[(mid, s)]

    solve(0, T - 1)
    assert len(blocks) == T * (T - 1) // 2
    for (t, s), blk in blocks.items():
        _close(Phi[O.packed_index(t, s)], blk, 1e-11)
    for t in range(2, T):
        for s in range(t - 1):
            for k in range(s + 1, t):
                _close(Phi[O.packed_index(t, k)] @ Phi[O.packed_index(k, s)], Phi[O.packed_index(t, s)], 1e-11)


# ------------------------------------------------------------------ tube
def test_tube_identity_A_is_exclusive_cumsum():
    T, n = 7, 5
    w = _rand(T, n, seed=6)[5]
    r = O.tube_item(np.broadcast_to(np.eye(n), (T, n, n)), w)
    ref = np.concatenate([np.zeros((1, n)), np.cumsum(w, axis=0)[:-1]])
    _close(r, ref)


def test_tube_scalar_closed_form_uses_abs():
    T, n = 6, 3
    a = np.array([0.5, -2.0, 3.0, -0.25, 1.5, 9.0])
    w = _rand(T, n, seed=7)[5]
    r = O.tube_item(a[:, None, None] * np.eye(n), w)
    for t in range(T):
        ref = sum(abs(np.prod(a[s:t])) * w[s] for s in range(t)) if t else np.zeros(n)
        _close(r[t], ref)


def test_tube_bruteforce_and_fused_variant():
    T, n = 5, 4
    A, _, _, _, _, w, _ = _rand(T, n, seed=8)
    Phi = O.system_response_item(A)
    r = O.tube_item(A, w)
    Phi2, r2 = O.system_response_tube_item(A, w)
    assert np.array_equal(Phi, Phi2) and np.array_equal(r, r2)
    for t in range(T):
        for i in range(n):
            acc = 0.0
            for s in range(t):
                for j in range(n):
                    acc += abs(Phi[O.packed_index(t, s)][i, j]) * w[s, j]
            assert abs(r[t, i] - acc) <= 1e-12 * max(1.0, abs(acc))
    assert np.all(r[0] == 0)


def test_tube_containment_invariant_and_tightness():
    """'All rollouts remain within their tubes'.  For the box tube: any |d_s| <= w_s
    gives |sum_s Phi(t,s) d_s| <= r_t, with equality in row i for d_s = w_s * sign(Phi(t,s)[i,:])."""
    T, n = 8, 6
    A, _, _, _, _, w, _ = _rand(T, n, seed=9)
    w = np.abs(w) * 1e3
    Phi = O.system_response_item(A)
    r = O.tube_item(A, w)
    rng = np.random.default_rng(0)
    for _ in range(50):
        d = rng.uniform(-1, 1, (T, n)) * w
        for t in range(1, T):
            v = sum(Phi[O.packed_index(t, s)] @ d[s] for s in range(t))
            assert np.all(np.abs(v) <= r[t] * (1 + 1e-12) + 1e-300)
    for t in range(1, T):
        for i in range(n):
            v = sum(Phi[O.packed_index(t, s)] @ (w[s] * np.sign(Phi[O.packed_index(t, s)][i])) for s in range(t))
            assert abs(v[i] - r[t, i]) <= 1e-12 * max(1.0, r[t, i])


def test_tube_linear_monotone_in_w():
    T, n = 6, 4
    A, _, _, _, _, w, _ = _rand(T, n, seed=10)
    w = np.abs(w)
    w2 = np.abs(_rand(T, n, seed=11)[5])
    _close(O.tube_item(A, 2.0 * w + 3.0 * w2), 2.0 * O.tube_item(A, w) + 3.0 * O.tube_item(A, w2), 1e-11)
    assert np.all(O.tube_item(A, w + w2) >= O.tube_item(A, w) - 1e-15)


# ------------------------------------------------------------------ rollout
# --------------------------------------------------------------------------- row-wise two-norm tube (12e), NEXT-2
def test_tube2_identity_A_and_rotation_closed_forms():
    """A = I: each row of Phi E_s has one entry => tau_t = sum_{s<t} w_s.  Rotations R(th_t) with w_s = c_s (1,1):
    rows of R(.) c_s have two-norm c_s => tau_t = sum_{s<t} c_s whatever the angles."""
    rng = np.random.default_rng(5)
    T, n = 7, 5
    w = rng.uniform(0.0, 1.0, (T, n))
    A = np.broadcast_to(np.eye(n), (T, n, n)).copy()
    tau = O.tube_row2norm_item(A, w)
    np.testing.assert_allclose(tau[0], 0.0)
    np.testing.assert_allclose(tau[1:], np.cumsum(w, axis=0)[:-1], rtol=1e-13)
    th = rng.uniform(-2.0, 2.0, T)
    R = np.stack([np.array([[np.cos(a), -np.sin(a)], [np.sin(a), np.cos(a)]]) for a in th])
    c = rng.uniform(0.1, 1.0, T)
    tau = O.tube_row2norm_item(R, np.stack([c, c], axis=1))
    np.testing.assert_allclose(tau[1:, 0], np.cumsum(c)[:-1], rtol=1e-13)
    np.testing.assert_allclose(tau[1:, 1], np.cumsum(c)[:-1], rtol=1e-13)


def test_tube2_bruteforce_python_loops():
    import math

    W = dense_random(1, 5, 4, 1, seed=31)
    A, w = W.A[0].astype(np.float64), W.w[0].astype(np.float64)
    T, n = 5, 4
    got = O.tube_row2norm_item(W.A[0], W.w[0])
    for t in range(1, T):
        for i in range(n):
            tot = 0.0
            for s in range(t):
                M = np.eye(n)
                for k in range(s, t):          # Phi(t,s) = A_{t-1} ... A_s by explicit left products
                    M = A[k] @ M
                tot += math.sqrt(sum((M[i, j] * w[s][j]) ** 2 for j in range(n)))
            assert abs(got[t, i] - tot) <= 1e-13 * max(1.0, abs(tot))


def test_tube2_containment_cauchy_schwarz_and_tightness():
    """Disturbances d_s = E_s v_s with ||v_s||_2 <= 1: |sum_s Phi(t,s) d_s|_i <= tau_t[i], with equality in row i
    for v_s = row_i(Phi(t,s) E_s) / its norm (PAPER.md:218 containment; Cauchy-Schwarz)."""
    rng = np.random.default_rng(9)
    W = dense_random(1, 6, 7, 1, seed=77)
    A, w = W.A[0], W.w[0].astype(np.float64) * 1e3
    T, n = 6, 7
    tau = O.tube_row2norm_item(A, w)
    Phi = O.system_response_item(A)
    for t in range(1, T):
        for _ in range(20):
            dev = np.zeros(n)
            for s in range(t):
                v = rng.normal(size=n)
                v /= max(1.0, np.linalg.norm(v))
                dev += Phi[O.packed_index(t, s)] @ (w[s] * v)
            assert np.all(np.abs(dev) <= tau[t] * (1 + 1e-12))
        i = t % n
        dev = 0.0
        for s in range(t):
            rowE = Phi[O.packed_index(t, s)][i] * w[s]
            dev += rowE @ (rowE / np.linalg.norm(rowE))
        assert abs(dev - tau[t, i]) <= 1e-12 * tau[t, i]


def test_tube2_sandwiched_by_box_tube():
    """||v||_2 <= ||v||_1 <= sqrt(n) ||v||_2 row by row: box/sqrt(n) <= tau <= box (the box tube is pinned above)."""
    W = generate(config(0))
    A, w = W.A[0], W.w[0]
    n = A.shape[-1]
    box, tau = O.tube_item(A, w), O.tube_row2norm_item(A, w)
    assert np.all(tau <= box * (1 + 1e-12)) and np.all(tau >= box / np.sqrt(n) * (1 - 1e-12))
    assert np.any(tau < 0.9 * box)                       # and it is a different quantity
    np.testing.assert_allclose(O.tube_row2norm(W.A, W.w)[0], tau, rtol=0, atol=0)
    np.testing.assert_allclose(O.tube_row2norm_item(A, 3.0 * w.astype(np.float64)), 3.0 * tau, rtol=1e-13)   # homogeneous in w


# --------------------------------------------------------------------------- observer propagation (14), NEXT-1
def _obs_inputs(T, n, p, seed):
    rng = np.random.default_rng(seed)
    A = np.eye(n)[None] + rng.normal(0.0, 0.4 / np.sqrt(n), (T, n, n))
    return A, rng.normal(0.0, 0.3, (T, n, p)), rng.normal(0.0, 0.5, (T, p, n))


def test_observer_zero_gain_and_scalar_closed_form():
    A, Lt, C = _obs_inputs(6, 5, 2, 1)
    X, Y = O.observer_response_item(A, 0.0 * Lt, C)
    np.testing.assert_allclose(X, O.system_response_item(A), rtol=1e-12, atol=1e-14)   # L = 0: open loop
    assert np.all(Y == 0.0)
    T, n = 6, 3
    a, l = np.linspace(0.5, 1.5, T), np.linspace(-0.4, 0.3, T)
    I = np.eye(n)
    X, Y = O.observer_response_item(a[:, None, None] * I, l[:, None, None] * I, np.broadcast_to(I, (T, n, n)))
    for k in range(1, T):
        for j in range(k):
            pr = np.prod(a[j:k] + l[j:k])
            np.testing.assert_allclose(X[O.packed_index(k, j)], pr * I, rtol=1e-13)
            np.testing.assert_allclose(Y[O.packed_index(k, j)], pr * l[j] * I, rtol=1e-13)


def test_observer_bruteforce_left_products_and_inverse_identity():
    """PhiX(k,j) = Abar_{k-1} ... Abar_j by explicit LEFT products (the oracle multiplies on the right), and the
    strictly-lower blocks of (I - Z blkdiag(Abar))^{-1} (the identity (12c) has for the closed loop)."""
    T, n, p = 5, 4, 2
    A, Lt, C = _obs_inputs(T, n, p, 2)
    X, Y = O.observer_response_item(A, Lt, C)
    Abar = [A[j] + Lt[j] @ C[j] for j in range(T)]
    M = np.eye(T * n)
    for j in range(T - 1):
        M[(j + 1) * n:(j + 2) * n, j * n:(j + 1) * n] = -Abar[j]
    Minv = np.linalg.inv(M)
    for k in range(1, T):
        for j in range(k):
            P = np.eye(n)
            for i in range(j, k):
                P = Abar[i] @ P
            np.testing.assert_allclose(X[O.packed_index(k, j)], P, rtol=1e-12, atol=1e-14)
            np.testing.assert_allclose(X[O.packed_index(k, j)], Minv[k * n:(k + 1) * n, j * n:(j + 1) * n], rtol=1e-10, atol=1e-12)
            np.testing.assert_allclose(Y[O.packed_index(k, j)], P @ Lt[j], rtol=1e-12, atol=1e-14)


def test_observer_semigroup_is_what_the_scan_uses():
    """[PhiX | PhiY](t,s) = PhiX(t,k) [PhiX | PhiY](k,s) for every s < k < t: the combine of the time-parallel scan."""
    T, n, p = 7, 3, 2
    A, Lt, C = _obs_inputs(T, n, p, 3)
    X, Y = O.observer_response_item(A, Lt, C)
    q = O.packed_index
    for t in range(2, T):
        for s in range(t - 1):
            for k in range(s + 1, t):
                np.testing.assert_allclose(X[q(t, s)], X[q(t, k)] @ X[q(k, s)], rtol=1e-11, atol=1e-13)
                np.testing.assert_allclose(Y[q(t, s)], X[q(t, k)] @ Y[q(k, s)], rtol=1e-11, atol=1e-13)
    Xb, Yb = O.observer_response(A[None], Lt[None], C[None])
    assert np.array_equal(Xb[0], X) and np.array_equal(Yb[0], Y)


def test_rollout_identity_A_is_cumsum():
    T, n, m = 6, 4, 2
    _, B, c, x0, u, _, _ = _rand(T, n, m, seed=12)
    X = O.rollout_item(np.broadcast_to(np.eye(n), (T, n, n)), B, c, x0, u)
    b = np.einsum("tnm,tm->tn", B, u) + c
    _close(X, x0[None] + np.cumsum(b, axis=0))


def test_rollout_constant_A_no_input_is_powers():
    T, n = 6, 4
    A0 = _rand(1, n, seed=13)[0][0]
    x0 = _rand(1, n, seed=14)[3]
    X = O.rollout_item(np.broadcast_to(A0, (T, n, n)), None, None, x0, None)
    for t in range(T):
        _close(X[t], np.linalg.matrix_power(A0, t + 1) @ x0)


def test_rollout_superposition_with_phi():
    """x_t = Phi(t,0) x0 + sum_{s=1}^{t} Phi(t,s) b_{s-1}, Phi(t,t) = I: ties rollout to Phi.
    Uses T+1 nodes so that Phi(T, .) exists: feed the Phi oracle A padded with one extra step."""
    T, n, m = 6, 4, 2
    A, B, c, x0, u, _, _ = _rand(T, n, m, seed=15)
    X = O.rollout_item(A, B, c, x0, u)
    Apad = np.concatenate([A, np.eye(n)[None]])          # nodes 0..T, uses A_0..A_{T-1}
    Phi = O.system_response_item(Apad)
    b = np.einsum("tnm,tm->tn", B, u) + c
    for t in range(1, T + 1):
        v = Phi[O.packed_index(t, 0)] @ x0 + b[t - 1]
        for s in range(1, t):
            v = v + Phi[O.packed_index(t, s)] @ b[s - 1]
        _close(X[t - 1], v, 1e-11)


def test_rollout_affine_scan_composition():
    """north_star: compose (A_t, b_t); (A2,b2) o (A1,b1) = (A2 A1, A2 b1 + b2).  A Hillis-Steele inclusive
    scan over these pairs applied to x0 equals the recursion."""
    T, n, m = 9, 3, 2
    A, B, c, x0, u, _, _ = _rand(T, n, m, seed=16)
    X = O.rollout_item(A, B, c, x0, u)
    elems = [(A[t], B[t] @ u[t] + c[t]) for t in range(T)]
    d = 1
    while d < T:
        new = list(elems)
        for t in range(d, T):
            A2, b2 = elems[t]
            A1, b1 = elems[t - d]
            new[t] = (A2 @ A1, A2 @ b1 + b2)
        elems = new
        d *= 2
    for t in range(T):
        _close(X[t], elems[t][0] @ x0 + elems[t][1], 1e-11)


def test_rollout_B_and_c_enter_with_plus_sign_single_step():
    A = np.array([[[2.0, 0.0], [0.0, 3.0]]])
    X = O.rollout_item(A, np.array([[[1.0], [10.0]]]), np.array([[100.0, 1000.0]]), np.array([1.0, 1.0]),
                       np.array([[5.0]]))
    assert np.array_equal(X, np.array([[2 + 5 + 100.0, 3 + 50 + 1000.0]]))


# ------------------------------------------------------------------ adjoint
def test_adjoint_dot_product_identity_u_and_x0():
    """(10) chained: exact because x is affine in (x0, u): sum_t g_t.(x_t(u+du) - x_t(u)) = sum_t grad_u[t].du_t
    for ANY finite du, and likewise for dx0."""
    T, n, m = 7, 5, 3
    A, B, c, x0, u, _, g = _rand(T, n, m, seed=17)
    lam, gu, gx0 = O.adjoint_item(A, B, g)
    rng = np.random.default_rng(1)
    du = rng.normal(size=(T, m))
    dx0 = rng.normal(size=n)
    X0 = O.rollout_item(A, B, c, x0, u)
    lhs = np.sum(g * (O.rollout_item(A, B, c, x0, u + du) - X0))
    assert abs(lhs - np.sum(gu * du)) <= 1e-11 * max(1.0, abs(lhs))
    lhs = np.sum(g * (O.rollout_item(A, B, c, x0 + dx0, u) - X0))
    assert abs(lhs - gx0 @ dx0) <= 1e-11 * max(1.0, abs(lhs))
    # one-hot perturbations pin the time index of grad_u
    for t in range(T):
        for k in range(m):
            du = np.zeros((T, m))
            du[t, k] = 1.0
            lhs = np.sum(g * (O.rollout_item(A, B, c, x0, u + du) - X0))
            assert abs(lhs - gu[t, k]) <= 1e-11 * max(1.0, abs(lhs))


def test_adjoint_equals_sum_of_phi_transposes():
    """lam_t = sum_{k>=t} Phi(k,t)^T g_k, Phi(t,t) = I, over nodes 1..T (A padded like the rollout pin)."""
    T, n = 6, 4
    A, B, _, _, _, _, g = _rand(T, n, seed=18)
    lam, _, _ = O.adjoint_item(A, B, g)
    Apad = np.concatenate([A, np.eye(n)[None]])
    Phi = O.system_response_item(Apad)
    for t in range(1, T + 1):
        v = g[t - 1].copy()
        for k in range(t + 1, T + 1):
            v = v + Phi[O.packed_index(k, t)].T @ g[k - 1]
        _close(lam[t - 1], v, 1e-11)


def test_adjoint_identity_A_is_reverse_cumsum():
    T, n = 6, 3
    g = _rand(T, n, seed=19)[6]
    lam, gu, gx0 = O.adjoint_item(np.broadcast_to(np.eye(n), (T, n, n)), None, g)
    _close(lam, np.cumsum(g[::-1], axis=0)[::-1])
    assert gu is None
    _close(gx0, g.sum(axis=0))


def test_adjoint_central_finite_differences():
    T, n, m = 5, 4, 2
    A, B, c, x0, u, _, g = _rand(T, n, m, seed=20)
    _, gu, _ = O.adjoint_item(A, B, g)
    L = lambda uu: np.sum(g * O.rollout_item(A, B, c, x0, uu))
    h = 1e-3
    for t in range(T):
        for k in range(m):
            e = np.zeros((T, m))
            e[t, k] = h
            fd = (L(u + e) - L(u - e)) / (2 * h)
            assert abs(fd - gu[t, k]) <= 1e-8 * max(1.0, abs(fd))


# ------------------------------------------------------------------ batched wrappers / generator ties
def test_batched_wrappers_match_items():
    W = dense_random(3, 5, 4, 2, seed=21)
    X = O.rollout(W.A, W.B, W.c, W.x0, W.u)
    Phi = O.system_response(W.A)
    r = O.tube(W.A, W.w)
    lam, gu, gx0 = O.adjoint(W.A, W.B, W.g)
    for b in range(3):
        assert np.array_equal(X[b], O.rollout_item(W.A[b], W.B[b], W.c[b], W.x0[b], W.u[b]))
        assert np.array_equal(Phi[b], O.system_response_item(W.A[b]))
        assert np.array_equal(r[b], O.tube_item(W.A[b], W.w[b]))
        l2, gu2, gx2 = O.adjoint_item(W.A[b], W.B[b], W.g[b])
        assert np.array_equal(lam[b], l2) and np.array_equal(gu[b], gu2) and np.array_equal(gx0[b], gx2)


def test_generator_rigid_translation_is_fixed_point_of_phi():
    """L 1 = 0 => rigid translations tau = [e_d (x) 1; 0] satisfy A_t tau = tau, hence Phi(t,s) tau = tau."""
    W = generate(config(0))
    A = W.A[0].astype(np.float64)
    N = W.meta["N"]
    Phi = O.system_response_item(A)
    for d in range(3):
        tau = np.zeros(6 * N)
        tau[d:3 * N:3] = 1.0
        for p in range(Phi.shape[0]):
            assert np.max(np.abs(Phi[p] @ tau - tau)) < 1e-5      # fp32-rounded entries of A


def test_generator_free_fall_of_centre_of_mass():
    """With u = 0 the spring forces cancel in the mean: vbar_{t+1} = (1 - dt c) vbar_t - 9.81 dt e_z."""
    W = generate(config(0))
    N, T = W.meta["N"], W.meta["T"]
    X = O.rollout_item(W.A[0], W.B[0], W.c[0], W.x0[0], np.zeros_like(W.u[0]))
    v = np.concatenate([W.x0[0][None].astype(np.float64), X])[:, 3 * N:].reshape(T + 1, N, 3).mean(axis=1)
    for t in range(T):
        ref = (1 - 0.01 * 0.5) * v[t] + np.array([0, 0, -9.81 * 0.01])
        assert np.max(np.abs(v[t + 1] - ref)) < 1e-5


def test_rel_err_metric():
    assert O.rel_err(np.array([1.0, 2.0, 4.0]), np.array([1.0, 2.0, 5.0])) == pytest.approx(0.2)
    assert O.rel_err(np.zeros(3), np.zeros(3)) == 0.0


def test_observer_achievability_identity_of_12c():
    """Second identity of (12c) for the observer side, Phi_x (I - Z A) - Phi_y (Z C) = I, in blocks:
    PhiX(k,j) - PhiX(k,j+1) A_j = PhiX(k,j+1) Lt_j C_j for j < k (PhiX(k,k) = I).  It holds for the oracle's PhiX with
    the gain that closes the loop around A_j (DESIGN.md q17), and shows which response block that gain multiplies:
    the observation of step j enters through PhiX(k,j+1) Lt_j, one block to the right of the PhiY(k,j) = PhiX(k,j) Lt_j
    that (14) prints (DESIGN.md q20)."""
    T, n, p = 6, 4, 2
    A, Lt, C = _obs_inputs(T, n, p, 9)
    X, _ = O.observer_response_item(A, Lt, C)
    blk = lambda k, j: np.eye(n) if k == j else X[O.packed_index(k, j)]
    N = T * n
    Px, Py = np.zeros((N, N)), np.zeros((N, T * p))       # Py(k, j+1) := PhiX(k,j+1) Lt_j
    ZA, ZC = np.zeros((N, N)), np.zeros((T * p, N))
    for k in range(T):
        for j in range(k + 1):
            Px[k * n:(k + 1) * n, j * n:(j + 1) * n] = blk(k, j)
            if j >= 1:
                Py[k * n:(k + 1) * n, j * p:(j + 1) * p] = blk(k, j) @ Lt[j - 1]
    for j in range(T - 1):
        ZA[(j + 1) * n:(j + 2) * n, j * n:(j + 1) * n] = A[j]
        ZC[(j + 1) * p:(j + 2) * p, j * n:(j + 1) * n] = C[j]
    np.testing.assert_allclose(Px @ (np.eye(N) - ZA) - Py @ ZC, np.eye(N), rtol=0, atol=1e-12)
    # the oracle's own shifted-gain output is exactly that Py (strictly-lower blocks; the diagonal block of Py is
    # PhiX(k,k) Lt_{k-1} = Lt_{k-1}), and the printed form of (14) is NOT: it breaks the identity
    _, Ys = O.observer_response_item(A, Lt, C, shifted_gain=True)
    _, Yp = O.observer_response_item(A, Lt, C)
    Py2, Py3 = np.zeros_like(Py), np.zeros_like(Py)
    for k in range(T):
        if k >= 1:
            Py2[k * n:(k + 1) * n, k * p:(k + 1) * p] = Lt[k - 1]
            Py3[k * n:(k + 1) * n, k * p:(k + 1) * p] = Lt[k - 1]
        for j in range(k):
            Py2[k * n:(k + 1) * n, j * p:(j + 1) * p] = Ys[O.packed_index(k, j)]
            Py3[k * n:(k + 1) * n, j * p:(j + 1) * p] = Yp[O.packed_index(k, j)]
    np.testing.assert_allclose(Py2, Py, rtol=0, atol=1e-13)
    assert np.all(Py2[:, :p] == 0.0)
    assert np.max(np.abs(Px @ (np.eye(N) - ZA) - Py3 @ ZC - np.eye(N))) > 1e-3
