"""Pins for oracle.assemble_output_feedback (eq.(15)) against things other than
itself.  The operators Phibar (state feedback) and Phihat (observer) are built here from gains K_k, Lt_k with the
pinned oracles system_response / observer_response; the assembled Phi must then
  * satisfy BOTH achievability identities of (12c),
  * reproduce a step-by-step simulation of plant + predictor-form observer + controller u = K xhat,
  * equal the blocks of the system response of the augmented closed loop in (x, x - xhat),
  * reduce to the open loop for L = 0 (no information, no action) and for K = 0.
Conventions (DESIGN.md q20, q21): the disturbance w~_k enters x_k directly (Phi(k,k) = I, w~_0 = x_0); the observation
noise e~_k is that of the measurement of x_{k-1} (PAPER.md:125 y_{k+1} = h(q_k) + F e_k), so it enters the estimation
error of step k through Lt_{k-1}: Phihat^y(k,j) = Phihat^x(k,j) Lt_{j-1}, j >= 1."""
import numpy as np

from oracle import ltv_oracle as O


def _setup(T, n, m, p, seed, Kscale=0.3, Lscale=0.3):
    rng = np.random.default_rng(seed)
    A = np.eye(n)[None] + rng.normal(0.0, 0.4 / np.sqrt(n), (T, n, n))
    B = rng.normal(0.0, 1.0, (T, n, m))
    C = rng.normal(0.0, 1.0 / np.sqrt(n), (T, p, n))
    K = Kscale * rng.normal(0.0, 1.0 / np.sqrt(n), (T, m, n))
    Lt = Lscale * rng.normal(0.0, 1.0, (T, n, p))
    return A, B, C, K, Lt


def _dense(blocks, T, n, ncol=None):
    """packed strictly-lower blocks (t,s) + identity diagonal -> dense [T n, T n]"""
    D = np.eye(T * n)
    for t in range(1, T):
        for s in range(t):
            D[t * n:(t + 1) * n, s * n:(s + 1) * n] = blocks[O.packed_index(t, s)]
    return D


def _operators(A, B, C, K, Lt):
    T, n, _ = A.shape
    m, p = B.shape[2], C.shape[1]
    Atil = A + B @ K
    PbX = _dense(O.system_response_item(Atil), T, n)
    PbU = np.zeros((T * m, T * n))
    for k in range(T):
        PbU[k * m:(k + 1) * m] = K[k] @ PbX[k * n:(k + 1) * n]
    PhX = _dense(O.observer_response_item(A, Lt, C)[0], T, n)
    PhY = np.zeros((T * n, T * p))
    for j in range(1, T):
        PhY[:, j * p:(j + 1) * p] = PhX[:, j * n:(j + 1) * n] @ Lt[j - 1]
    return PbX, PbU, PhX, PhY


def test_assembly_satisfies_both_identities_of_12c():
    T, n, m, p = 5, 4, 2, 2
    A, B, C, K, Lt = _setup(T, n, m, p, 1)
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A, *_operators(A, B, C, K, Lt))
    N = T * n
    M, ZB, ZC = np.eye(N) - O.shift_operator(A), O.shift_operator(B), O.shift_operator(C)
    Phi = np.block([[Pxw, Pxe], [Puw, Pue]])
    np.testing.assert_allclose(np.hstack([M, -ZB]) @ Phi, np.hstack([np.eye(N), np.zeros((N, T * p))]), atol=1e-12)
    np.testing.assert_allclose(Phi @ np.vstack([M, -ZC]), np.vstack([np.eye(N), np.zeros((T * m, N))]), atol=1e-12)


def test_assembly_reproduces_the_simulated_closed_loop():
    T, n, m, p = 6, 4, 2, 2
    A, B, C, K, Lt = _setup(T, n, m, p, 2)
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A, *_operators(A, B, C, K, Lt))
    rng = np.random.default_rng(3)
    w, e = rng.normal(size=(T, n)), rng.normal(size=(T, p))
    e[0] = 0.0                                         # no measurement precedes step 0
    x, xh = w[0].copy(), np.zeros(n)                   # x_0 = w~_0, xhat_0 = 0
    X, U = [], []
    for k in range(T):
        u = K[k] @ xh
        X.append(x.copy()); U.append(u.copy())
        if k + 1 < T:
            y = C[k] @ x + e[k + 1]                    # measurement of x_k, noise e~_{k+1}
            xh = A[k] @ xh + B[k] @ u - Lt[k] @ (y - C[k] @ xh)
            x = A[k] @ x + B[k] @ u + w[k + 1]
    np.testing.assert_allclose(np.concatenate(X), Pxw @ w.ravel() + Pxe @ e.ravel(), atol=1e-11)
    np.testing.assert_allclose(np.concatenate(U), Puw @ w.ravel() + Pue @ e.ravel(), atol=1e-11)


def test_assembly_is_the_augmented_closed_loop_response():
    """xi = (x, eps), eps = x - xhat: xi_{k+1} = [[A + B K, -B K], [0, A + Lt C]] xi_k + [I; I] w~ + [0; Lt] e~.
    Phi^xw(k,j) = [I 0] Phi_aug(k,j) [I; I],  Phi^xe(k,j) = [I 0] Phi_aug(k,j) [0; Lt_{j-1}] - what the existing Phi scan
    computes when it is run on the 2n-state augmented system (the GPU test does exactly that)."""
    T, n, m, p = 5, 3, 2, 2
    A, B, C, K, Lt = _setup(T, n, m, p, 4)
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A, *_operators(A, B, C, K, Lt))
    Aaug = np.zeros((T, 2 * n, 2 * n))
    Aaug[:, :n, :n] = A + B @ K
    Aaug[:, :n, n:] = -(B @ K)
    Aaug[:, n:, n:] = A + Lt @ C
    Paug = O.system_response_item(Aaug)
    for k in range(T):
        for j in range(k + 1):
            G = np.eye(2 * n) if k == j else Paug[O.packed_index(k, j)]
            np.testing.assert_allclose(Pxw[k * n:(k + 1) * n, j * n:(j + 1) * n], G[:n, :n] + G[:n, n:], atol=1e-12)
            np.testing.assert_allclose(Puw[k * m:(k + 1) * m, j * n:(j + 1) * n],
                                       K[k] @ (G[:n, :n] + G[:n, n:] - G[n:, :n] - G[n:, n:]), atol=1e-12)
            if j >= 1:
                np.testing.assert_allclose(Pxe[k * n:(k + 1) * n, j * p:(j + 1) * p], G[:n, n:] @ Lt[j - 1], atol=1e-12)
    assert np.max(np.abs(Pxe[:, :p])) == 0.0


def test_assembly_limits_no_observer_gain_and_no_feedback_gain():
    T, n, m, p = 5, 4, 2, 2
    A, B, C, K, Lt = _setup(T, n, m, p, 5)
    open_loop = _dense(O.system_response_item(A), T, n)
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A, *_operators(A, B, C, K, 0.0 * Lt))
    np.testing.assert_allclose(Pxw, open_loop, atol=1e-12)          # no information: the controller cannot act
    assert np.max(np.abs(Puw)) < 1e-12 and np.max(np.abs(Pxe)) == 0.0 and np.max(np.abs(Pue)) == 0.0
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A, *_operators(A, B, C, 0.0 * K, Lt))
    np.testing.assert_allclose(Pxw, open_loop, atol=1e-12)          # no feedback: the estimate is never used
    assert np.max(np.abs(Puw)) == 0.0 and np.max(np.abs(Pue)) == 0.0 and np.max(np.abs(Pxe)) < 1e-12


def test_output_feedback_tube_contains_the_simulated_loop_and_is_tight():
    """(12e): for any ||d_j||_2 <= 1, ||g_j||_2 <= 1 the simulated state obeys |x_k[i]| <= tau_k[i] when w~_j = E_j d_j
    (j < k; no direct term), e~_j = F~_j g_j; equality in row i for the aligned disturbances."""
    T, n, m, p = 5, 4, 2, 2
    A, B, C, K, Lt = _setup(T, n, m, p, 7)
    rng = np.random.default_rng(8)
    w, f = rng.uniform(0.1, 1.0, (T, n)), rng.uniform(0.1, 1.0, (T, p))
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A, *_operators(A, B, C, K, Lt))
    tau = O.output_feedback_tube(Pxw, Pxe, w, f)
    assert np.all(tau[0] == 0.0)
    k = T - 1
    for i in range(n):
        # aligned worst case for row i of x_k, disturbances at steps j < k only
        wt, et = np.zeros((T, n)), np.zeros((T, p))
        for j in range(k):
            r = Pxw[k * n + i, j * n:(j + 1) * n] * w[j]
            wt[j] = w[j] * r / np.linalg.norm(r)
            if j >= 1:
                q = Pxe[k * n + i, j * p:(j + 1) * p] * f[j - 1]
                et[j] = f[j - 1] * q / np.linalg.norm(q)
        xk = (Pxw @ wt.ravel() + Pxe @ et.ravel())[k * n + i]
        assert abs(xk - tau[k, i]) <= 1e-12 * tau[k, i]
    for _ in range(20):
        d = rng.normal(size=(T, n)); d /= np.maximum(1.0, np.linalg.norm(d, axis=1, keepdims=True))
        g = rng.normal(size=(T, p)); g /= np.maximum(1.0, np.linalg.norm(g, axis=1, keepdims=True))
        wt, et = w * d, np.vstack([np.zeros((1, p)), f[:-1] * g[1:]])
        wt[k:] = 0.0
        x = (Pxw @ wt.ravel() + Pxe @ et.ravel()).reshape(T, n)
        assert np.all(np.abs(x[k]) <= tau[k] * (1 + 1e-12))


def test_output_feedback_tube_without_feedback_is_the_row2norm_tube():
    T, n, m, p = 5, 4, 2, 2
    A, B, C, K, Lt = _setup(T, n, m, p, 9)
    w, f = np.random.default_rng(1).uniform(0.1, 1.0, (T, n)), np.ones((T, p))
    Pxw, _, Pxe, _ = O.assemble_output_feedback(A, *_operators(A, B, C, 0.0 * K, Lt))
    np.testing.assert_allclose(O.output_feedback_tube(Pxw, Pxe, w, f), O.tube_row2norm_item(A, w), rtol=1e-10, atol=1e-12)


# ------------------------------------------------------------------ (12d), both terms, rows on [z; v]
def _simulate(A, B, C, K, Lt, wt, et):
    """plant + predictor-form observer + controller u = K xhat, step by step (q21 conventions); returns X[T,n], U[T,m]"""
    T, n = wt.shape
    x, xh = wt[0].copy(), np.zeros(n)
    X, U = [], []
    for k in range(T):
        u = K[k] @ xh
        X.append(x.copy()); U.append(u.copy())
        if k + 1 < T:
            y = C[k] @ x + et[k + 1]
            xh = A[k] @ xh + B[k] @ u - Lt[k] @ (y - C[k] @ xh)
            x = A[k] @ x + B[k] @ u + wt[k + 1]
    return np.array(X), np.array(U)


def test_closed_loop_constraint_margins_contain_the_simulated_loop_and_are_tight():
    """(12d): with w~_j = E_j d_j, e~_j = F~_j g_j, ||d_j||_2, ||g_j||_2 <= 1 injected at steps j < k only, the SIMULATED
    closed loop obeys c^T [x_k; u_k] <= sigma_k[i]; the aligned disturbances reach it.  Rows mix state and input."""
    T, n, m, p, nc = 6, 4, 2, 2, 3
    A, B, C, K, Lt = _setup(T, n, m, p, 21)
    rng = np.random.default_rng(22)
    w, f = rng.uniform(0.1, 1.0, (T, n)), rng.uniform(0.1, 1.0, (T, p))
    Hx, Hu = rng.normal(size=(T, nc, n)), rng.normal(size=(T, nc, m))
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A, *_operators(A, B, C, K, Lt))
    sig = O.output_feedback_constraint_tightening(Pxw, Puw, Pxe, Pue, w, f, Hx, Hu)
    assert np.all(sig[0] == 0.0) and np.all(sig[1:] > 0.0)
    for k in (2, T - 1):
        for i in range(nc):
            wt, et = np.zeros((T, n)), np.zeros((T, p))
            for j in range(k):
                rw = (Hx[k, i] @ Pxw[k * n:(k + 1) * n, j * n:(j + 1) * n] + Hu[k, i] @ Puw[k * m:(k + 1) * m, j * n:(j + 1) * n]) * w[j]
                wt[j] = w[j] * rw / np.linalg.norm(rw)
                if j >= 1:
                    re = (Hx[k, i] @ Pxe[k * n:(k + 1) * n, j * p:(j + 1) * p] + Hu[k, i] @ Pue[k * m:(k + 1) * m, j * p:(j + 1) * p]) * f[j - 1]
                    et[j] = f[j - 1] * re / np.linalg.norm(re)
            X, U = _simulate(A, B, C, K, Lt, wt, et)
            val = Hx[k, i] @ X[k] + Hu[k, i] @ U[k]
            assert abs(val - sig[k, i]) <= 1e-11 * sig[k, i]
        for _ in range(20):
            d = rng.normal(size=(T, n)); d /= np.maximum(1.0, np.linalg.norm(d, axis=1, keepdims=True))
            g = rng.normal(size=(T, p)); g /= np.maximum(1.0, np.linalg.norm(g, axis=1, keepdims=True))
            wt, et = w * d, np.vstack([np.zeros((1, p)), f[:-1] * g[1:]])
            wt[k:] = 0.0
            et[k:] = 0.0
            X, U = _simulate(A, B, C, K, Lt, wt, et)
            assert np.all(np.abs(Hx[k] @ X[k] + Hu[k] @ U[k]) <= sig[k] * (1 + 1e-12))


def test_closed_loop_constraint_margins_special_cases():
    T, n, m, p = 5, 4, 2, 2
    A, B, C, K, Lt = _setup(T, n, m, p, 23)
    rng = np.random.default_rng(24)
    w, f = rng.uniform(0.1, 1.0, (T, n)), rng.uniform(0.1, 1.0, (T, p))
    ops = O.assemble_output_feedback(A, *_operators(A, B, C, K, Lt))
    # identity state rows, no input part: the output-feedback tube (12e)
    Hx = np.broadcast_to(np.eye(n), (T, n, n))
    sig = O.output_feedback_constraint_tightening(*ops, w, f, Hx, np.zeros((T, n, m)))
    np.testing.assert_allclose(sig, O.output_feedback_tube(ops[0], ops[2], w, f), rtol=1e-12, atol=0)
    # input rows only: scalar loops over the blocks of Phi^uw, Phi^ue
    Hu = rng.normal(size=(T, 3, m))
    sig = O.output_feedback_constraint_tightening(*ops, w, f, np.zeros((T, 3, n)), Hu)
    for k in range(T):
        for i in range(3):
            acc = 0.0
            for j in range(k):
                s1 = sum((sum(Hu[k, i, a] * ops[1][k * m + a, j * n + c] for a in range(m)) * w[j, c]) ** 2 for c in range(n))
                acc += np.sqrt(s1)
                if j >= 1:
                    s2 = sum((sum(Hu[k, i, a] * ops[3][k * m + a, j * p + q] for a in range(m)) * f[j - 1, q]) ** 2 for q in range(p))
                    acc += np.sqrt(s2)
            assert abs(acc - sig[k, i]) <= 1e-12 * max(1.0, acc)
    # no feedback (K = 0): Phi^u = 0, Phi^xe = 0, Phi^xw = open loop -> the open-loop margins of constraint_tightening
    ops0 = O.assemble_output_feedback(A, *_operators(A, B, C, 0.0 * K, Lt))
    Hx = rng.normal(size=(T, 3, n))
    sig0 = O.output_feedback_constraint_tightening(*ops0, w, f, Hx, Hu)
    np.testing.assert_allclose(sig0, O.constraint_tightening_item(A, w, Hx), rtol=1e-10, atol=1e-12)


def test_backward_recursion_of_the_general_assembly_equals_eq15():
    """The identity the device call ltv_scan_output_feedback_assemble is built on, checked against (15) AS EVALUATED BY THE
    ORACLE on dense operators, for a general achievable Phibar (not generated from gains):
        Phi^xw(k,j) = Phi^xw(k,j+1) Abar_j - Phibar^x(k,j+1) Lt_j C_j,  Phi^xw(k,k) = I;   same for Phi^uw with Phibar^u, start 0;
        Phi^xe(k,j) = (Phi^xw - Phibar^x)(k,j) Lt_{j-1},   Phi^ue(k,j) = (Phi^uw - Phibar^u)(k,j) Lt_{j-1}   (j >= 1)."""
    from assembly_inputs import blk, general_phibar, observer_operators

    rng = np.random.default_rng(77)
    T, n, m, p = 7, 6, 2, 3
    A = np.eye(n)[None] + rng.normal(0.0, 0.4 / np.sqrt(n), (T, n, n))
    B = rng.normal(0.0, 1.0, (T, n, m))
    C = rng.normal(0.0, 1.0 / np.sqrt(n), (T, p, n))
    Lt = 0.3 * rng.normal(0.0, 1.0, (T, n, p))
    PbX, PbU = general_phibar(A, B, seed=5)
    for k in range(T):
        assert np.allclose(blk(PbX, k, k, n, n), np.eye(n), atol=1e-12)          # what the call takes for granted
    # the state-feedback achievability constraint holds (so this IS a response the first SLS stage could return)
    ZB = np.zeros((T * n, T * m))
    for t in range(T - 1):
        ZB[(t + 1) * n:(t + 2) * n, t * m:(t + 1) * m] = B[t]
    assert np.allclose((np.eye(T * n) - O.shift_operator(A)) @ PbX - ZB @ PbU, np.eye(T * n), atol=1e-10)
    PhX, PhY = observer_operators(A, Lt, C)
    Pxw, Puw, Pxe, Pue = O.assemble_output_feedback(A, PbX, PbU, PhX, PhY)
    Abar = A + Lt @ C
    err = 0.0
    for k in range(1, T):
        X, U = np.eye(n), np.zeros((m, n))
        for j in range(k - 1, -1, -1):
            X = X @ Abar[j] - blk(PbX, k, j + 1, n, n) @ Lt[j] @ C[j]
            U = U @ Abar[j] - blk(PbU, k, j + 1, m, n) @ Lt[j] @ C[j]
            err = max(err, np.abs(X - blk(Pxw, k, j, n, n)).max(), np.abs(U - blk(Puw, k, j, m, n)).max())
            if j >= 1:
                err = max(err, np.abs((X - blk(PbX, k, j, n, n)) @ Lt[j - 1] - blk(Pxe, k, j, n, p)).max())
                err = max(err, np.abs((U - blk(PbU, k, j, m, n)) @ Lt[j - 1] - blk(Pue, k, j, m, p)).max())
            else:
                assert np.abs(blk(Pxe, k, 0, n, p)).max() == 0.0 and np.abs(blk(Pue, k, 0, m, p)).max() == 0.0
    assert err < 1e-12
    # the gain-defined controller is the special case Phibar^u(k,j) = K_k Phibar^x(k,j)
    assert np.abs(blk(Puw, 3, 3, m, n)).max() < 1e-12 and np.allclose(blk(Pxw, 3, 3, n, n), np.eye(n))


def test_difference_recursion_of_the_gain_defined_response_equals_eq15():
    """The identity the COLUMN route of ltv_scan_output_feedback_response is built on, against (15) as evaluated by the oracle
    on dense operators, for a controller given by gains (u = K xhat, Phibar = (I - Z(A + B K))^-1): the difference
    D = Phi^xw - Phibar^x obeys
        D(k,j) = D(k,j+1) Abar_j - [Phibar^x(k,j+1) B_j] K_j,   D(k,k) = 0,   Abar_j = A_j + Lt_j C_j,
    (the general recursion minus Phibar^x(k,j) = Phibar^x(k,j+1)(A_j + B_j K_j)), and Phi^xe(k,j) = D(k,j) Lt_{j-1}: no
    difference of nearly equal operators appears - which is why the device carries D and not Phi^xw when the gains are small."""
    from assembly_inputs import blk, observer_operators

    rng = np.random.default_rng(91)
    T, n, m, p = 7, 6, 2, 3
    A = np.eye(n)[None] + rng.normal(0.0, 0.4 / np.sqrt(n), (T, n, n))
    B = rng.normal(0.0, 1.0, (T, n, m))
    C = rng.normal(0.0, 1.0 / np.sqrt(n), (T, p, n))
    K = 0.3 * rng.normal(0.0, 1.0 / np.sqrt(n), (T, m, n))
    Lt = 0.3 * rng.normal(0.0, 1.0, (T, n, p))
    Atil = A + B @ K
    PbX = np.eye(T * n)
    for t, row in O.phi_rows_item(Atil):
        for s_ in range(t):
            PbX[t * n:(t + 1) * n, s_ * n:(s_ + 1) * n] = row[s_]
    PbU = np.vstack([K[k] @ PbX[k * n:(k + 1) * n] for k in range(T)])
    PhX, PhY = observer_operators(A, Lt, C)
    Pxw, _, Pxe, _ = O.assemble_output_feedback(A, PbX, PbU, PhX, PhY)
    Abar = A + Lt @ C
    err = 0.0
    for k in range(1, T):
        D = np.zeros((n, n))
        for j in range(k - 1, -1, -1):
            D = D @ Abar[j] - blk(PbX, k, j + 1, n, n) @ B[j] @ K[j]
            err = max(err, np.abs(D + blk(PbX, k, j, n, n) - blk(Pxw, k, j, n, n)).max())
            if j >= 1:
                err = max(err, np.abs(D @ Lt[j - 1] - blk(Pxe, k, j, n, p)).max())
    assert err < 1e-12
    # small gains: D is small against Phi^xw, the case in which (Phi^xw - Phibar^x) Lt computed in fp32 loses digits
    Ks = 1e-4 * K
    Ds = -(B[0] @ Ks[0])                                   # D(1,0)
    assert np.abs(Ds).max() < 1e-3 * np.abs(A[0]).max()
