"""fp64 CPU oracle for the LTV-scan hot path.  TEST INFRASTRUCTURE - NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference` legs of `bench.py`
may import this module.  It shares no code with `paper_2606_14188_b200/` (the CUDA path) and neither
imports the other; both get their inputs from `workloads/`.

What it is: the plain definition, written out in the paper's order, in fp64 (numpy; `@` = BLAS dgemm /
dgemv used as a library step).  The method reaches EXACTLY (up to rounding order) the result of the
sequential recursion - "We obtain the solution to (14) by a forward parallel associative scan"
 - so the oracle is that recursion, with no blocking, fusion or reordering.

  rollout          x_{t+1} = A_t x_t + B_t u_t + c_t                 PAPER.md:53 eq.(2), :139 eq.(12b)
                                                                     linearised about the nominal
                                                                     trajectory (:150); affine term per
                                                                     BASELINE.json north_star (i)
  system_response  Phi(t,t-1) = A_{t-1}; Phi(t,s) = A_{t-1} Phi(t-1,s)   strictly-lower blocks of
                                                                     (I - Z A)^{-1}
                                                                     eq.(12c) with Z of :150; recursion
                                                                     shape of :159 eq.(14)
  tube             r_0 = 0; r_t = sum_{s<t} |Phi(t,s)| w_s           PAPER.md:147 eq.(12e) in the
                                                                     north_star (ii) form (element-wise
                                                                     abs, box disturbance |d_s| <= w_s)
  tube_row2norm    tau_0 = 0; tau_t[i] = sum_{s<t} ||row_i(Phi(t,s) E_s)||_2    PAPER.md:147 eq.(12e) as printed
                                                                     (row-wise two-norm, :150), with the
                                                                     stand-in E_s = diag(w_s) (SURVEY 8f
                                                                     NEXT-2; reading q3b)
  constraint_tightening  sigma_0 = 0; sigma_k[i] = sum_{j<k} ||c_{k,i}^T Phi(k,j) E_j||_2      PAPER.md:144-145 eq.(12d), state part
                                                                     of the constraint rows only, Phi^w = Phi,
                                                                     E_j = diag(w_j) (DESIGN.md
                                                                     readings q3b, q19)
  observer_response  PhiX(k,k) = I; PhiX(k,j) = PhiX(k,j+1) (A_j + L_j^T C_j);     PAPER.md:157-160 eq.(14), read with
                   PhiY(k,j) = PhiX(k,j) L_j^T,  0 <= j < k <= T-1                 k-independent gains L_j (:177; SURVEY
                                                                     8f NEXT-1, reading q15)
  kalman_recursion Pi_0 = Xi Xi^T; L_{j+1} = -(F_j F_j^T + C_j Pi_j C_j^T)^{-1} C_j Pi_j A_j^T;   PAPER.md:152-155 eq.(13), with the
                   Pi_{j+1} = E_j E_j^T + A_j Pi_j A_j^T + A_j Pi_j C_j^T L_{j+1}             k-independent reading of :177 and
                                                                     the stand-ins E_j = diag(e_j),
                                                                     F_j = diag(f_j) (
                                                                     DESIGN.md readings q3b, q17, q18)
  riccati_scan     the same Pi_j by the associative combination rules (16) with the initial values   PAPER.md:166-177 eq.(16)(17); (16) is
                   (17), folded in the order Pi_j = P~ of e_{j-1} (x) ... (x) e_0 (x) e_init          garbled in the source and
                                                                     is re-derived from the conditional
                                                                     value function of :166 (DESIGN.md q14)
  assemble_output_feedback   Phi^xw = Phibar^x + Phihat^x - Phibar^x M Phihat^x,  Phi^uw = Phibar^u (I - M Phihat^x),      PAPER.md:162-164 eq.(15),
                   Phi^xe = Phihat^y - Phibar^x M Phihat^y,  Phi^ue = -Phibar^u M Phihat^y,  M = I - Z A                 dense block operators
                                                                     (DESIGN.md q20, q21)
  output_feedback_constraint_tightening   sigma_k[i] = sum_{j<k} ||c_{k,i}^T Phi^w(k,j) E_j||_2 + ||c_{k,i}^T Phi^e(k,j) F~_j||_2,     PAPER.md:144-145 eq.(12d) as
                   c on [z_k; v_k], Phi^w = [Phi^xw; Phi^uw], Phi^e = [Phi^xe; Phi^ue] of (15)                    printed, both terms (NEXT-4)
  adjoint          lam_T = g_T; lam_t = A_t^T lam_{t+1} + g_t;       PAPER.md:106-110 eq.(10) chained
                   grad_u[t] = B_t^T lam_{t+1}; grad_x0 = A_0^T lam_1   over the horizon; north_star (iii)

Index conventions (DESIGN.md "Readings" q1, q2, q5): nodes 0 <= s < t <= T-1, P = T(T-1)/2 blocks,
packed block index p = t(t-1)/2 + s; X[t] = x_{t+1}; g[t-1] = g_t; lam[t-1] = lam_t; lam_{T+1} = 0.

Inputs are the fp32 arrays handed to the GPU, promoted to fp64 here (never a separate fp64 copy).

Pins (tests/test_oracle_pins.py): every function below is pinned by closed forms, the defining identity
(12c), brute force on tiny inputs, a hand-computed worked example (tests/golden/hand_example.txt) and the
tube-containment / adjoint dot-product invariants.  kalman_recursion / riccati_* are pinned in
tests/test_oracle_pins_kalman.py (brute-force Gaussian conditioning, information form, DARE fixed point from
scipy, Lyapunov sum through Phi, Joseph form + gain optimality, scan = recursion, associativity);
assemble_output_feedback in tests/test_oracle_pins_assembly.py (both achievability identities of (12c), a step-by-step
simulation of plant + observer + controller, the augmented closed-loop system, the limits L = 0 and K = 0);
output_feedback_constraint_tightening there too (worst-case containment with tightness on the simulated loop for state
AND input rows, identity state rows = the output-feedback tube, K = 0 = the open-loop margins).
Nothing in this file is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def _f64(a):
    return None if a is None else np.asarray(a, dtype=np.float64)


def packed_index(t: int, s: int) -> int:
    """Row-packed position of block (t, s), 0 <= s < t."""
    return t * (t - 1) // 2 + s


# --------------------------------------------------------------------------- rollout
def rollout_item(A, B, c, x0, u):
    """One batch item.  A[T,n,n], B[T,n,m] or None, c[T,n] or None, x0[n], u[T,m] or None -> X[T,n]
    with X[t] = x_{t+1}."""
    A = _f64(A)
    T, n, _ = A.shape
    X = np.empty((T, n))
    x = _f64(x0).copy()
    for t in range(T):
        x = A[t] @ x
        if B is not None and u is not None:
            x = x + _f64(B[t]) @ _f64(u[t])
        if c is not None:
            x = x + _f64(c[t])
        X[t] = x
    return X


def rollout(A, B, c, x0, u):
    """Batched: A[batch,T,n,n] ... -> X[batch,T,n]."""
    nb = A.shape[0]
    sel = lambda a, b: None if a is None else a[b]
    return np.stack([rollout_item(A[b], sel(B, b), sel(c, b), x0[b], sel(u, b)) for b in range(nb)])


# --------------------------------------------------------------------------- Phi
def phi_rows_item(A):
    """Generator over block rows for one item: yields (t, row) for t = 1..T-1 where row[s] = Phi(t,s),
    s = 0..t-1, via Phi(t,t-1) = A_{t-1}, Phi(t,s) = A_{t-1} Phi(t-1,s)."""
    T = A.shape[0]
    prev = []
    for t in range(1, T):
        At = _f64(A[t - 1])
        row = [At @ prev[s] for s in range(t - 1)]
        row.append(At.copy())
        yield t, row
        prev = row


def system_response_item(A):
    """All blocks of one item, packed: Phi[P,n,n], Phi[t(t-1)/2+s] = A_{t-1} ... A_s."""
    T, n, _ = A.shape
    Phi = np.empty((T * (T - 1) // 2, n, n))
    for t, row in phi_rows_item(A):
        for s in range(t):
            Phi[packed_index(t, s)] = row[s]
    return Phi


def system_response(A):
    return np.stack([system_response_item(A[b]) for b in range(A.shape[0])])


def observer_response_item(A, Lt, C, shifted_gain=False):
    """Closed-loop observer propagation of one item, eq.(14) in the paper's own order: for every
    k, PhiX(k,k) = I and, for j = k-1 down to 0, PhiX(k,j) = PhiX(k,j+1) (A_j + L_j^T C_j) (RIGHT multiplication),
    PhiY(k,j) = PhiX(k,j) L_j^T.  Lt[j] = L_j^T [n,p], C[j] [p,n].  Returns packed PhiX[P,n,n], PhiY[P,n,p].
    shifted_gain=True returns instead the Phihat^y that satisfies the second achievability identity of (12c)
     and enters the assembly (15): PhiY(k,j) = PhiX(k,j) Lt[j-1] for j >= 1, PhiY(k,0) = 0 (DESIGN.md
    readings q20, q21; pinned by test_observer_achievability_identity_of_12c)."""
    A, Lt, C = _f64(A), _f64(Lt), _f64(C)
    T, n, _ = A.shape
    p = Lt.shape[-1]
    PhiX = np.empty((T * (T - 1) // 2, n, n))
    PhiY = np.empty((T * (T - 1) // 2, n, p))
    for k in range(1, T):
        X = np.eye(n)
        for j in range(k - 1, -1, -1):
            X = X @ (A[j] + Lt[j] @ C[j])
            PhiX[packed_index(k, j)] = X
            if not shifted_gain:
                PhiY[packed_index(k, j)] = X @ Lt[j]
            else:
                PhiY[packed_index(k, j)] = X @ Lt[j - 1] if j >= 1 else np.zeros((n, p))
    return PhiX, PhiY


def observer_response(A, Lt, C, shifted_gain=False):
    out = [observer_response_item(A[b], Lt[b], C[b], shifted_gain) for b in range(A.shape[0])]
    return np.stack([o[0] for o in out]), np.stack([o[1] for o in out])


# --------------------------------------------------------------------------- assembly (15)
def shift_operator(A):
    """Z blkdiag(A_0 .. A_{T-1}) as a dense [T n, T n] matrix: block (t+1, t) = A_t (Z = block down-shift, PAPER.md:150;
    A_{T-1} falls off the end).  Works for any per-step blocks A[T, r, c] (returns [T r, T c])."""
    A = _f64(A)
    T, r, c = A.shape
    Z = np.zeros((T * r, T * c))
    for t in range(T - 1):
        Z[(t + 1) * r:(t + 2) * r, t * c:(t + 1) * c] = A[t]
    return Z


def assemble_output_feedback(A, PhibarX, PhibarU, PhihatX, PhihatY):
    """Eq.(15) written out on dense block operators over the T steps of one item:
        M = I - Z A
        Phi^xw = Phibar^x + Phihat^x - Phibar^x M Phihat^x        Phi^uw = Phibar^u (I - M Phihat^x)
        Phi^xe = Phihat^y - Phibar^x M Phihat^y                   Phi^ue = -Phibar^u M Phihat^y
    A[T,n,n]; PhibarX, PhihatX [T n, T n]; PhibarU [T m, T n]; PhihatY [T n, T p], all block lower triangular.
    Returns (Phixw, Phiuw, Phixe, Phiue)."""
    A = _f64(A)
    Pbx, Pbu, Phx, Phy = _f64(PhibarX), _f64(PhibarU), _f64(PhihatX), _f64(PhihatY)
    N = Pbx.shape[0]
    M = np.eye(N) - shift_operator(A)
    Phixw = Pbx + Phx - Pbx @ M @ Phx
    Phiuw = Pbu @ (np.eye(N) - M @ Phx)
    Phixe = Phy - Pbx @ M @ Phy
    Phiue = -Pbu @ M @ Phy
    return Phixw, Phiuw, Phixe, Phiue


def output_feedback_tube(Phixw, Phixe, w, f):
    """Reachable-tube width of eq.(12e) as printed, both terms, for one item:
        tau_k[i] = sum_{j=0}^{k-1} ( || row_i(Phi^xw(k,j) E_j) ||_2 + || row_i(Phi^xe(k,j) F~_j) ||_2 ),
    E_j = diag(w[j]); F~_j = diag(f[j-1]) scales the noise of the measurement of x_{j-1} (DESIGN.md q21; no such term
    for j = 0).  Phixw [T n, T n], Phixe [T n, T p] dense (from assemble_output_feedback); w[T,n], f[T,p] -> tau[T,n]."""
    Pw, Pe, w, f = _f64(Phixw), _f64(Phixe), _f64(w), _f64(f)
    T, n = w.shape
    p = f.shape[1]
    tau = np.zeros((T, n))
    for k in range(1, T):
        for j in range(k):
            blk = Pw[k * n:(k + 1) * n, j * n:(j + 1) * n] @ np.diag(w[j])
            tau[k] += np.sqrt(np.sum(blk ** 2, axis=1))
            if j >= 1:
                ble = Pe[k * n:(k + 1) * n, j * p:(j + 1) * p] @ np.diag(f[j - 1])
                tau[k] += np.sqrt(np.sum(ble ** 2, axis=1))
    return tau


def output_feedback_constraint_tightening(Phixw, Phiuw, Phixe, Phiue, w, f, Hx, Hu):
    """Constraint-tightening margins of eq.(12d) as printed, BOTH terms, constraint rows acting on
    the stacked (state, input) pair [z_k; v_k], for one item:
        sigma_0 = 0;   sigma_k[i] = sum_{j=0}^{k-1} ( || c_{k,i}^T Phi^w(k,j) E_j ||_2 + || c_{k,i}^T Phi^e(k,j) F~_j ||_2 ),
    c_{k,i}^T = [Hx[k,i,:], Hu[k,i,:]] (n + m entries),  Phi^w(k,j) = [Phi^xw(k,j); Phi^uw(k,j)] ((n+m) x n),
    Phi^e(k,j) = [Phi^xe(k,j); Phi^ue(k,j)] ((n+m) x p), E_j = diag(w[j]); F~_j = diag(f[j-1]) scales the noise of the
    measurement of x_{j-1} (DESIGN.md q21: no such term for j = 0).  The dense operators are those of
    assemble_output_feedback: Phixw [T n, T n], Phiuw [T m, T n], Phixe [T n, T p], Phiue [T m, T p].
    w[T,n], f[T,p], Hx[T,nc,n], Hu[T,nc,m] -> sigma[T,nc].  One block, one row, one norm at a time."""
    Pxw, Puw, Pxe, Pue = _f64(Phixw), _f64(Phiuw), _f64(Phixe), _f64(Phiue)
    w, f, Hx, Hu = _f64(w), _f64(f), _f64(Hx), _f64(Hu)
    T, n = w.shape
    p = f.shape[1]
    nc, m = Hu.shape[1], Hu.shape[2]
    sigma = np.zeros((T, nc))
    for k in range(1, T):
        for j in range(k):
            Pw = np.vstack([Pxw[k * n:(k + 1) * n, j * n:(j + 1) * n], Puw[k * m:(k + 1) * m, j * n:(j + 1) * n]])
            Pe = np.vstack([Pxe[k * n:(k + 1) * n, j * p:(j + 1) * p], Pue[k * m:(k + 1) * m, j * p:(j + 1) * p]])
            for i in range(nc):
                c = np.concatenate([Hx[k, i], Hu[k, i]])
                sigma[k, i] += np.sqrt(np.sum((c @ Pw @ np.diag(w[j])) ** 2))
                if j >= 1:
                    sigma[k, i] += np.sqrt(np.sum((c @ Pe @ np.diag(f[j - 1])) ** 2))
    return sigma


# --------------------------------------------------------------------------- Kalman recursion (13), Riccati scan (16)(17)
def kalman_recursion_item(A, C, e, f, Pi0):
    """Backward-Kalman recursion of eq.(13), one item, written out step by step:
        Pi_0 = Xi Xi^T (given as Pi0);   for j = 0 .. T-1:
        L_{j+1}  = -(F_j F_j^T + C_j Pi_j C_j^T)^{-1} C_j Pi_j A_j^T                     [p,n]
        Pi_{j+1} = E_j E_j^T + A_j Pi_j A_j^T + A_j Pi_j C_j^T L_{j+1}                   [n,n]
    with E_j = diag(e[j]), F_j = diag(f[j]) (f > 0).  A[T,n,n], C[T,p,n], e[T,n], f[T,p], Pi0[n,n] symmetric PSD.
    Returns Pi[T+1,n,n] (Pi[j] = Pi_j) and Lt[T,n,p] with Lt[j] = L_{j+1}^T: the gain formed from (A_j, C_j, Pi_j),
    i.e. the one that closes the loop around A_j, A_j + Lt[j] C_j - the array `observer_response` takes (q17)."""
    A, C, e, f, Pi0 = _f64(A), _f64(C), _f64(e), _f64(f), _f64(Pi0)
    T, n, _ = A.shape
    p = C.shape[1]
    Pi = np.empty((T + 1, n, n))
    Lt = np.empty((T, n, p))
    Pi[0] = Pi0
    for j in range(T):
        E = np.diag(e[j])
        F = np.diag(f[j])
        S = F @ F.T + C[j] @ Pi[j] @ C[j].T
        L = -np.linalg.solve(S, C[j] @ Pi[j] @ A[j].T)
        Pi[j + 1] = E @ E.T + A[j] @ Pi[j] @ A[j].T + A[j] @ Pi[j] @ C[j].T @ L
        Lt[j] = L.T
    return Pi, Lt


def kalman_recursion(A, C, e, f, Pi0):
    out = [kalman_recursion_item(A[b], C[b], e[b], f[b], Pi0[b]) for b in range(A.shape[0])]
    return np.stack([o[0] for o in out]), np.stack([o[1] for o in out])


def riccati_combine(x, y):
    """Combination rule (16) of two conditional value functions (:166), x = (A~,D~,P~)_{i,m} and
    y = (A~,D~,P~)_{m,l}, giving (A~,D~,P~)_{i,l}:
        P~_{i,l} = A~_{i,m}^T (I + P~_{m,l} D~_{i,m})^{-1} P~_{m,l} A~_{i,m} + P~_{i,m}
        A~_{i,l} = A~_{m,l} (I + D~_{i,m} P~_{m,l})^{-1} A~_{i,m}
        D~_{i,l} = A~_{m,l} (I + D~_{i,m} P~_{m,l})^{-1} D~_{i,m} A~_{m,l}^T + D~_{m,l}
    (the source prints an unbalanced parenthesis in the first rule; this is the form that follows from eliminating
    the intermediate argument of the two value functions of :166, reading q14)."""
    A1, D1, P1 = x
    A2, D2, P2 = y
    I = np.eye(A1.shape[0])
    G = I + D1 @ P2
    P = A1.T @ np.linalg.solve(G.T, P2 @ A1) + P1
    A = A2 @ np.linalg.solve(G, A1)
    D = A2 @ np.linalg.solve(G, D1) @ A2.T + D2
    return A, D, P


def riccati_scan_item(A, C, e, f, Pi0):
    """Pi_j of eq.(13) through the associative elements of (16)(17): step i contributes
    e_i = (A~ = A_i^T, D~ = C_i^T (F_i F_i^T)^{-1} C_i, P~ = E_i E_i^T), the initial uncertainty contributes
    e_init = (0, 0, Xi Xi^T) ("P~_{1,0} = Xi Xi^T, A~_{1,0} = D~_{1,0} = 0"), and
    Pi_j = P~ part of e_{j-1} (x) e_{j-2} (x) ... (x) e_0 (x) e_init - here folded one element at a time, newest on
    the left; any bracketing gives the same result (the operator is associative; pinned in the tests)."""
    A, C, e, f, Pi0 = _f64(A), _f64(C), _f64(e), _f64(f), _f64(Pi0)
    T, n, _ = A.shape
    Z = np.zeros((n, n))
    acc = (Z, Z, Pi0)
    Pi = np.empty((T + 1, n, n))
    Pi[0] = Pi0
    for i in range(T):
        elem = (A[i].T, C[i].T @ np.diag(1.0 / f[i] ** 2) @ C[i], np.diag(e[i] ** 2))
        acc = riccati_combine(elem, acc)
        Pi[i + 1] = acc[2]
    return Pi


def phi_block(A, t: int, s: int):
    """Single block Phi(t,s) = A_{t-1} A_{t-2} ... A_s of one item (left factors applied last),
    for sampling outputs at sizes where the whole triangle is too big to hold."""
    P = _f64(A[s]).copy()
    for k in range(s + 1, t):
        P = _f64(A[k]) @ P
    return P


# --------------------------------------------------------------------------- tube
def tube_item(A, w):
    """r[T,n]: r_0 = 0, r_t = sum_{s=0}^{t-1} |Phi(t,s)| w_s."""
    T, n, _ = A.shape
    w = _f64(w)
    r = np.zeros((T, n))
    for t, row in phi_rows_item(A):
        acc = np.zeros(n)
        for s in range(t):
            acc = acc + np.abs(row[s]) @ w[s]
        r[t] = acc
    return r


def tube(A, w):
    return np.stack([tube_item(A[b], w[b]) for b in range(A.shape[0])])


def tube_row2norm_item(A, w):
    """tau[T,n]: tau_0 = 0, tau_t[i] = sum_{s=0}^{t-1} sqrt(sum_j (Phi(t,s)[i,j] w_s[j])^2)  -  eq.(12e),
    PAPER.md:147, state-disturbance term with E_s = diag(w_s)."""
    T, n, _ = A.shape
    w = _f64(w)
    tau = np.zeros((T, n))
    for t, row in phi_rows_item(A):
        acc = np.zeros(n)
        for s in range(t):
            PE = row[s] * w[s][None, :]                 # Phi(t,s) E_s
            acc = acc + np.sqrt(np.sum(PE * PE, axis=1))  # row-wise two-norm
        tau[t] = acc
    return tau


def tube_row2norm(A, w):
    return np.stack([tube_row2norm_item(A[b], w[b]) for b in range(A.shape[0])])


def constraint_tightening_item(A, w, Hc):
    """Constraint-tightening margins of eq.(12d), one item, process-disturbance term:
        sigma_0 = 0;   sigma_k[i] = sum_{j=0}^{k-1} || c_{k,i}^T Phi(k,j) E_j ||_2,   k = 1 .. T-1,
    with c_{k,i}^T = Hc[k,i,:] (the state part of constraint row i at step k; Hc[0] is not used), Phi(k,j) the
    system-response blocks of (12c) and E_j = diag(w[j]).  Written in the paper's order: one block, one row, one norm
    at a time.  A[T,n,n], w[T,n], Hc[T,nc,n] -> sigma[T,nc]."""
    A, w, Hc = _f64(A), _f64(w), _f64(Hc)
    T, n, _ = A.shape
    nc = Hc.shape[1]
    Phi = system_response_item(A)
    sigma = np.zeros((T, nc))
    for k in range(1, T):
        for j in range(k):
            PE = Phi[packed_index(k, j)] @ np.diag(w[j])
            for i in range(nc):
                sigma[k, i] += np.sqrt(np.sum((Hc[k, i] @ PE) ** 2))
    return sigma


def constraint_tightening(A, w, Hc):
    return np.stack([constraint_tightening_item(A[b], w[b], Hc[b]) for b in range(A.shape[0])])


def system_response_tube_item(A, w):
    """Phi and r of one item in one pass over the rows (what the fused GPU call returns)."""
    T, n, _ = A.shape
    w = _f64(w)
    Phi = np.empty((T * (T - 1) // 2, n, n))
    r = np.zeros((T, n))
    for t, row in phi_rows_item(A):
        acc = np.zeros(n)
        for s in range(t):
            Phi[packed_index(t, s)] = row[s]
            acc = acc + np.abs(row[s]) @ w[s]
        r[t] = acc
    return Phi, r


# --------------------------------------------------------------------------- adjoint
def adjoint_item(A, B, g):
    """lam[T,n] (lam[t-1] = lam_t), grad_u[T,m], grad_x0[n] for L = sum_{t=1}^{T} l_t(x_t),
    g[t-1] = dl_t/dx_t."""
    A = _f64(A)
    g = _f64(g)
    T, n, _ = A.shape
    lam = np.empty((T, n))
    lam[T - 1] = g[T - 1]                      # lam_T = g_T   (lam_{T+1} = 0, no A_T exists)
    for t in range(T - 1, 0, -1):              # lam_t = A_t^T lam_{t+1} + g_t
        lam[t - 1] = A[t].T @ lam[t] + g[t - 1]
    grad_u = None
    if B is not None:
        B = _f64(B)
        grad_u = np.stack([B[t].T @ lam[t] for t in range(T)])   # B_t^T lam_{t+1}
    grad_x0 = A[0].T @ lam[0]                  # A_0^T lam_1
    return lam, grad_u, grad_x0


def adjoint(A, B, g):
    outs = [adjoint_item(A[b], None if B is None else B[b], g[b]) for b in range(A.shape[0])]
    lam = np.stack([o[0] for o in outs])
    gu = None if B is None else np.stack([o[1] for o in outs])
    gx0 = np.stack([o[2] for o in outs])
    return lam, gu, gx0


# --------------------------------------------------------------------------- error metric
def rel_err(got, ref) -> float:
    """north_star parity metric, per output tensor: max|got - ref| / max|ref|."""
    ref = _f64(ref)
    den = float(np.max(np.abs(ref))) if ref.size else 0.0
    num = float(np.max(np.abs(_f64(got) - ref))) if ref.size else 0.0
    return num / den if den > 0 else num
