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
  observer_response  PhiX(k,k) = I; PhiX(k,j) = PhiX(k,j+1) (A_j + L_j^T C_j);     PAPER.md:157-160 eq.(14), read with
                   PhiY(k,j) = PhiX(k,j) L_j^T,  0 <= j < k <= T-1                 k-independent gains L_j (:177; SURVEY
                                                                     8f NEXT-1, reading q15)
  adjoint          lam_T = g_T; lam_t = A_t^T lam_{t+1} + g_t;       PAPER.md:106-110 eq.(10) chained
                   grad_u[t] = B_t^T lam_{t+1}; grad_x0 = A_0^T lam_1   over the horizon; north_star (iii)

Index conventions (DESIGN.md "Readings" q1, q2, q5): nodes 0 <= s < t <= T-1, P = T(T-1)/2 blocks,
packed block index p = t(t-1)/2 + s; X[t] = x_{t+1}; g[t-1] = g_t; lam[t-1] = lam_t; lam_{T+1} = 0.

Inputs are the fp32 arrays handed to the GPU, promoted to fp64 here (never a separate fp64 copy).

Pins (tests/test_oracle_pins.py): every function below is pinned by closed forms, the defining identity
(12c), brute force on tiny inputs, a hand-computed worked example (tests/golden/hand_example.txt) and the
tube-containment / adjoint dot-product invariants.  Nothing in this file is "parity unpinned".
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


def observer_response_item(A, Lt, C):
    """Closed-loop observer propagation of one item, eq.(14) in the paper's own order: for every
    k, PhiX(k,k) = I and, for j = k-1 down to 0, PhiX(k,j) = PhiX(k,j+1) (A_j + L_j^T C_j) (RIGHT multiplication),
    PhiY(k,j) = PhiX(k,j) L_j^T.  Lt[j] = L_j^T [n,p], C[j] [p,n].  Returns packed PhiX[P,n,n], PhiY[P,n,p]."""
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
            PhiY[packed_index(k, j)] = X @ Lt[j]
    return PhiX, PhiY


def observer_response(A, Lt, C):
    out = [observer_response_item(A[b], Lt[b], C[b]) for b in range(A.shape[0])]
    return np.stack([o[0] for o in out]), np.stack([o[1] for o in out])


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
