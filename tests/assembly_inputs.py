"""Test inputs for eq.(15) with a GENERAL state-feedback response Phibar (not generated from gains): any block-lower-
triangular Phibar^u (diagonal included) with Phibar^x = (I - Z A)^-1 (I + Z B Phibar^u) satisfies the state-feedback
achievability constraint [I - Z A, -Z B][Phibar^x; Phibar^u] = I of (12c), and Phibar^x(k,k) = I.  Test infrastructure
(imports the oracle's shift operator); fp64 throughout, the callers round to fp32 once."""
import numpy as np

from oracle import ltv_oracle as O


def general_phibar(A, B, seed, scale=0.3):
    """A[T,n,n], B[T,n,m] -> dense (PbX [T n, T n], PbU [T m, T n]) in fp64."""
    A, B = np.asarray(A, dtype=np.float64), np.asarray(B, dtype=np.float64)
    T, n, m = B.shape
    rng = np.random.default_rng(seed)
    PbU = np.zeros((T * m, T * n))
    for k in range(T):
        for j in range(k + 1):
            PbU[k * m:(k + 1) * m, j * n:(j + 1) * n] = scale * rng.normal(0.0, 1.0 / np.sqrt(n), (m, n))
    ZB = np.zeros((T * n, T * m))
    for t in range(T - 1):
        ZB[(t + 1) * n:(t + 2) * n, t * m:(t + 1) * m] = B[t]
    PbX = np.linalg.solve(np.eye(T * n) - O.shift_operator(A), np.eye(T * n) + ZB @ PbU)
    return PbX, PbU


def observer_operators(A, Lt, C):
    """Dense Phihat^x [T n, T n] (identity diagonal) and Phihat^y [T n, T p] (the shifted-gain form of q20 / q21)."""
    A, Lt, C = [np.asarray(a, dtype=np.float64) for a in (A, Lt, C)]
    T, n, _ = A.shape
    p = C.shape[1]
    blocks = O.observer_response_item(A, Lt, C)[0]
    PhX = np.eye(T * n)
    for t in range(1, T):
        for s in range(t):
            PhX[t * n:(t + 1) * n, s * n:(s + 1) * n] = blocks[O.packed_index(t, s)]
    PhY = np.zeros((T * n, T * p))
    for j in range(1, T):
        PhY[:, j * p:(j + 1) * p] = PhX[:, j * n:(j + 1) * n] @ Lt[j - 1]
    return PhX, PhY


def blk(D, k, j, r, c):
    return D[k * r:(k + 1) * r, j * c:(j + 1) * c]
