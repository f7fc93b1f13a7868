"""Seeded semi-implicit mass-spring rope / cloth LTV workloads (BASELINE.json `configs[0..4]`).

The paper ("linearizations of the dynamics ... about the nominal trajectory") gets its
A_t, B_t from the implicit-differentiation Jacobians (8)(9) of a simulator that is not
in the container.  BASELINE.json replaces them with this generator; DESIGN.md "Input recipe" lists the
readings (q6-q13 of SURVEY.md section 8c) taken here.  Only INPUTS are built here - nothing of the method.

State ordering: x = [p_0 .. p_{N-1}, v_0 .. v_{N-1}], three floats per node, n = 6N.
    A_t = [[I - dt^2 L_t, dt I], [-dt L_t, (1 - dt c) I]],   L_t = (weighted graph Laplacian) (x) I_3
    B   : grasp q on node a, axis d: column 3q+d; row 3a+d gets dt^2, row 3N+3a+d gets dt
    c_t : -9.81*dt on the z-velocity rows 3N+3i+2
Arrays are built in fp64 and cast ONCE to fp32; that fp32 array is what both the oracle (promoted to fp64)
and the GPU consume.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 20260614
DT = 0.01
DAMP = 0.5
GRAV = 9.81
SPACING = 0.02

# index k-1 <-> config Ck of SURVEY.md section 8 / BASELINE.json configs[k-1]
CONFIGS = [
    dict(name="C1_rope8", graph="chain", N=8, m=6, T=16, batch=1),
    dict(name="C2_rope50", graph="chain", N=50, m=6, T=32, batch=64),
    dict(name="C3_cloth10", graph="grid", G=10, N=100, m=6, T=32, batch=16),
    dict(name="C4_cloth20", graph="grid", G=20, N=400, m=12, T=16, batch=4),
    dict(name="C5_rope30", graph="chain", N=30, m=6, T=64, batch=64),
]


def config(index: int, **overrides) -> dict:
    """Config `index` in 0..4 (C1..C5) with n = 6N filled in; overrides e.g. batch=256, T=8."""
    cfg = dict(CONFIGS[index])
    cfg["index"] = index
    cfg.update(overrides)
    cfg["n"] = 6 * cfg["N"]
    cfg.setdefault("seed", SEED_BASE + index)
    return cfg


@dataclass
class LTVInputs:
    A: np.ndarray   # [batch, T, n, n] fp32, A[b,t,i,j] = d x_{t+1,i} / d x_{t,j}
    B: np.ndarray   # [batch, T, n, m]
    c: np.ndarray   # [batch, T, n]
    x0: np.ndarray  # [batch, n]
    u: np.ndarray   # [batch, T, m]
    w: np.ndarray   # [batch, T, n]  (w_s >= 0)
    g: np.ndarray   # [batch, T, n]  g[b, t-1] = dL/dx_t
    meta: dict = field(default_factory=dict)

    @property
    def shape(self):
        b, T, n, _ = self.A.shape
        return b, T, n, self.B.shape[-1]

    def item_slice(self, b0: int, b1: int) -> "LTVInputs":
        s = slice(b0, b1)
        return LTVInputs(self.A[s], self.B[s], self.c[s], self.x0[s], self.u[s], self.w[s], self.g[s],
                         dict(self.meta))


def _edges(cfg):
    """(i, j, kind) arrays; kind 0 = structural / rope, 1 = shear."""
    if cfg["graph"] == "chain":
        N = cfg["N"]
        i = np.arange(N - 1)
        return i, i + 1, np.zeros(N - 1, dtype=np.int64)
    G = cfg["G"]
    nid = lambda r, c: r * G + c
    ei, ej, kind = [], [], []
    for r in range(G):            # horizontal
        for c in range(G - 1):
            ei.append(nid(r, c)); ej.append(nid(r, c + 1)); kind.append(0)
    for r in range(G - 1):        # vertical
        for c in range(G):
            ei.append(nid(r, c)); ej.append(nid(r + 1, c)); kind.append(0)
    for r in range(G - 1):        # both diagonals of every cell
        for c in range(G - 1):
            ei.append(nid(r, c)); ej.append(nid(r + 1, c + 1)); kind.append(1)
            ei.append(nid(r, c + 1)); ej.append(nid(r + 1, c)); kind.append(1)
    return np.array(ei), np.array(ej), np.array(kind)


def _grasp_nodes(cfg):
    if cfg["graph"] == "chain":
        return [0, cfg["N"] - 1]
    G = cfg["G"]
    corners = [0, G - 1, (G - 1) * G, G * G - 1]
    return corners[: cfg["m"] // 3]


def _rest_positions(cfg):
    N = cfg["N"]
    p = np.zeros((N, 3))
    if cfg["graph"] == "chain":
        p[:, 0] = SPACING * np.arange(N)
    else:
        G = cfg["G"]
        r, c = np.divmod(np.arange(N), G)
        p[:, 0] = SPACING * c
        p[:, 1] = SPACING * r
    return p


def generate(cfg: dict, item_range=None, chunk: int = 256) -> LTVInputs:
    """Build the fp32 inputs of `cfg` (see `config`).  `item_range=(b0,b1)` builds only those batch
    items; the random draws are always made for the whole batch first so item b is identical whichever
    range it is built in (rank sharding, bounded CPU samples)."""
    N, n, m, T, batch = cfg["N"], cfg["n"], cfg["m"], cfg["T"], cfg["batch"]
    rng = np.random.default_rng(cfg["seed"])
    ei, ej, kind = _edges(cfg)
    E = len(ei)
    if cfg["graph"] == "chain":
        k_lo, k_hi = np.full(E, 50.0), np.full(E, 150.0)
    else:
        k_lo = np.where(kind == 0, 100.0, 20.0)
        k_hi = np.where(kind == 0, 200.0, 60.0)

    # fixed draw order: k_e, eps, x0-noise, u, w, g  (one vectorised draw per array)
    k_e = k_lo + (k_hi - k_lo) * rng.random((batch, E))
    eps = rng.uniform(-1.0, 1.0, (batch, T, E))
    x0_noise = rng.normal(0.0, 1e-3, (batch, n))
    u = rng.normal(0.0, 0.1, (batch, T, m))
    w = rng.uniform(0.0, 1e-3, (batch, T, n))
    g = rng.normal(0.0, 1.0, (batch, T, n))

    b0, b1 = (0, batch) if item_range is None else item_range
    nb = b1 - b0

    x0 = np.concatenate([_rest_positions(cfg).reshape(-1), np.zeros(3 * N)])[None, :] + x0_noise[b0:b1]

    Bmat = np.zeros((n, m))
    for q, a in enumerate(_grasp_nodes(cfg)):
        for d in range(3):
            Bmat[3 * a + d, 3 * q + d] = DT * DT
            Bmat[3 * N + 3 * a + d, 3 * q + d] = DT
    cvec = np.zeros(n)
    cvec[3 * N + 2 :: 3] = -GRAV * DT

    A32 = np.empty((nb, T, n, n), dtype=np.float32)
    absD = np.zeros((E, N))
    absD[np.arange(E), ei] = 1.0
    absD[np.arange(E), ej] = 1.0
    idN = np.arange(N)
    for c0 in range(0, nb, chunk):
        c1 = min(nb, c0 + chunk)
        k = k_e[b0 + c0 : b0 + c1, None, :] * (1.0 + 0.1 * eps[b0 + c0 : b0 + c1])  # [cb,T,E]
        cb = c1 - c0
        Lg = np.zeros((cb, T, N, N))
        Lg[:, :, ei, ej] = -k
        Lg[:, :, ej, ei] = -k
        Lg[:, :, idN, idN] = k @ absD                                               # weighted degree
        # A as [cb, T, 2, N, 3, 2, N, 3]  (block-row, node, axis, block-col, node, axis)
        Ab = np.zeros((cb, T, 2, N, 3, 2, N, 3))
        for d in range(3):
            Ab[:, :, 0, :, d, 0, :, d] = -DT * DT * Lg
            Ab[:, :, 0, idN, d, 0, idN, d] += 1.0
            Ab[:, :, 0, idN, d, 1, idN, d] = DT
            Ab[:, :, 1, :, d, 0, :, d] = -DT * Lg
            Ab[:, :, 1, idN, d, 1, idN, d] = 1.0 - DT * DAMP
        A32[c0:c1] = Ab.reshape(cb, T, n, n).astype(np.float32)
        del Ab, Lg

    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    meta = dict(cfg)
    meta["item_range"] = (b0, b1)
    return LTVInputs(
        A=A32,
        B=f32(np.broadcast_to(Bmat, (nb, T, n, m))),
        c=f32(np.broadcast_to(cvec, (nb, T, n))),
        x0=f32(x0),
        u=f32(u[b0:b1]),
        w=f32(w[b0:b1]),
        g=f32(g[b0:b1]),
        meta=meta,
    )


def dense_random(batch: int, T: int, n: int, m: int, seed: int, scale: float = 0.5) -> LTVInputs:
    """Non-config parity workload: dense A_t = I + N(0, scale/sqrt(n)), random B_t, c_t (general LTV).
    The paper's real Jacobians are dense ((8)(9); 'dense matrix multiplications',
    PAPER.md:166), so no kernel may rely on the mass-spring sparsity pattern."""
    rng = np.random.default_rng(seed)
    A = np.eye(n)[None, None] + rng.normal(0.0, scale / np.sqrt(n), (batch, T, n, n))
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return LTVInputs(
        A=f32(A),
        B=f32(rng.normal(0.0, 1.0, (batch, T, n, m))),
        c=f32(rng.normal(0.0, 0.1, (batch, T, n))),
        x0=f32(rng.normal(0.0, 1.0, (batch, n))),
        u=f32(rng.normal(0.0, 0.1, (batch, T, m))),
        w=f32(rng.uniform(0.0, 1e-3, (batch, T, n))),
        g=f32(rng.normal(0.0, 1.0, (batch, T, n))),
        meta=dict(name="dense_random", n=n, m=m, T=T, batch=batch, seed=seed),
    )


def small_integer(batch: int, T: int, n: int, m: int, seed: int, density: float = 0.15) -> LTVInputs:
    """Integer-valued workload: sparse entries in {-1, 0, 1}, integer B, c, x0, u, w, g.  All partial
    products stay far below 2^24 at the sizes the tests use, so fp32 / 3xTF32 arithmetic is EXACT and the
    GPU must reproduce the fp64 result bit for bit (SURVEY.md section 8c pin vii)."""
    rng = np.random.default_rng(seed)
    mask = rng.random((batch, T, n, n)) < density / max(1.0, n / 16.0)
    vals = rng.integers(-1, 2, (batch, T, n, n))
    A = np.where(mask, vals, 0).astype(np.float64)
    idx = np.arange(n)
    A[:, :, idx, idx] = 1.0
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return LTVInputs(
        A=f32(A),
        B=f32(rng.integers(-1, 2, (batch, T, n, m))),
        c=f32(rng.integers(-1, 2, (batch, T, n))),
        x0=f32(rng.integers(-2, 3, (batch, n))),
        u=f32(rng.integers(-1, 2, (batch, T, m))),
        w=f32(rng.integers(0, 3, (batch, T, n))),
        g=f32(rng.integers(-1, 2, (batch, T, n))),
        meta=dict(name="small_integer", n=n, m=m, T=T, batch=batch, seed=seed),
    )


def observation_model(batch: int, T: int, n: int, p: int, seed: int, kind: str = "track") -> dict:
    """Inputs of the output-feedback stage (eq.(13)): observation Jacobians C_j, the disturbance
    scalings E_j = diag(e_j), F_j = diag(f_j) and the initial uncertainty Pi_0 = Xi Xi^T.  The paper's C, E, F, Xi come
    from its perception stack and calibration, which are not in the container; stand-ins:
      kind "track"  C_j selects p position coordinates spread evenly over the first n/2 state entries (tracked points
                    on the object, constant in j but stored per step)
      kind "dense"  C_j ~ N(0, 1/sqrt(n)) i.i.d. per step
      e ~ U[2e-4, 1e-3] (process), f ~ U[1e-3, 5e-3] (observation), Xi = 1e-2 (I + 0.1 N(0, 1/sqrt(n))).
    Returns fp32 arrays C[batch,T,p,n], e[batch,T,n], f[batch,T,p], Pi0[batch,n,n] (Pi0 exactly symmetric)."""
    rng = np.random.default_rng(seed)
    if kind == "track":
        half = max(p, n // 2)
        cols = (np.arange(p) * half) // p
        C = np.zeros((batch, T, p, n))
        C[:, :, np.arange(p), cols] = 1.0
    elif kind == "dense":
        C = rng.normal(0.0, 1.0 / np.sqrt(n), (batch, T, p, n))
    else:
        raise ValueError(kind)
    e = rng.uniform(2e-4, 1e-3, (batch, T, n))
    f = rng.uniform(1e-3, 5e-3, (batch, T, p))
    Xi = 1e-2 * (np.eye(n)[None] + 0.1 * rng.normal(0.0, 1.0 / np.sqrt(n), (batch, n, n)))
    Pi0 = (Xi @ np.swapaxes(Xi, 1, 2)).astype(np.float32)
    Pi0 = np.ascontiguousarray(0.5 * (Pi0 + np.swapaxes(Pi0, 1, 2)))
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return dict(C=f32(C), e=f32(e), f=f32(f), Pi0=f32(Pi0))
