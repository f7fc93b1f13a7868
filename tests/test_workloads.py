"""The seeded generators: shapes, structure (readings q6-q13 in DESIGN.md), determinism."""
import numpy as np
import pytest

from workloads import CONFIGS, config, dense_random, generate, small_integer
from workloads.mass_spring import _edges


def test_config_table_matches_baseline_json():
    exp = [(48, 6, 16, 1), (300, 6, 32, 64), (600, 6, 32, 16), (2400, 12, 16, 4), (180, 6, 64, 64)]
    for k, e in enumerate(exp):
        c = config(k)
        assert (c["n"], c["m"], c["T"], c["batch"]) == e
    assert len(CONFIGS) == 5


def test_edge_counts():
    assert len(_edges(config(0))[0]) == 7
    assert len(_edges(config(1))[0]) == 49
    ei, ej, kind = _edges(config(2))
    assert (kind == 0).sum() == 180 and (kind == 1).sum() == 162
    ei, ej, kind = _edges(config(3))
    assert (kind == 0).sum() == 760 and (kind == 1).sum() == 722
    assert len(set(zip(ei.tolist(), ej.tolist()))) == len(ei)


@pytest.mark.parametrize("k,over", [(0, {}), (2, dict(batch=2, T=3))])
def test_structure_of_A_B_c(k, over):
    cfg = config(k, **over)
    W = generate(cfg)
    b, T, n, m = W.shape
    N = cfg["N"]
    assert W.A.dtype == np.float32 and W.A.shape == (cfg["batch"], cfg["T"], n, n)
    A = W.A.astype(np.float64)
    dt, damp = 0.01, 0.5
    # blocks: top-right dt I, bottom-right (1 - dt c) I, bottom-left = (top-left - I)/dt
    assert np.allclose(A[:, :, :3 * N, 3 * N:], dt * np.eye(3 * N), atol=1e-9)
    assert np.allclose(A[:, :, 3 * N:, 3 * N:], (1 - dt * damp) * np.eye(3 * N), atol=1e-7)
    TL = A[:, :, :3 * N, :3 * N] - np.eye(3 * N)
    assert np.allclose(TL / dt, A[:, :, 3 * N:, :3 * N], atol=1e-4)
    L = -A[:, :, 3 * N:, :3 * N] / dt                     # L (x) I3
    assert np.allclose(L, np.swapaxes(L, -1, -2), atol=1e-5)
    assert np.allclose(L.sum(-1), 0, atol=2e-3)           # rows of a Laplacian sum to zero
    Lr = L.reshape(b, T, N, 3, N, 3)
    for d in range(3):
        for e in range(3):
            if d != e:
                assert np.all(Lr[:, :, :, d, :, e] == 0)  # Kronecker with I3
    # per-step jitter is within +-10 % of the step mean and really varies with t and b
    offd = Lr[:, :, 0, 0, 1, 0]
    assert np.all(offd < 0) and np.ptp(offd) > 0
    # B: dt^2 on position rows, dt on velocity rows of the grasped nodes; c: gravity on z velocities
    Bm = W.B[0, 0].astype(np.float64)
    assert np.count_nonzero(Bm) == 2 * m
    assert np.isclose(Bm[0, 0], dt * dt) and np.isclose(Bm[3 * N, 0], dt)
    cv = W.c[0, 0].astype(np.float64)
    assert np.allclose(cv[3 * N + 2::3], -9.81 * dt) and np.count_nonzero(cv) == N
    assert np.all(W.w >= 0) and W.w.max() <= 1e-3


def test_deterministic_and_item_range_consistent():
    cfg = config(4, batch=6, T=4)
    W = generate(cfg)
    W2 = generate(cfg)
    assert np.array_equal(W.A, W2.A) and np.array_equal(W.g, W2.g)
    Ws = generate(cfg, item_range=(2, 5))
    for name in ("A", "B", "c", "x0", "u", "w", "g"):
        assert np.array_equal(getattr(Ws, name), getattr(W, name)[2:5]), name
    Wc = generate(cfg, chunk=4)
    assert np.array_equal(Wc.A, W.A)
    assert not np.array_equal(generate(config(4, batch=6, T=4, seed=1)).A, W.A)


def test_rest_state_spacing():
    W = generate(config(2, batch=1, T=1))
    p = W.x0[0, :300].reshape(100, 3)
    assert abs(p[1, 0] - p[0, 0] - 0.02) < 5e-3 and abs(p[10, 1] - p[0, 1] - 0.02) < 5e-3


def test_aux_workloads():
    D = dense_random(2, 3, 8, 2, seed=5)
    assert D.A.shape == (2, 3, 8, 8) and np.count_nonzero(D.A) == D.A.size
    I = small_integer(2, 4, 16, 2, seed=5)
    assert np.array_equal(I.A, np.round(I.A)) and np.abs(I.A).max() == 1
