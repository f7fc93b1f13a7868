"""The C-ABI library loads, exports every symbol include/ltv_scan.h declares, and validates its arguments on
the host before touching the GPU (no compute calls here: runs without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    import __graft_entry__ as G

    G.build()
    import paper_2606_14188_b200 as lib

    return lib


def test_exports_match_header(L):
    hdr = open(os.path.join(ROOT, "include", "ltv_scan.h")).read()
    declared = set(re.findall(r"LTV_API[^;(]*?\b(ltv_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(L.EXPORTS)
    raw = ctypes.CDLL(L.LIB_PATH)
    for name in declared:
        assert hasattr(raw, name), name


def test_status_strings_and_version(L):
    assert L.lib.ltv_status_string(0) == b"LTV_OK"
    assert L.lib.ltv_status_string(5) == b"LTV_ERR_WORKSPACE_TOO_SMALL"
    assert L.lib.ltv_version() >= 100


def test_block_index_is_column_packed(L):
    T = 7
    seen = []
    for s in range(T - 1):
        for t in range(s + 1, T):
            seen.append(L.ltv_phi_block_index(T, t, s))
    assert seen == list(range(T * (T - 1) // 2))
    assert L.ltv_phi_block_index(T, 3, 3) == -1 and L.ltv_phi_block_index(T, T, 0) == -1


def test_workspace_sizes(L):
    assert L.ltv_scan_workspace_bytes(L.LTV_OP_ROLLOUT, 4, 8, 48, 6) == 0
    n, T, b = 300, 32, 64
    need = L.ltv_scan_workspace_bytes(L.LTV_OP_SYSTEM_RESPONSE_TUBE, b, T, n, 0)
    assert need >= b * (T * (T - 1) // 2) * 2 * n * 4          # two n-tiles of 160 columns
    assert L.ltv_scan_workspace_bytes(L.LTV_OP_SYSTEM_RESPONSE_TUBE, b, T, 301, 0) == 0
    big = L.ltv_scan_workspace_bytes(L.LTV_OP_PIPELINE_HOST, b, T, n, 6)
    assert big > b * (T * (T - 1) // 2) * n * n * 4 + b * T * n * n * 4
    small = L.ltv_scan_workspace_bytes(L.LTV_OP_PIPELINE_HOST_NO_PHI, b, T, n, 6)
    assert b * T * n * n * 4 < small < big - b * (T * (T - 1) // 2) * n * n * 4


def test_host_side_validation_needs_no_gpu(L):
    f = ctypes.c_void_p
    buf = (ctypes.c_float * 64)()
    p = ctypes.cast(buf, f)
    odd = f(ctypes.addressof(buf) + 4)
    r = L.lib.ltv_scan_rollout
    assert r(None, None, None, p, None, p, 1, 1, 4, 0, None, 0, None) == 1          # NULL A
    assert r(p, None, None, p, None, p, 0, 1, 4, 0, None, 0, None) == 2             # batch 0
    assert r(p, None, None, p, None, p, 1, 1, 6, 0, None, 0, None) == 3             # n % 4
    assert r(p, None, None, p, None, p, 1, 1, 8196, 0, None, 0, None) == 3          # n too large
    assert r(odd, None, None, p, None, p, 1, 1, 4, 0, None, 0, None) == 4           # alignment
    s = L.lib.ltv_scan_system_response_tube
    assert s(p, p, p, None, 1, 2, 4, 0, 0, p, 1 << 20, None) == 1                   # NULL r_out
    assert s(p, p, p, p, 1, 2, 4, 3, 0, p, 1 << 20, None) == 2                      # unknown layout
    assert s(p, p, p, p, 1, 2, 4, 0, 2, p, 1 << 20, None) == 2                      # unknown flag
    assert s(p, p, p, p, 1, 2, 4, 0, L.LTV_TUBE_ROW_2NORM, p, 8, None) == 5         # known flag passes on
    for layout in (L.LTV_PHI_ROW_PACKED, L.LTV_PHI_SQUARE_GRID, L.LTV_PHI_COLUMN_PACKED):
        assert s(p, p, p, p, 1, 2, 4, layout, 0, p, 8, None) == 5                   # workspace too small
    assert (L.LTV_PHI_ROW_PACKED, L.LTV_PHI_SQUARE_GRID, L.LTV_PHI_COLUMN_PACKED) == (0, 1, 2)   # 0, 1
    nat = L.ltv_scan_workspace_bytes(L.LTV_OP_SYSTEM_RESPONSE_TUBE, 2, 5, 48, 0)
    rel = L.ltv_scan_workspace_bytes(L.LTV_OP_SYSTEM_RESPONSE_TUBE_RELAYOUT, 2, 5, 48, 0)
    assert rel - nat >= 2 * 10 * 48 * 48 * 4                                        # + a column-packed copy of Phi
    assert L.ltv_phi_block_index_layout(5, 3, 1, L.LTV_PHI_ROW_PACKED) == 4
    assert L.ltv_phi_block_index_layout(5, 3, 1, L.LTV_PHI_SQUARE_GRID) == 16
    assert L.ltv_phi_block_index_layout(5, 3, 1, L.LTV_PHI_COLUMN_PACKED) == L.ltv_phi_block_index(5, 3, 1) == 5
    chunks0 = L.ltv_get_option(L.LTV_OPT_PIPELINE_CHUNKS)
    assert chunks0 == 16                                                           # the documented default
    assert L.ltv_set_option(L.LTV_OPT_PIPELINE_CHUNKS, 2) is None and L.ltv_get_option(L.LTV_OPT_PIPELINE_CHUNKS) == 2
    L.ltv_set_option(L.LTV_OPT_PIPELINE_CHUNKS, chunks0)
    assert L.lib.ltv_set_option(L.LTV_OPT_VECTOR_CLUSTER, 17) == 2 and L.lib.ltv_set_option(9, 1) == 2
    assert L.ltv_get_option(L.LTV_OPT_VECTOR_CLUSTER) == 0 and L.lib.ltv_get_option(9) == -1
    o = L.lib.ltv_scan_observer_response
    assert o(p, None, p, p, p, p, 1, 2, 4, 2, 0, 0, p, 1 << 20, None) == 1              # NULL Lt
    assert o(p, p, p, p, p, p, 1, 2, 4, 0, 0, 0, p, 1 << 20, None) == 2                 # p = 0
    assert o(p, p, p, p, p, p, 1, 2, 4, 33, 0, 0, p, 1 << 20, None) == 3                # p > 32
    assert o(p, p, p, p, p, p, 1, 2, 4, 2, L.LTV_PHI_COLUMN_PACKED, 0, p, 8, None) == 5 # workspace too small
    assert o(p, p, p, p, p, p, 1, 2, 4, 2, L.LTV_PHI_ROW_PACKED, 0, p, 1 << 20, None) == 2   # observer: native layout only
    assert o(p, p, p, p, p, p, 1, 2, 4, 2, L.LTV_PHI_COLUMN_PACKED, 4, p, 1 << 20, None) == 2  # unknown flag
    assert L.ltv_observer_row_floats(300, 6) == 308 and L.ltv_observer_row_floats(48, 4) == 52
    assert L.ltv_scan_workspace_bytes(L.LTV_OP_OBSERVER_RESPONSE, 2, 4, 128, 6) > 0
    k = L.lib.ltv_scan_kalman_gains
    assert k(p, p, p, p, None, p, p, 1, 2, 4, 2, 0, p, 1 << 20, None) == 1              # NULL Pi0
    assert k(p, p, p, p, p, p, p, 1, 2, 4, 0, 0, p, 1 << 20, None) == 2                 # p = 0
    assert k(p, p, p, p, p, p, p, 1, 2, 4, 2, 4, p, 1 << 20, None) == 2                 # unknown flag
    assert k(p, p, p, p, p, p, p, 1, 2, 4, 2, 3, p, 1 << 20, None) == 2                 # scan AND recursion
    assert k(p, p, p, p, p, p, p, 1, 2, 128, 2, 1, p, 1 << 20, None) == 3               # scan path needs n <= 64
    assert k(p, p, p, p, p, p, p, 1, 2, 4, 33, 0, p, 1 << 20, None) == 3                # p > 32
    assert k(p, p, p, odd, p, p, p, 1, 2, 4, 2, 0, p, 1 << 20, None) == 4               # misaligned f
    assert k(p, p, p, p, p, p, p, 1, 2, 4, 2, 0, p, 8, None) == 5                       # workspace too small
    n, T, b = 300, 32, 64
    need = L.ltv_scan_workspace_bytes(L.LTV_OP_KALMAN_GAINS, b, T, n, 6)
    assert 2 * b * n * n * 4 <= need <= 2 * b * n * n * 4 + 2 * b * 6 * n * 4 + 4096    # Abar, Yt, G, K
    assert L.ltv_scan_workspace_bytes(L.LTV_OP_KALMAN_GAINS, b, T, n, 33) == 0
    c = L.lib.ltv_scan_constraint_tightening
    assert c(p, p, None, p, 1, 2, 4, 2, 0, p, 1 << 20, None) == 1                       # NULL Hc
    assert c(p, p, p, p, 1, 2, 4, 0, 0, p, 1 << 20, None) == 2                          # nc = 0
    assert c(p, p, p, p, 1, 2, 4, 2, 0, p, 8, None) == 5                                # workspace too small
    need = L.ltv_scan_workspace_bytes(L.LTV_OP_CONSTRAINT_TIGHTENING, b, T, n, 6)
    assert 2 * b * (T - 1) * 6 * n * 4 <= need <= 2 * b * (T - 1) * 6 * n * 4 + 1024   # two stacks of (T-1) nc rows
    o = L.lib.ltv_scan_output_feedback_response
    assert o(p, p, None, p, p, p, p, p, None, p, 1, 2, 4, 2, 2, 0, p, 1 << 24, None) == 1   # NULL Kfb
    assert o(p, p, p, p, p, p, p, p, None, p, 1, 2, 4, 0, 2, 0, p, 1 << 24, None) == 2      # m = 0
    assert o(p, p, p, p, p, p, p, p, None, p, 1, 2, 4, 2, 40, 0, p, 1 << 24, None) == 3     # p > 32
    assert o(p, p, p, p, p, p, p, p, None, p, 1, 2, 4100, 2, 2, 0, p, 1 << 24, None) == 3   # 2n beyond the scan's limit
    assert o(p, p, p, p, p, p, p, p, None, p, 1, 2, 4, 2, 2, 0, p, 8, None) == 5            # workspace too small
    blk = b * (T * (T - 1) // 2) * n * n * 4
    try:
        L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 1)
        need = L.ltv_scan_workspace_bytes(L.LTV_OP_OUTPUT_FEEDBACK, b, T, n, 0)
        assert need >= 2 * blk                                 # cross scan: Phihat^x and the cross block (Phibar^x sits in the output)
        L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 2)
        assert L.ltv_scan_workspace_bytes(L.LTV_OP_OUTPUT_FEEDBACK, b, T, n, 0) >= need   # gains' sizes unknown: room for either route
        assert L.ltv_scan_workspace_bytes(L.LTV_OP_OUTPUT_FEEDBACK, b, T, n, 9) == need   # m or p > 8: cross scan only
        need = L.ltv_scan_workspace_bytes(L.LTV_OP_OUTPUT_FEEDBACK, b, T, n, 6)
        assert blk <= need < 2 * blk                           # column recursion: Phibar^x + two column buffers of D
    finally:
        L.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 0)
    assert L.lib.ltv_set_option(L.LTV_OPT_OUTPUT_FEEDBACK_ROUTE, 3) == 2
    need48 = L.ltv_scan_workspace_bytes(L.LTV_OP_OUTPUT_FEEDBACK, b, T, 48, 0)
    assert need48 >= 4 * b * (T * (T - 1) // 2) * 48 * 48 * 4  # n < 96: Phi of the 2n-state augmented system
    oc = L.lib.ltv_scan_output_feedback_constraints
    args7 = (p, p, p, p, p, p, p)
    assert oc(*args7, p, p, p, p, p, 1, 2, 4, 2, 2, 3, 0, None, 1 << 24, None) == 1         # NULL workspace
    assert oc(*args7, None, p, p, p, p, 1, 2, 4, 2, 2, 3, 0, p, 1 << 24, None) == 1         # nc > 0 but Hx NULL
    assert oc(*args7, p, p, p, p, p, 1, 2, 4, 0, 2, 3, 0, p, 1 << 24, None) == 2            # m = 0
    assert oc(*args7, p, p, p, p, p, 1, 2, 4, 2, 2, 3, 1, p, 1 << 24, None) == 2            # flags
    assert oc(*args7, p, p, p, p, p, 1, 2, 4, 2, 33, 3, 0, p, 1 << 24, None) == 3           # p > 32
    assert oc(*args7, p, p, p, p, p, 1, 2, 4, 2, 2, 3, 0, p, 8, None) == 5                  # workspace too small
    wsb = L.lib.ltv_scan_output_feedback_constraints_workspace_bytes
    assert wsb(b, T, n, 6, 6) >= b * T * 4 * n * n * 4 + 2 * b * (T - 1) * 12 * 2 * n * 4    # A_aug + two stacks
    assert wsb(b, T, n, 0, 6) == 0 and wsb(b, T, 4100, 6, 6) == 0
    a = L.lib.ltv_scan_adjoint
    assert a(p, None, p, p, p, None, 1, 2, 4, 2, None, 0, None) == 1                # grad_u wanted, B NULL
    assert a(p, p, None, p, None, None, 1, 2, 4, 2, None, 0, None) == 1             # NULL g


def test_valid_call_without_gpu_fails_loudly(L):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    f = ctypes.c_void_p
    buf = (ctypes.c_float * 64)()
    base = (ctypes.addressof(buf) + 15) & ~15
    p = f(base)
    st = L.lib.ltv_scan_rollout(p, None, None, p, None, p, 1, 1, 4, 0, None, 0, None)
    assert st in (6, 7)                                                            # ARCH or CUDA, never OK
