"""B200-native LTV-scan hot path of CORD-SLS (arxiv 2606.14188): rollout, system response + tube, adjoint.
Thin ctypes binding over the C-ABI library built from csrc/ (see include/ltv_scan.h)."""
from .binding import (  # noqa: F401
    EXPORTS,
    LIB_PATH,
    LTV_OP_ADJOINT,
    LTV_OP_PIPELINE_HOST,
    LTV_OP_ROLLOUT,
    LTV_OP_SYSTEM_RESPONSE_TUBE,
    LTV_PHI_COLUMN_PACKED,
    LtvError,
    lib,
    ltv_launch_count,
    ltv_phi_block_index,
    ltv_scan_adjoint,
    ltv_scan_pipeline_host,
    ltv_scan_rollout,
    ltv_scan_system_response_tube,
    ltv_scan_workspace_bytes,
)
