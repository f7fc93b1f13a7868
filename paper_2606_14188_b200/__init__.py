"""B200-native LTV-scan hot path of CORD-SLS (arxiv 2606.14188): rollout, system response + tube, adjoint.
Thin ctypes binding over the C-ABI library built from csrc/ (see include/ltv_scan.h).

The binding (and with it libltvscan.so) is loaded on first attribute access, so that
`paper_2606_14188_b200.build` can be imported to compile the library before it exists.  There is no CPU
fallback: touching any API name without the built library raises ImportError."""
import importlib

_API = (
    "EXPORTS", "LIB_PATH", "LTV_OP_ADJOINT", "LTV_OP_PIPELINE_HOST", "LTV_OP_PIPELINE_HOST_NO_PHI", "LTV_OP_OBSERVER_RESPONSE",
    "LTV_OP_ROLLOUT",
    "LTV_OP_SYSTEM_RESPONSE_TUBE", "LTV_PHI_COLUMN_PACKED", "LTV_PHI_ROW_PACKED", "LTV_PHI_SQUARE_GRID", "LTV_OP_SYSTEM_RESPONSE_TUBE_RELAYOUT",
    "ltv_phi_block_index_layout", "LTV_TUBE_ROW_2NORM", "LTV_OBSERVER_SHIFTED_GAIN", "PROFILE_CLASSES", "LtvError", "lib",
    "ltv_launch_count", "ltv_phi_block_index", "ltv_profile_collect", "ltv_profile_enable",
    "ltv_scan_adjoint", "ltv_scan_pipeline_host", "ltv_scan_rollout", "ltv_scan_system_response_tube",
    "ltv_scan_workspace_bytes", "ltv_scan_observer_response", "ltv_observer_row_floats", "ltv_scan_kalman_gains",
    "ltv_set_option", "ltv_get_option", "ltv_scan_all", "ltv_scan_all_is_fused", "ltv_scan_rollout_adjoint", "ltv_scan_output_feedback_constraints", "LTV_OPT_VECTOR_CLUSTER", "LTV_OPT_PIPELINE_CHUNKS", "LTV_OPT_OUTPUT_FEEDBACK_ROUTE",
    "LTV_OP_KALMAN_GAINS", "LTV_OP_OUTPUT_FEEDBACK", "ltv_scan_output_feedback_response", "LTV_KALMAN_SCAN", "LTV_KALMAN_RECURSION", "LTV_OP_CONSTRAINT_TIGHTENING", "ltv_scan_constraint_tightening",
    "ltv_static_scratch_bytes", "ltv_scan_system_response_tube_static", "LTV_ERR_STATIC_SCRATCH_LIMIT",
    "ltv_scan_output_feedback_assemble", "ltv_scan_operator_constraint_margins",
    "ltv_phi_row_shard_blocks", "ltv_phi_row_shard_block_index", "ltv_scan_system_response_tube_rows",
)
__all__ = list(_API)


def __getattr__(name):
    if name in _API:
        binding = importlib.import_module(".binding", __name__)
        return getattr(binding, name)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
