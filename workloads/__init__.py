"""Seeded synthetic input generators shared by the oracle tests and the CUDA tests.

This package holds NONE of the method's arithmetic (no rollout, no Phi, no tube, no
adjoint, no Kalman recursion): it only builds the inputs A_t, B_t, c_t, x0, u_t, w_s, g_t and the
observation-model stand-ins C_j, e_j, f_j, Pi_0.  The oracle
(`oracle/`) and the CUDA path (`paper_2606_14188_b200/`) never import each other; both
are fed from here.
"""
from .mass_spring import (  # noqa: F401
    CONFIGS,
    LTVInputs,
    config,
    generate,
    dense_random,
    small_integer,
    observation_model,
)
