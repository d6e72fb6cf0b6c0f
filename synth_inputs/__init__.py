"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

Holds none of the method's arithmetic (no rates, RHS, Jacobian, LU or integrator).
`configs.CONFIGS` lists BASELINE.json's five configurations.
"""
from .mechanism import (mech_h2, mech_c1, mech_c4, mech_decay, make_mechanism, mech_h2co, mech_c1_irrev,  # noqa: F401
                        mech_rowkinds, with_row_kinds,
                        PLAIN, THREE_BODY, LINDEMANN, TROE)
from .states import ignition_states, dirichlet_states, paper_rhs_states, P_ATM  # noqa: F401
from .configs import CONFIGS, make_config  # noqa: F401
