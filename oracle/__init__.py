"""CPU oracle (TEST INFRASTRUCTURE — see oracle/tpt_oracle.h).

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline/--impl reference legs.
"""
from .binding import (  # noqa: F401
    DIRS_XYZ,
    DIRS_YZ,
    DIRS_Z,
    OraclePlan,
    apply_operator_flux,
    dense_solve_3d,
    divergence,
    face_shapes,
    gradient,
    project,
    eig_1d,
    num_threads,
    operator_1d,
    residual_norms,
    symmetrize_1d,
)
