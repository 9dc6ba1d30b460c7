"""CPU oracle for the mgrhd source update -- TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  See mgrhd_oracle.cpp for what it computes and how
it is pinned.
"""
from .oracle import (  # noqa: F401
    OracleModel,
    build,
    chi_flux,
    chi_mean,
    free_slopes,
    imex_step_1d,
    transport_add,
    arrowhead_solve,
    lu_solve,
    planck_dY,
    planck_Xi,
    planck_Y,
    planck_Z,
    source_update,
    vP,
)
