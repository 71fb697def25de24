"""CPU oracle for the SFFT subtraction path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports the CUDA package and shares no code
with it.  See oracle/sfft_oracle.c for what is computed and which passage each
function follows.
"""
from .sfft_oracle import (  # noqa: F401
    OracleError,
    build,
    build_system,
    build_system_dense,
    convolve_stamp,
    convolve_stamp_at,
    coord,
    design_matrix,
    lag_sum,
    num_poly,
    num_threads,
    num_unknowns,
    poly_image,
    poly_index,
    solve,
    subtract,
    subtract_at,
    system_entry,
    weighted_image,
)
