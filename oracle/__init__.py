"""CPU oracle for the SFFT hot path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2109_09334_b200`` (the CUDA path) and neither imports the other.

The arithmetic lives in ``sfft_oracle.c`` (plain C, direct pixel sums, no FFT); this
file only compiles it with gcc and marshals numpy arrays through ctypes.
"""
from .binding import (  # noqa: F401
    POLY, BSPLINE, build_library, num_threads, num_terms, num_axis, terms, axis_table,
    num_unknowns, design_matrix, gram, normal_bruteforce, diag_and_rhs, lag_tables, gather,
    normal_from_lags, solve, difference, difference_at, corr_diff_one, weighted_ref,
    cpr_num_unknowns, cpr_constrain, cpr_expand, mask_fill, rect_select, rect_expand,
)
from . import decorr  # noqa: F401,E402   (NEXT-3, App. C; numpy)
