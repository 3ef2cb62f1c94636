"""CPU oracle of the per-zone burn -- TEST INFRASTRUCTURE ONLY (see bz_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this package.  It never imports paper_1711_06203_b200 and vice versa.
"""
from .oracle import (  # noqa: F401
    burn, rates, oexp, olog, lu_factor, lu_solve, bdf_coeffs, wrms, max_threads, interchanges, event_counts, COUNTER_NAMES,
    build_d, TRACE_FIELDS,
)
