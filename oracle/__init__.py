"""fp64 CPU oracle (TEST INFRASTRUCTURE ONLY — see oracle/opmc.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  The product (paper_1409_8336_b200) never does.
"""
from .binding import Oracle, build_oracle, philox4x32_10  # noqa: F401
