"""CPU oracle for the geometric-network step (TEST INFRASTRUCTURE, see gn_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_0908_3934_b200.
"""
from .binding import Oracle, build_lib, lib, CLASS_FIELDS  # noqa: F401
