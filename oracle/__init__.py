"""CPU oracle for the geometric-network step (TEST INFRASTRUCTURE, see gn_oracle.c).

This package is for tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs only, and it never touches the CUDA package.
"""
from .binding import Oracle, build_lib, lib, CLASS_FIELDS  # noqa: F401
