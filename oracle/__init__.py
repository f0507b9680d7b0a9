"""CPU oracle of the implicit-filter hot path -- TEST INFRASTRUCTURE, not product code.

Written from /root/reference/PAPER.md (see implicit_filter_oracle.c for the citations).  May be imported
only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
"""
from .oracle import GAMMA, TOL, OracleMesh, build, filter_and_spectrum, spectrum, threads

__all__ = ["GAMMA", "TOL", "OracleMesh", "build", "filter_and_spectrum", "spectrum", "threads"]
