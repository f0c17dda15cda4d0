"""CPU oracle for the HORIZON GRMHD substep -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_1102_5202_b200 and neither imports the other.
"""
from .binding import Oracle, OracleParams, lib  # noqa: F401
