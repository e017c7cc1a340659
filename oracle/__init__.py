"""CPU fp64 oracle for the LinMin hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
import this package.  It shares no code with paper_1402_2518_b200/csrc and never imports it.
See oracle/linmin_oracle.c for what is computed and the PAPER.md passages it follows.
"""
from .oracle import OracleResult, build, solve, max_threads  # noqa: F401
