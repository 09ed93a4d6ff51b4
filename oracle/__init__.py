"""CPU oracle for the NSPT series star-product and the TEK staple.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2001_02835_b200 (the CUDA path) and never
imports it.  See oracle/nspt_oracle.c (the arithmetic) and oracle/nspt_oracle.py (ctypes
wrapper, dagger, literal staple of eq. 2.3, error bounds).
"""
from .nspt_oracle import (  # noqa: F401
    build,
    num_threads,
    series_mul,
    series_mul_rows,
    dagger,
    staple,
    series_exp,
    exp_bound,
    force,
    product_bound,
    staple_bound,
    per_order_error,
)
