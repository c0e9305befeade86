"""FP64 CPU oracle for RM synthesis (arxiv 1810.06250).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_1810_06250_b200.
"""
from .oracle import (  # noqa: F401
    build, lambda_sq, plan_scalars, rmsf, synth_naive, synth_table,
    tolerance_scale, peaks, Plan, make_plan, rmclean, rmsf_double_width,
)
