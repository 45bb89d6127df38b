"""CPU oracle for the TRIMEG-C1 marker push -- TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_2606_24327_b200.
"""
from .oracle import Oracle, build_oracle, oracle_threads  # noqa: F401
