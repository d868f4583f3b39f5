"""CPU oracle for the photon tracer: TEST INFRASTRUCTURE, not product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  See oracle/rt_oracle.cpp for what it computes and
the passages of PAPER.md it follows.
"""
from .binding import *  # noqa: F401,F403
