"""fp64 CPU oracle for the CHIMERA-2.0 hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares nothing with paper_2504_02034_b200 (see chim_oracle.c header).
"""
from .binding import *  # noqa: F401,F403
