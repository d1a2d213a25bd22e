"""CPU oracle for arXiv 2004.00923's hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2004_00923_b200 and shares no code with it.
"""
from .holo_oracle import *  # noqa: F401,F403
