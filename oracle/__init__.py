"""CPU oracle (test infrastructure, NOT the product).  See oracle/sht_oracle.cpp for what it computes and why.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.
It imports nothing from paper_2311_14670_b200.
"""
from .oracle import *  # noqa: F401,F403
