"""CPU oracle for the COLA hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_2302_00850_b200 and imports nothing from it.
See oracle/cola_oracle.c for the statement of the method and its citations.
"""
from .oracle import *  # noqa: F401,F403
