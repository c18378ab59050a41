"""The oracle: TEST INFRASTRUCTURE, not the product.

A plain fp64 CPU implementation (oracle/wcoracle.c, naive loops) of what the hot path of
arXiv:1011.3318 computes, written from the paper and BASELINE.json:north_star.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import it.
It shares no code with paper_1011_3318_b200/ and neither imports the other.
"""
from .wcoracle import *  # noqa: F401,F403
