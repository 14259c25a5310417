"""fp64 CPU oracle of the HASTE hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_2606_01117_b200.
"""
from .oracle import *  # noqa: F401,F403
