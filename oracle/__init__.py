"""CPU oracle for the GRay photon-geodesic hot path.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_1303_5057_b200.
"""
from .gray_oracle import *  # noqa: F401,F403
