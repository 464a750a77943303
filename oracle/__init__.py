"""fp64 CPU oracle for the NEP hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_2107_08119_b200."""
from .nep_oracle import *  # noqa: F401,F403
