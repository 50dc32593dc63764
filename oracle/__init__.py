"""CPU oracle of the ILE factored-likelihood hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_2210_07912_b200 and never imports it.
See rift_oracle.c for the arithmetic and its citations; this file only builds and marshals.
"""
from .oracle import *  # noqa: F401,F403
from . import precompute_oracle  # noqa: F401,E402  (NEXT-3, Eq. (D4a-c))
