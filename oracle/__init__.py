"""CPU oracle of the IMEXLBM hot path — TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_2201_11330_b200.
"""
from .binding import Oracle, lattice, feq, num_threads  # noqa: F401
