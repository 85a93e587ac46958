"""CPU oracle of the coupled ACM LB step -- test infrastructure, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
leg may import this package.  It imports nothing from paper_2012_06144_b200.
"""
from .oracle import Oracle, lattice  # noqa: F401
