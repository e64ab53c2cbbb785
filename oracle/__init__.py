"""CPU oracle of the STREAmS hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
leg may import this package.  It shares no code with paper_2004_02276_b200.
"""
