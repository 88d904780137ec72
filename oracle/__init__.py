"""CPU oracle of the pre-positioning hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_2606_29565_b200 and neither imports the other.
Parity status: every oracle function is pinned (tests/test_oracle_*.py); none is "parity unpinned".
"""
