"""Serial fp64 CPU oracle of the DIES IRE hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import it.
"""
