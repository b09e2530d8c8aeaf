"""CPU oracle for the Swendsen-Wang sweep -- TEST INFRASTRUCTURE, not product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  The product (paper_1208_2080_b200) never does.
"""
