"""CPU oracle for the hydro hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_2007_05218_b200 (the CUDA
path) and neither imports the other.
"""
