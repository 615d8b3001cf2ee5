"""CPU oracle for the RGF sweep -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares nothing with paper_1107_5300_b200 (the CUDA path).
"""
