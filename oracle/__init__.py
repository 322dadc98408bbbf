"""CPU oracle for the closed-shell (T) energy -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_1609_08094_b200's CUDA path.
"""
