"""CPU oracle -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_1312_2234_b200 (the CUDA path) except the
seeded input generators in paper_1312_2234_b200.workloads, which hold no method arithmetic.
"""
