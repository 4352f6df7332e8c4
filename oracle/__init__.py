"""CPU oracle for the arXiv 2311.15088 particle pipeline -- TEST INFRASTRUCTURE ONLY (see ref.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
"""
