"""CPU oracle for the arXiv 1005.3276 hot path.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_1005_3276_b200/csrc.
"""
