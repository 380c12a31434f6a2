"""fp64 CPU oracle for the TF-regularised CBCT hot path.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_1008_2042_b200 and
shares no code with the CUDA path.
"""
