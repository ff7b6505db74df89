"""Test-infrastructure oracle for the NVFP4 GEMV hot path (see nvfp4_oracle.py).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package; the product (paper_2606_13233_b200) never does.
"""
