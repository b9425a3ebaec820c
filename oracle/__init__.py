"""CPU oracle for the COSEnu RK4 hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  The product (paper_2203_12866_b200) never does.
"""
