"""CPU ORACLE -- test infrastructure only (see oracle/orc.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  The product (paper_2409_16053_b200) never does.
"""
