"""ORACLE: plain single-threaded fp64 CPU restatement of the hot path (test infrastructure only).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package; the product (paper_2010_11540_b200) never does.
"""
