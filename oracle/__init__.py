"""ORACLE — test infrastructure only (see oracle/dwf_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_2203_17119_b200.
"""
