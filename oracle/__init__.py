"""ORACLE — test infrastructure only (see oracle/stratego_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from the product package.
"""
