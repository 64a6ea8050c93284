"""CPU oracle — TEST INFRASTRUCTURE ONLY (see oracle/neighbors.c, oracle/tree.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports the CUDA package.
"""
