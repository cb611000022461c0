"""ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle/oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2209_15445_b200.adept (the CUDA binding).
"""
