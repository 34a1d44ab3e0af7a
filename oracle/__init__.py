"""FP64 CPU oracle for the MSFT forward simulation -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The product (paper_2202_03411_b200) never does.
"""
