"""CPU oracle for the MPCD solvent step -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  See oracle/mpcd_oracle.c for the header.
"""
