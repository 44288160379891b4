"""CPU oracle for the dipolar-GPE SSCN step -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  See oracle/dgpe_oracle.h for what it computes and what pins it.
"""
