"""ORACLE -- test infrastructure, not the product.  See kvr_oracle.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import, build or call anything in this package.  It imports nothing from paper_2606_17107_b200.
"""
