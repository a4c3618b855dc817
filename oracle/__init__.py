"""CPU oracle of the single-pulse-detection path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package (see oracle/spd_oracle.c for the header and the pins).
"""
