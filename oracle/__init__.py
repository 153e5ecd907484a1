"""CPU oracle for Matching Pursuit -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The arithmetic is plain C (mp_oracle.c); this package is a ctypes binding.
"""
from .mp_oracle import *  # noqa: F401,F403
