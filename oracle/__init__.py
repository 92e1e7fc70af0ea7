"""CPU oracle (test infrastructure, not the product).  See oracle/fxo.cpp for the header.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports the CUDA package.
"""
from .fxo import *  # noqa: F401,F403
