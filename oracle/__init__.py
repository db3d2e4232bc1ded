"""CPU oracle of the cuHARM hot path — TEST INFRASTRUCTURE ONLY (see oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It never imports the CUDA package.
"""
from .oracle import *  # noqa: F401,F403
