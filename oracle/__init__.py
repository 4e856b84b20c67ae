"""CPU oracle for RANLUX++ (arxiv 2106.02504) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this package.  It shares nothing with the CUDA path.
"""
from .oracle import *  # noqa: F401,F403
