"""CPU oracle for the Ipatia+exponential NLL hot path (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  Nothing here imports paper_1706_01420_b200 and vice versa.
"""
from .binding import *  # noqa: F401,F403
