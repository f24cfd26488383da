"""CPU oracle for Langevin Speculative Dynamics -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package.  It never imports paper_2606_02455_b200 and shares no code with it.
"""
from .binding import *  # noqa: F401,F403
