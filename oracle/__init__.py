"""CPU oracle of the CaLES hot path -- TEST INFRASTRUCTURE ONLY (see oracle/cales_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
"""
from .binding import *  # noqa: F401,F403
