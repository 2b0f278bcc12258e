"""CPU oracle of the CHORUS-MHD hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2502_17805_b200 except the seeded input
generators (paper_2502_17805_b200.inputs), which hold none of the method's arithmetic.
"""
from .binding import Oracle, lib, physics_struct  # noqa: F401
