"""CPU oracle of the SFUMATO# AMR hydro step.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The product (paper_2604_21438_b200) never does.  See sfh_oracle.cpp.
"""
from .binding import OracleMesh, lib  # noqa: F401
