"""CPU oracle of the SFUMATO# AMR hydro step.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The product (paper_2604_21438_b200) never does.  See sfh_oracle.cpp.
"""
from .binding import OracleMesh, lib, oracle_for  # noqa: F401
from .norms import parity_errors  # noqa: F401
