"""CPU oracle for the explicit phase-field fracture hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this package.  It shares no code with paper_2606_23458_b200 (the CUDA product path).
"""
from .pff_oracle import OracleMesh, Material, build, element_response, oracle_from  # noqa: F401
