"""CPU oracle of the pyJac v2 hot path -- TEST INFRASTRUCTURE (see pyjac_oracle.cpp header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
"""
from .oracle import Oracle, DESC_FIELDS

__all__ = ["Oracle", "DESC_FIELDS"]
