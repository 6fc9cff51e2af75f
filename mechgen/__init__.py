"""Seeded synthetic inputs (mechanisms and thermochemical states) for pyjac-b200.

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA product
(`paper_1809_01029_b200/`).  It holds no arithmetic of the method (no rate laws, no source terms,
no Jacobian): it only draws random mechanism descriptions and states with the shapes of the paper's
workloads (Table 4, Table 7; recipe in DESIGN.md "Input recipe").

A mechanism is a plain dict of numpy arrays ("desc arrays") whose keys mirror the fields of
`pyjac_mech_desc` in include/pyjac.h.
"""
from .mechanism import (CONFIGS, R_GAS, P_ATM, ELEMENTARY, THIRD_BODY, FALLOFF_LINDEMANN,
                        FALLOFF_TROE, FALLOFF_SRI, PLOG, CHEBYSHEV, CONP, CONV, CSR, CSC,
                        make_mechanism, config_mechanism, config_states, make_states, MechBuilder)
from .hand import hand_ab, hand_four, hand_unbalanced, hand_all_types, hand_chem_activated, hand_rev_explicit

__all__ = [n for n in dir() if not n.startswith("_")]
