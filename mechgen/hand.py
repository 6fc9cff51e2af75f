"""Small hand-built mechanisms used as pins of the oracle.

Only descriptions live here; the expected numbers are derived in tests/ (closed forms) or cited from
SURVEY.md section 8c-8.
"""
from __future__ import annotations

import numpy as np

from .mechanism import (MechBuilder, ELEMENTARY, THIRD_BODY, FALLOFF_LINDEMANN, FALLOFF_TROE,
                        FALLOFF_SRI, PLOG, CHEBYSHEV, P_ATM)


def _const_cp(a0, a5, a6):
    return [a0, 0.0, 0.0, 0.0, 0.0, a5, a6]


def hand_ab():
    """P1: two species A, B (B last), one reversible reaction A <=> B."""
    mb = MechBuilder()
    mb.add_species(30.0, _const_cp(4.0, -1000.0, 3.0))
    mb.add_species(30.0, _const_cp(4.5, -6000.0, 2.0))
    mb.add_reaction({0: 1}, {1: 1}, A=1e10, beta=0.5, Ta=15000.0, rev=True)
    return mb.build()


def hand_four(order=(0, 1, 2, 3)):
    """P2: A = X, B = X2, C = X3 (W = 10, 20, 30) and inert bath N (W = 28).

    R1: 2A <=> B elementary; R2: 2A + M <=> B + M third body, alpha_C = 3;
    R3: C (+M) -> A + B irreversible Lindemann falloff, default efficiencies.
    `order` permutes the species (order[i] = original species placed at position i); the default
    puts the bath gas last, order=(1, 2, 3, 0) puts A last (variant P2b: dense rows).
    """
    W = [10.0, 20.0, 30.0, 28.0]
    thermo = [_const_cp(2.5, 2.0e4, 5.0), _const_cp(3.5, 1.0e3, 7.0), _const_cp(4.5, 3.0e3, 9.0),
              _const_cp(3.5, -1.0e3, 6.5)]
    pos = {orig: i for i, orig in enumerate(order)}
    mb = MechBuilder()
    for orig in order:
        mb.add_species(W[orig], thermo[orig])
    A, B, C = pos[0], pos[1], pos[2]
    mb.add_reaction({A: 2}, {B: 1}, A=2.0e9, beta=0.3, Ta=1500.0, rev=True, type=ELEMENTARY)
    mb.add_reaction({A: 2}, {B: 1}, A=5.0e8, beta=-0.5, Ta=500.0, rev=True, type=THIRD_BODY, eff={C: 3.0})
    mb.add_reaction({C: 1}, {A: 1, B: 1}, A=3.0e12, beta=0.2, Ta=20000.0, rev=False,
                    type=FALLOFF_LINDEMANN, low=(4.0e14, -0.8, 18000.0))
    return mb.build()


def hand_unbalanced():
    """Reading A1: three species, A -> 2 B with W that do NOT balance (W_A != 2 W_B); C inert, last.

    The direct sum of omega_Ns over reactions (0 here) and the mass-conservation value differ.
    """
    mb = MechBuilder()
    mb.add_species(10.0, _const_cp(3.0, 500.0, 4.0))
    mb.add_species(7.0, _const_cp(2.5, 9000.0, 3.0))
    mb.add_species(28.0, _const_cp(3.5, -1000.0, 6.0))
    mb.add_reaction({0: 1}, {1: 2}, A=1.0e6, beta=0.0, Ta=8000.0, rev=False)
    return mb.build()


def hand_all_types(last_reacts=True, last_eff=True, seed=7):
    """Six species / ten reactions covering every reaction type, both dense-row mechanisms optional.

    Compositions: S0 = X, S1 = X2, S2 = X3, S3 = X4, S4 = Y, S5 = bath (composition Z2) so every
    reaction below is element balanced when the bath only appears on both sides or not at all;
    `last_reacts` adds S5 as a net-zero catalyst-like participant (nu' = nu'' = 1).
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    mb = MechBuilder()
    W = [5.0, 10.0, 15.0, 20.0, 9.0, 28.0]
    for k in range(6):
        lo = np.array([3.0 + 0.4 * k, 1.2e-3, -3.0e-7, 4.0e-11, -2.0e-15, 1000.0 * (k - 2.5), 4.0 + k])
        hi = lo.copy()
        hi[1:5] *= 0.8
        # continuity at T_mid = 1000 of cp, H, S
        T = 1000.0
        cp_lo = np.polyval(lo[4::-1], T); cp_hi = np.polyval(hi[4::-1], T)
        hi[0] += cp_lo - cp_hi
        H = lambda a: a[0] * T + a[1] * T**2 / 2 + a[2] * T**3 / 3 + a[3] * T**4 / 4 + a[4] * T**5 / 5 + a[5]
        S = lambda a: a[0] * np.log(T) + a[1] * T + a[2] * T**2 / 2 + a[3] * T**3 / 3 + a[4] * T**4 / 4 + a[6]
        hi[5] += H(lo) - H(hi); hi[6] += S(lo) - S(hi)
        mb.add_species(W[k], lo, hi, 1000.0)
    L = 5
    cat = {L: 1} if last_reacts else {}
    eL = {L: 2.5} if last_eff else {}
    mb.add_reaction({0: 2}, {1: 1}, A=3e9, beta=0.4, Ta=2000.0, rev=True)                                   # elementary, nu'=2
    mb.add_reaction({0: 1, 1: 1, **cat}, {2: 1, **cat}, A=2e8, beta=-0.3, Ta=1000.0, rev=True)               # last species both sides
    mb.add_reaction({0: 1, 2: 1}, {3: 1}, A=7e8, beta=0.1, Ta=500.0, rev=True, type=THIRD_BODY,
                    eff={1: 2.0, 4: 0.0, **eL})
    mb.add_reaction({3: 1}, {1: 2}, A=4e13, beta=0.0, Ta=22000.0, rev=True, type=FALLOFF_LINDEMANN,
                    low=(6e15, -1.0, 20000.0), eff={0: 1.5})
    mb.add_reaction({2: 1}, {0: 1, 1: 1}, A=9e12, beta=0.5, Ta=18000.0, rev=True, type=FALLOFF_TROE,
                    low=(2e16, -1.5, 17000.0), troe=(0.6, 200.0, 1500.0, 5000.0), eff={3: 4.0, **eL})
    mb.add_reaction({3: 1}, {0: 1, 2: 1}, A=5e12, beta=-0.2, Ta=25000.0, rev=False, type=FALLOFF_TROE,
                    low=(8e15, -0.7, 21000.0), troe=(0.35, 800.0, 3000.0, None))
    mb.add_reaction({1: 1, 0: 1}, {2: 1}, A=6e9, beta=0.2, Ta=300.0, rev=True, type=FALLOFF_SRI,
                    low=(3e12, -0.4, 100.0), sri=(0.9, 400.0, 2500.0, 1.3, 0.2), collider=4)
    mb.add_reaction({1: 2}, {3: 1}, A=1.0, rev=True, type=PLOG,
                    plog=[(0.1 * P_ATM, 2e7, 0.5, 3000.0), (1.0 * P_ATM, 9e7, 0.4, 3300.0),
                          (10.0 * P_ATM, 5e8, 0.2, 3500.0), (100.0 * P_ATM, 1e9, 0.1, 3900.0)])
    coef = rng.uniform(-1, 1, size=(5, 3)) * 0.5 ** np.add.outer(np.arange(5), np.arange(3))
    coef[0, 0] = 7.5
    mb.add_reaction({2: 1, 0: 1}, {1: 2}, A=1.0, rev=True, type=CHEBYSHEV,
                    cheb=dict(Tmin=300.0, Tmax=3000.0, Pmin=0.01 * P_ATM, Pmax=100.0 * P_ATM, coef=coef))
    mb.add_reaction({1: 1, 2: 1}, {0: 1, 3: 1}, A=1e10, beta=0.0, Ta=6000.0, rev=False)                      # irreversible 2-2
    return mb.build()


def hand_chem_activated():
    """Five species A, B, C, D and bath N (last): every falloff form once as a chemically-activated reaction
    (k = k_0 F / (1 + P_r)) next to its plain falloff twin with the same parameters, plus one
    elementary reaction so that all species take part.  A = X, B = X, C = X2, D = X2 (isomers), so A + B <=> C is
    balanced."""
    mb = MechBuilder()
    W = [10.0, 10.0, 20.0, 20.0, 28.0]
    th = [_const_cp(2.6, 1.5e4, 5.0), _const_cp(2.9, 1.1e4, 5.5), _const_cp(3.6, 2.0e3, 7.0), _const_cp(3.9, 1.0e3, 7.5),
          _const_cp(3.5, -1.0e3, 6.5)]
    for w, t in zip(W, th):
        mb.add_species(w, t)
    A, B, C, D = 0, 1, 2, 3
    hi = dict(A=3.0e10, beta=0.4, Ta=2500.0)
    low = (7.0e11, -0.6, 1200.0)
    eff = {C: 2.5, D: 0.4}
    for chem in (True, False):
        mb.add_reaction({A: 1, B: 1}, {C: 1}, rev=True, type=FALLOFF_LINDEMANN, low=low, eff=eff, chem_activated=chem, **hi)
        mb.add_reaction({A: 2}, {D: 1}, rev=True, type=FALLOFF_TROE, low=low, troe=(0.6, 200.0, 1800.0, 5000.0), eff=eff,
                        chem_activated=chem, **hi)
        mb.add_reaction({A: 1, B: 1}, {D: 1}, rev=False, type=FALLOFF_SRI, low=low, sri=(0.8, 300.0, 2000.0, 1.2, 0.1),
                        chem_activated=chem, **hi)
    mb.add_reaction({C: 1}, {D: 1}, A=4.0e7, beta=0.2, Ta=6000.0, rev=True)
    return mb.build()


def hand_rev_explicit():
    """Five species and bath N (last): explicit reverse Arrhenius parameters (k_r given, not k_f / K_c) on an
    elementary, a third-body, a Troe falloff and a chemically-activated Lindemann reaction, next to K_c-based ones."""
    mb = MechBuilder()
    W = [10.0, 10.0, 20.0, 20.0, 30.0, 28.0]
    th = [_const_cp(2.6, 1.5e4, 5.0), _const_cp(2.9, 1.1e4, 5.5), _const_cp(3.6, 2.0e3, 7.0), _const_cp(3.9, 1.0e3, 7.5),
          _const_cp(4.4, -2.0e3, 8.0), _const_cp(3.5, -1.0e3, 6.5)]
    for w, t in zip(W, th):
        mb.add_species(w, t)
    A, B, C, D, E = 0, 1, 2, 3, 4
    mb.add_reaction({A: 1, B: 1}, {C: 1}, A=2.0e9, beta=0.3, Ta=1500.0, rev=True, rev_params=(5.0e11, -0.2, 9000.0))
    mb.add_reaction({A: 2}, {D: 1}, A=5.0e8, beta=-0.5, Ta=500.0, rev=True, type=THIRD_BODY, eff={C: 3.0, E: 0.5},
                    rev_params=(2.0e10, 0.1, 7000.0))
    mb.add_reaction({A: 1, C: 1}, {E: 1}, A=3.0e10, beta=0.4, Ta=2500.0, rev=True, type=FALLOFF_TROE,
                    low=(7.0e11, -0.6, 1200.0), troe=(0.6, 200.0, 1800.0, 5000.0), eff={D: 2.0},
                    rev_params=(8.0e12, 0.0, 15000.0))
    mb.add_reaction({B: 1, D: 1}, {E: 1}, A=1.0e10, beta=0.2, Ta=1000.0, rev=True, type=FALLOFF_LINDEMANN,
                    low=(3.0e11, -0.4, 800.0), chem_activated=True, rev_params=(4.0e12, -0.3, 12000.0))
    mb.add_reaction({C: 1}, {D: 1}, A=4.0e7, beta=0.2, Ta=6000.0, rev=True)
    mb.add_reaction({A: 1, B: 1}, {D: 1}, A=6.0e8, beta=0.1, Ta=2000.0, rev=True)
    return mb.build()
