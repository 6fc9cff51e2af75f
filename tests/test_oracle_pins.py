"""Pins of the oracle against things other than itself (CPU only).

P1 golden numbers (tests/golden/p1_ab.txt), P2 hand-derived 4-species mechanism, P3 long-double
4th-order finite differences, P4 complex step, P5 mass conservation, P6 constructed equilibrium,
P7 brute-force sparsity pattern, P8 Euler homogeneity, P9 cross-mode identity, P10 reductions of each
rate law to a textbook special case, P11 dense/sparse/CSR/CSC consistency, A1 unbalanced mechanism.
"""
import math
import os

import numpy as np
import pytest

import mechgen as mg
from mechgen import MechBuilder
from oracle import Oracle

R = 8314.46261815324
PATM = 101325.0
HERE = os.path.dirname(os.path.abspath(__file__))


def jac_tol(ref):
    rowmax = np.abs(ref).max(axis=-1, keepdims=True)
    return np.maximum(np.maximum(1e-8 * np.abs(ref), 1e-12 * rowmax), 1e-300)


def golden(name):
    out = {}
    for line in open(os.path.join(HERE, "golden", name)):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        out[k] = np.array([float(x) for x in v])
    return out


# ---------------------------------------------------------------- P1
def test_p1_two_species_golden():
    g = golden("p1_ab.txt")
    o = Oracle(mg.hand_ab())
    T, P, V = 1500.0, 202650.0, 1e-3
    nA = 0.3 * P * V / (R * T)
    it = o.intermediates(mg.CONP, [T, V, nA], P)
    for key, val in (("kf", it["kf"][0]), ("Kc", it["Kc"][0]), ("kr", it["kr"][0]), ("C_A", it["C"][0]),
                     ("C_B", it["C"][1]), ("q", it["q"][0])):
        assert val == pytest.approx(g[key][0], rel=2e-14), key
    f = o.source(mg.CONP, [T, V, nA], [P])[0]
    assert f[0] == pytest.approx(g["conp_dT_dt"][0], rel=1e-13)
    assert f[1] == pytest.approx(g["conp_dV_dt"][0], rel=1e-13)
    assert f[2] == pytest.approx(g["dnA_dt"][0], rel=1e-13)
    J = o.jacobian_dense(mg.CONP, [T, V, nA], [P])[0]
    np.testing.assert_allclose(J.reshape(-1), g["conp_J"], rtol=2e-13)
    f = o.source(mg.CONV, [T, P, nA], [V])[0]
    assert f[0] == pytest.approx(g["conv_dT_dt"][0], rel=1e-13)
    assert f[1] == pytest.approx(g["conv_dP_dt"][0], rel=1e-13)
    J = o.jacobian_dense(mg.CONV, [T, P, nA], [V])[0]
    np.testing.assert_allclose(J.reshape(-1), g["conv_J"], rtol=2e-13)


def test_p1_closed_forms():
    """Closed forms of SURVEY.md 8c-7 P1, evaluated here with python floats."""
    o = Oracle(mg.hand_ab())
    T, P, V = 1234.5, 3.3e5, 2.5e-2
    nA = 0.62 * P * V / (R * T)
    kf = 1e10 * T ** 0.5 * math.exp(-15000.0 / T)
    gA = 4.0 * (1 - math.log(T)) - 1000.0 / T - 3.0      # g/RT of a constant-cp species
    gB = 4.5 * (1 - math.log(T)) - 6000.0 / T - 2.0
    Kc = math.exp(-(gB - gA))
    kr = kf / Kc
    CA = nA / V
    q = kf * CA - kr * (P / (R * T) - CA)
    Jp = o.jacobian_dense(mg.CONP, [T, V, nA], [P])[0]
    Jv = o.jacobian_dense(mg.CONV, [T, P, nA], [V])[0]
    fp = o.source(mg.CONP, [T, V, nA], [P])[0]
    fv = o.source(mg.CONV, [T, P, nA], [V])[0]
    assert fp[2] == pytest.approx(-V * q, rel=1e-12) and fv[2] == pytest.approx(-V * q, rel=1e-12)
    assert fp[1] == pytest.approx(V / T * fp[0], rel=1e-12)          # W_A = W_B: S = 0
    assert fv[1] == pytest.approx(P / T * fv[0], rel=1e-12)
    HA, HB = R * (4.0 * T - 1000.0), R * (4.5 * T - 6000.0)
    D = CA * 4.0 * R + (P / (R * T) - CA) * 4.5 * R
    assert fp[0] == pytest.approx((HA - HB) * q / D, rel=1e-12)
    assert Jp[2, 2] == pytest.approx(-(kf + kr), rel=1e-12)
    assert Jv[2, 2] == pytest.approx(-(kf + kr), rel=1e-12)
    assert Jp[2, 1] == pytest.approx(kr * P / (R * T), rel=1e-12)
    assert Jv[2, 1] == pytest.approx(kr * V / (R * T), rel=1e-12)


# ---------------------------------------------------------------- P2
def _four_state():
    T, P, V = 1400.0, 5.0 * PATM, 0.02
    X = np.array([0.15, 0.25, 0.1, 0.5])
    return T, P, V, X * P * V / (R * T)


def test_p2_four_species_hand_derived():
    m = mg.hand_four()
    o = Oracle(m)
    T, P, V, n = _four_state()
    CA, CB, CC, CN = n / V
    Ctot = P / (R * T)
    g = lambda a0, a5, a6: a0 * (1 - math.log(T)) + a5 / T - a6
    gA, gB = g(2.5, 2.0e4, 5.0), g(3.5, 1.0e3, 7.0)
    Kc = math.exp(-(gB - 2 * gA)) / (PATM / (R * T))           # sum nu = -1
    k1 = 2.0e9 * T ** 0.3 * math.exp(-1500.0 / T)
    k2 = 5.0e8 * T ** -0.5 * math.exp(-500.0 / T)
    kinf = 3.0e12 * T ** 0.2 * math.exp(-20000.0 / T)
    k0 = 4.0e14 * T ** -0.8 * math.exp(-18000.0 / T)
    q1 = k1 * CA * CA - k1 / Kc * CB
    M2 = CA + CB + 3.0 * CC + CN
    q2 = M2 * (k2 * CA * CA - k2 / Kc * CB)
    Pr = k0 * Ctot / kinf
    q3 = Pr / (1 + Pr) * kinf * CC
    wA, wB, wC = -2 * q1 - 2 * q2 + q3, q1 + q2 + q3, -q3
    f = o.source(mg.CONP, np.concatenate([[T, V], n[:3]]), [P])[0]
    np.testing.assert_allclose(f[2:], V * np.array([wA, wB, wC]), rtol=1e-12)
    H = lambda a0, a5: R * (a0 * T + a5)
    wN = -(10 * wA + 20 * wB + 30 * wC) / 28.0
    assert abs(wN) < 1e-12 * max(abs(wA), abs(wB))             # balanced: bath gas inert
    N = H(2.5, 2.0e4) * wA + H(3.5, 1.0e3) * wB + H(4.5, 3.0e3) * wC
    D = R * (2.5 * CA + 3.5 * CB + 4.5 * CC + 3.5 * CN)
    assert f[0] == pytest.approx(-N / D, rel=1e-12)
    S = (1 - 10 / 28) * wA + (1 - 20 / 28) * wB + (1 - 30 / 28) * wC
    assert f[1] == pytest.approx(V * (T * R / P * S + f[0] / T), rel=1e-12)
    # hand-derived species-block entries (bath inert, default efficiency => G^Ns terms cancel)
    J = o.jacobian_dense(mg.CONP, np.concatenate([[T, V], n[:3]]), [P])[0]
    R2 = k2 * CA * CA - k2 / Kc * CB
    dq1 = np.array([2 * k1 * CA, -k1 / Kc, 0.0])
    dq2 = np.array([2 * M2 * k2 * CA, -M2 * k2 / Kc, (3.0 - 1.0) * R2])
    dq3 = np.array([0.0, 0.0, Pr / (1 + Pr) * kinf])
    blk = np.array([-2 * dq1 - 2 * dq2 + dq3, dq1 + dq2 + dq3, -dq3])
    np.testing.assert_allclose(J[2:, 2:], blk, rtol=1e-11, atol=0)
    # pattern: rows A, B = {A, B, C}; row C = {C} only
    ptr, idx = o.pattern(mg.CSR)
    rows = [list(idx[ptr[r]:ptr[r + 1]]) for r in range(5)]
    assert rows == [[0, 1, 2, 3, 4], [0, 1, 2, 3, 4], [0, 1, 2, 3, 4], [0, 1, 2, 3, 4], [0, 1, 4]]


def test_p2b_last_species_reacting_gives_dense_rows():
    o = Oracle(mg.hand_four(order=(1, 2, 3, 0)))          # A last
    ptr, idx = o.pattern(mg.CSR)
    rows = [list(idx[ptr[r]:ptr[r + 1]]) for r in range(5)]
    # order B, C, N | A last.  Row B takes part in R1, R2 whose rates depend on the last species
    # => dense row; row C only in the irreversible R3: C -> A + B => {C}; N inert.
    assert rows == [[0, 1, 2, 3, 4], [0, 1, 2, 3, 4], [0, 1, 2, 3, 4], [0, 1, 3], [0, 1]]


# ---------------------------------------------------------------- P3 / P4
MECHS = {
    "all_types": lambda: (mg.hand_all_types(True, True), mg.make_states(6, 4, 11)),
    "all_types_inert": lambda: (mg.hand_all_types(False, False), mg.make_states(6, 4, 12)),
    "chem_activated": lambda: (mg.hand_chem_activated(), mg.make_states(5, 6, 13)),
    "rev_explicit": lambda: (mg.hand_rev_explicit(), mg.make_states(6, 6, 14)),
    "c1": lambda: (mg.config_mechanism(1), mg.config_states(1, 16)),
    "c2": lambda: (mg.config_mechanism(2), mg.config_states(2, 16)),
    "c3": lambda: (mg.config_mechanism(3), mg.config_states(3, 16)),
    "c4": lambda: (mg.config_mechanism(4), mg.config_states(4, 2)),
    "c5": lambda: (mg.config_mechanism(5), mg.config_states(5, 2)),
}


@pytest.mark.parametrize("name", list(MECHS))
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
def test_p4_complex_step(name, mode):
    m, st = MECHS[name]()
    o = Oracle(m)
    phi, par = o.pack(st, mode)
    J = o.jacobian_dense(mode, phi, par)
    for s in range(phi.shape[0]):
        Jc = o.cs_jacobian(mode, phi[s], par[s])
        err = np.abs(J[s] - Jc) / jac_tol(Jc)
        assert err.max() < 1e-3, (s, np.unravel_index(err.argmax(), err.shape))


@pytest.mark.parametrize("name", ["all_types", "c1", "c2", "c3"])
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
def test_p3_fourth_order_fd_long_double(name, mode):
    m, st = MECHS[name]()
    o = Oracle(m)
    phi, par = o.pack(st, mode)
    J = o.jacobian_dense(mode, phi, par)
    for s in range(min(phi.shape[0], 16)):
        Jf = o.fd_jacobian(mode, phi[s], par[s])
        rowmax = np.abs(J[s]).max(axis=1, keepdims=True)
        err = np.abs(J[s] - Jf) / np.maximum(np.maximum(np.abs(J[s]), 1e-6 * rowmax), 1e-300)
        assert err.max() < 1e-6, (s, err.max())


# ---------------------------------------------------------------- P5
def _nu(m):
    nu = np.zeros((m["n_species"], m["n_reactions"]))
    for i in range(m["n_reactions"]):
        for j in range(m["reac_ptr"][i], m["reac_ptr"][i + 1]):
            nu[m["reac_species"][j], i] -= m["reac_nu"][j]
        for j in range(m["prod_ptr"][i], m["prod_ptr"][i + 1]):
            nu[m["prod_species"][j], i] += m["prod_nu"][j]
    return nu


@pytest.mark.parametrize("c", [1, 2, 3, 4])
def test_p5_mass_conservation(c):
    m = mg.config_mechanism(c)
    o = Oracle(m)
    st = mg.config_states(c, 3)
    phi, par = o.pack(st, mg.CONP)
    nu = _nu(m)
    W = m["mol_weight"]
    for s in range(3):
        it = o.intermediates(mg.CONP, phi[s], par[s])
        wd = nu @ it["q"]                                  # Eq. 4 summed directly for ALL species
        scale = np.abs(nu) @ np.abs(it["q"])
        np.testing.assert_allclose(it["wdot"][:-1], wd[:-1], rtol=0, atol=1e-13 * scale.max())
        assert abs(W @ wd) <= 1e-12 * (W @ scale)
        assert abs(it["wdot"][-1] - wd[-1]) <= 1e-12 * scale.max()


def test_a1_unbalanced_mechanism_uses_mass_conservation():
    o = Oracle(mg.hand_unbalanced())
    T, P, V = 1600.0, 2e5, 0.1
    n = np.array([0.4, 0.1]) * P * V / (R * T)
    it = o.intermediates(mg.CONP, np.concatenate([[T, V], n]), P)
    q = it["q"][0]
    assert q > 0
    assert it["wdot"][2] == pytest.approx(-(10.0 * -q + 7.0 * 2 * q) / 28.0, rel=1e-13)   # not 0
    assert it["S"] == pytest.approx(24.0 / 28.0 * q, rel=1e-13)                          # not q


# ---------------------------------------------------------------- P6
@pytest.mark.parametrize("c", [1, 2, 3])
def test_p6_zero_net_rate_at_constructed_equilibrium(c):
    m = mg.config_mechanism(c)
    o = Oracle(m)
    ns = m["n_species"]
    rng = np.random.default_rng(c)
    T = 1500.0
    comp = m["composition"].astype(float)
    g = o.intermediates(mg.CONP, np.concatenate([[T, 1.0], np.full(ns - 1, 1e-3)]), 1e5)["g"]
    lam = rng.uniform(-2.0, 0.5, 4)
    lnC = np.log(PATM / (R * T)) - g + comp @ lam
    lnC = np.log(PATM / (R * T)) - g + comp @ lam
    # choose the N potential so that the bath gas (N2, last) is abundant: [C]_Ns = C_tot - sum is then
    # well conditioned (it is a difference in the reformulated state)
    lam[3] += 0.5 * (np.max(lnC[:-1]) + 2.0 - lnC[-1])
    lnC = np.log(PATM / (R * T)) - g + comp @ lam
    C = np.exp(lnC)
    V = 1.0
    P = C.sum() * R * T
    it = o.intermediates(mg.CONP, np.concatenate([[T, V], C[:-1] * V]), P)
    rev = m["reversible"].astype(bool)
    assert rev.sum() > 0
    rel = np.abs(it["Rf"][rev] - it["Rr"][rev]) / np.abs(it["Rf"][rev])
    # round-off only: exp() of arguments of size |ln C| ~ 1e2 carries ~1e-16 * 1e2 per factor
    assert rel.max() <= 1e-12 * max(1.0, np.abs(lnC).max()), rel.max()


# ---------------------------------------------------------------- P7
@pytest.mark.parametrize("name", ["four", "four_b", "all_types", "all_types_inert", "c1", "c2", "c3"])
def test_p7_pattern_equals_brute_force(name):
    if name == "four":
        m = mg.hand_four(); st = mg.make_states(4, 8, 3)
    elif name == "four_b":
        m = mg.hand_four(order=(1, 2, 3, 0)); st = mg.make_states(4, 8, 4)
    else:
        m, st = MECHS[name]()
    o = Oracle(m)
    nvar = o.nvar
    nzmask = np.zeros((nvar, nvar), bool)
    for mode in (mg.CONP, mg.CONV):
        phi, par = o.pack(st, mode)
        for s in range(min(8, phi.shape[0])):
            nzmask |= o.cs_jacobian(mode, phi[s], par[s]) != 0.0
    ptr, idx = o.pattern(mg.CSR)
    pat = np.zeros((nvar, nvar), bool)
    for r in range(nvar):
        pat[r, idx[ptr[r]:ptr[r + 1]]] = True
    assert pat[:2].all() and pat[:, :2].all()              # T, E rows and columns dense (S10)
    assert np.array_equal(pat[2:, 2:], nzmask[2:, 2:])      # species block: rule == numerical nonzeros
    # rows T and E are numerically dense wherever any species reacts
    assert nzmask[:2, 2:].all() or name.startswith("all_types")
    # CSC is the exact transpose view
    cptr, cidx = o.pattern(mg.CSC)
    patc = np.zeros((nvar, nvar), bool)
    for c in range(nvar):
        patc[cidx[cptr[c]:cptr[c + 1]], c] = True
        assert np.all(np.diff(cidx[cptr[c]:cptr[c + 1]]) > 0)
    assert np.array_equal(pat, patc)


# ---------------------------------------------------------------- P8, P9, P11
@pytest.mark.parametrize("name", ["all_types", "c1", "c2", "c3"])
def test_p8_euler_homogeneity_conp(name):
    m, st = MECHS[name]()
    o = Oracle(m)
    phi, par = o.pack(st, mg.CONP)
    J = o.jacobian_dense(mg.CONP, phi, par)
    f = o.source(mg.CONP, phi, par)
    for s in range(phi.shape[0]):
        x = phi[s].copy(); x[0] = 0.0
        lhs = J[s] @ x
        rhs = f[s].copy(); rhs[0] = 0.0
        scale = np.abs(J[s]) @ np.abs(x)
        assert np.all(np.abs(lhs - rhs) <= 1e-10 * scale + 1e-300)


@pytest.mark.parametrize("name", ["all_types", "c2", "c3"])
def test_p9_cross_mode_identity(name):
    m, st = MECHS[name]()
    o = Oracle(m)
    pp, qp = o.pack(st, mg.CONP); pv, qv = o.pack(st, mg.CONV)
    Jp = o.jacobian_dense(mg.CONP, pp, qp); Jv = o.jacobian_dense(mg.CONV, pv, qv)
    fp = o.source(mg.CONP, pp, qp); fv = o.source(mg.CONV, pv, qv)
    np.testing.assert_array_equal(fp[:, 2:], fv[:, 2:])
    np.testing.assert_allclose(Jp[:, 2:, 2:], Jv[:, 2:, 2:], rtol=1e-14)
    np.testing.assert_allclose(Jp[:, 2:, 0], Jv[:, 2:, 0], rtol=1e-14)


@pytest.mark.parametrize("name", ["all_types", "c1", "c3"])
def test_p11_dense_sparse_consistency(name):
    m, st = MECHS[name]()
    o = Oracle(m)
    phi, par = o.pack(st, mg.CONV)
    J = o.jacobian_dense(mg.CONV, phi, par)
    for fmt in (mg.CSR, mg.CSC):
        vals = o.jacobian_sparse(mg.CONV, fmt, phi, par)
        ptr, idx = o.pattern(fmt)
        dense = np.zeros_like(J)
        for a in range(o.nvar):
            sl = slice(ptr[a], ptr[a + 1])
            if fmt == mg.CSR:
                dense[:, a, idx[sl]] = vals[:, sl]
            else:
                dense[:, idx[sl], a] = vals[:, sl]
        np.testing.assert_array_equal(dense, J)          # off-pattern entries are exactly 0.0
