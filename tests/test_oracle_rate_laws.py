"""P10: each rate law reduces to a textbook special case (CPU only)."""
import math

import numpy as np
import pytest

import mechgen as mg
from mechgen import MechBuilder
from oracle import Oracle

R = 8314.46261815324
PATM = 101325.0
CP = lambda a0, a5, a6: [a0, 0, 0, 0, 0, a5, a6]


def _three(**rx):
    """A <=> B + C style test bed: species A, B, C, bath N (last)."""
    mb = MechBuilder()
    mb.add_species(30.0, CP(4.0, 1000.0, 5.0)); mb.add_species(10.0, CP(3.0, 9000.0, 4.0))
    mb.add_species(20.0, CP(3.5, 4000.0, 6.0)); mb.add_species(28.0, CP(3.5, -1000.0, 6.5))
    mb.add_reaction({0: 1}, {1: 1, 2: 1}, **rx)
    return mb.build()


def _state(T=1300.0, P=3 * PATM, V=0.05, X=(0.3, 0.2, 0.1, 0.4)):
    n = np.array(X) * P * V / (R * T)
    return np.concatenate([[T, V], n[:3]]), P


def _run(m, **kw):
    o = Oracle(m)
    phi, P = _state(**kw)
    return o, o.intermediates(mg.CONP, phi, P), o.source(mg.CONP, phi, [P])[0], o.jacobian_dense(mg.CONP, phi, [P])[0]


ARR = dict(A=4e13, beta=0.3, Ta=22000.0)
LOW = (6e15, -1.0, 20000.0)


def test_constant_cp_gibbs_closed_form():
    _, it, _, _ = _run(_three(**ARR))
    T = 1300.0
    for k, (a0, a5, a6) in enumerate([(4.0, 1000.0, 5.0), (3.0, 9000.0, 4.0), (3.5, 4000.0, 6.0), (3.5, -1000.0, 6.5)]):
        assert it["g"][k] == pytest.approx(a0 * (1 - math.log(T)) + a5 / T - a6, rel=1e-14)
        assert it["h"][k] == pytest.approx(R * (a0 * T + a5), rel=1e-14)
        assert it["cp"][k] == pytest.approx(R * a0, rel=1e-15)


def test_nasa_full_polynomial_against_numpy():
    m = mg.config_mechanism(1)
    o = Oracle(m)
    for T in (650.0, 1000.0, 1000.0001, 2400.0):
        phi = np.concatenate([[T, 1.0], np.full(12, 1e-4)])
        it = o.intermediates(mg.CONP, phi, 1e5)
        for k in range(13):
            a = m["nasa_lo"][7 * k:7 * k + 7] if T <= 1000.0 else m["nasa_hi"][7 * k:7 * k + 7]
            cp = np.polyval(a[4::-1], T)
            hint = np.polyval(np.concatenate([(a[:5] / np.arange(1, 6))[::-1], [a[5]]]), T) / T
            assert it["cp"][k] == pytest.approx(R * cp, rel=1e-13)
            assert it["h"][k] == pytest.approx(R * T * hint, rel=1e-12)
    # continuity at T_mid (generator property) seen through the oracle
    lo = o.intermediates(mg.CONP, np.concatenate([[1000.0, 1.0], np.full(12, 1e-4)]), 1e5)
    hi = o.intermediates(mg.CONP, np.concatenate([[1000.0 + 1e-9, 1.0], np.full(12, 1e-4)]), 1e5)
    np.testing.assert_allclose(lo["g"], hi["g"], rtol=1e-9)


def test_equilibrium_constant_sum_nu_term():
    _, it, _, _ = _run(_three(**ARR))
    T = 1300.0
    dg = it["g"][1] + it["g"][2] - it["g"][0]
    assert it["Kc"][0] == pytest.approx(math.exp(-dg) * (PATM / (R * T)) ** 1, rel=1e-13)
    assert it["kr"][0] == pytest.approx(it["kf"][0] / it["Kc"][0], rel=1e-15)


def test_troe_reduces_to_lindemann():
    lind = _run(_three(type=mg.FALLOFF_LINDEMANN, low=LOW, **ARR))
    troe = _run(_three(type=mg.FALLOFF_TROE, low=LOW, troe=(1.0, 123.0, 1e300, None), **ARR))
    assert troe[1]["F"][0] == pytest.approx(1.0, abs=1e-15)
    np.testing.assert_allclose(troe[2], lind[2], rtol=1e-14)
    np.testing.assert_allclose(troe[3], lind[3], rtol=1e-12, atol=1e-300)


def test_sri_reduces_to_lindemann():
    lind = _run(_three(type=mg.FALLOFF_LINDEMANN, low=LOW, **ARR))
    sri = _run(_three(type=mg.FALLOFF_SRI, low=LOW, sri=(0.0, 500.0, 1e300, 1.0, 0.0), **ARR))
    assert sri[1]["F"][0] == pytest.approx(1.0, abs=1e-15)
    np.testing.assert_allclose(sri[2], lind[2], rtol=1e-14)
    np.testing.assert_allclose(sri[3], lind[3], rtol=1e-12, atol=1e-300)


def test_falloff_limits():
    elem = _run(_three(**ARR))
    hi = _run(_three(type=mg.FALLOFF_LINDEMANN, low=(6e45, -1.0, 20000.0), **ARR))       # Pr -> inf: k -> k_inf
    np.testing.assert_allclose(hi[2], elem[2], rtol=1e-12)
    lo = _run(_three(type=mg.FALLOFF_LINDEMANN, low=(6e-15, -1.0, 20000.0), **ARR))      # Pr -> 0: c k_inf -> k0 [M]
    T = 1300.0
    k0 = 6e-15 * T ** -1.0 * math.exp(-20000.0 / T)
    Ctot = 3 * PATM / (R * T)
    assert lo[1]["c"][0] * lo[1]["kf"][0] == pytest.approx(k0 * Ctot, rel=1e-12)


def test_third_body_all_default_efficiencies_is_total_concentration():
    _, it, _, _ = _run(_three(type=mg.THIRD_BODY, **ARR))
    assert it["M"][0] == pytest.approx(3 * PATM / (R * 1300.0), rel=1e-14)
    _, it2, _, _ = _run(_three(type=mg.THIRD_BODY, eff={1: 2.5, 3: 0.0}, **ARR))
    C = it2["C"]
    assert it2["M"][0] == pytest.approx(C[0] + 2.5 * C[1] + C[2], rel=1e-14)


def test_plog_identical_points_is_arrhenius_and_node_values():
    elem = _run(_three(**ARR))
    pts = [(p * PATM, ARR["A"], ARR["beta"], ARR["Ta"]) for p in (0.1, 1.0, 10.0)]
    pl = _run(_three(type=mg.PLOG, plog=pts))
    np.testing.assert_allclose(pl[2], elem[2], rtol=1e-13)
    np.testing.assert_allclose(pl[3], elem[3], rtol=1e-11, atol=1e-300)
    # on a node and outside the table the value is that node's Arrhenius (reading S4)
    pts = [(1.0 * PATM, 1e10, 0.0, 5000.0), (10.0 * PATM, 1e12, 0.5, 8000.0)]
    m = _three(type=mg.PLOG, plog=pts)
    for P, (A, b, Ta) in ((1.0 * PATM, (1e10, 0.0, 5000.0)), (0.2 * PATM, (1e10, 0.0, 5000.0)),
                         (10.0 * PATM, (1e12, 0.5, 8000.0)), (80.0 * PATM, (1e12, 0.5, 8000.0))):
        _, it, _, _ = _run(m, P=P)
        assert it["kf"][0] == pytest.approx(A * 1300.0 ** b * math.exp(-Ta / 1300.0), rel=1e-13)
    # geometric mean of pressures -> geometric mean of rates
    _, it, _, _ = _run(m, P=math.sqrt(10.0) * PATM)
    k1 = 1e10 * math.exp(-5000.0 / 1300.0); k2 = 1e12 * 1300.0 ** 0.5 * math.exp(-8000.0 / 1300.0)
    assert it["kf"][0] == pytest.approx(math.sqrt(k1 * k2), rel=1e-12)


def test_chebyshev_special_cases():
    lim = dict(Tmin=300.0, Tmax=3000.0, Pmin=0.01 * PATM, Pmax=100.0 * PATM)
    _, it, _, J = _run(_three(type=mg.CHEBYSHEV, cheb=dict(coef=[[7.25]], **lim)))
    assert it["kf"][0] == pytest.approx(10 ** 7.25, rel=1e-13)
    # linear in T~ and P~: log10 k = e00 + e10 T~ + e01 P~
    coef = [[6.0, 0.3], [-0.7, 0.0]]
    _, it, _, _ = _run(_three(type=mg.CHEBYSHEV, cheb=dict(coef=coef, **lim)))
    T, P = 1300.0, 3 * PATM
    Tt = (2 / T - 1 / 300.0 - 1 / 3000.0) / (1 / 3000.0 - 1 / 300.0)
    Pt = (2 * math.log10(P) - math.log10(0.01 * PATM) - math.log10(100 * PATM)) / (math.log10(100 * PATM) - math.log10(0.01 * PATM))
    assert it["kf"][0] == pytest.approx(10 ** (6.0 + 0.3 * Pt - 0.7 * Tt), rel=1e-12)
    # against numpy's Chebyshev evaluation for a full grid
    rng = np.random.default_rng(0)
    c = rng.uniform(-1, 1, (7, 3)); c[0, 0] = 8.0
    _, it, _, _ = _run(_three(type=mg.CHEBYSHEV, cheb=dict(coef=c, **lim)))
    assert it["kf"][0] == pytest.approx(10 ** np.polynomial.chebyshev.chebval2d(Tt, Pt, c), rel=1e-11)


def test_zero_concentration_is_safe():
    """Reading S7: C_k = 0 gives finite values and the Jacobian still equals the complex step."""
    m = mg.hand_all_types(True, True)
    o = Oracle(m)
    st = mg.make_states(6, 1, 99)
    phi, par = o.pack(st, mg.CONP)
    phi[0, 2] = 0.0
    J = o.jacobian_dense(mg.CONP, phi, par)[0]
    Jc = o.cs_jacobian(mg.CONP, phi[0], par[0])
    assert np.isfinite(J).all()
    rowmax = np.abs(Jc).max(axis=1, keepdims=True)
    assert np.all(np.abs(J - Jc) <= np.maximum(1e-8 * np.abs(Jc), 1e-12 * rowmax))


# ---- chemically-activated bimolecular reactions (R8) ---------------------------------------
def _two(**rx):
    """A + B <=> C test bed (the bimolecular form chemical activation applies to); bath N last."""
    mb = MechBuilder()
    mb.add_species(10.0, CP(2.6, 15000.0, 5.0)); mb.add_species(20.0, CP(3.0, 9000.0, 4.0))
    mb.add_species(30.0, CP(3.8, 4000.0, 6.0)); mb.add_species(28.0, CP(3.5, -1000.0, 6.5))
    mb.add_reaction({0: 1, 1: 1}, {2: 1}, **rx)
    return mb.build()


@pytest.mark.parametrize("form", [dict(type=mg.FALLOFF_LINDEMANN), dict(type=mg.FALLOFF_TROE, troe=(0.6, 200.0, 1800.0, 5000.0)),
                                  dict(type=mg.FALLOFF_SRI, sri=(0.8, 300.0, 2000.0, 1.2, 0.1))])
def test_chem_activated_is_falloff_over_third_body_concentration(form):
    """k_chem = k_0 F / (1 + Pr) and k_falloff = k_inf F Pr / (1 + Pr) with Pr = k_0 [M] / k_inf: k_chem [M] = k_falloff.
    Ties the new form to the falloff forms already pinned above (same F: it depends on T and Pr only)."""
    eff = {0: 2.0, 2: 0.5}
    fall = _run(_two(low=LOW, eff=eff, **form, **ARR))
    chem = _run(_two(low=LOW, eff=eff, chem_activated=True, **form, **ARR))
    M = fall[1]["M"][0]
    assert chem[1]["M"][0] == M and chem[1]["Pr"][0] == pytest.approx(fall[1]["Pr"][0], rel=1e-15)
    assert chem[1]["F"][0] == pytest.approx(fall[1]["F"][0], rel=1e-15)
    np.testing.assert_allclose(chem[2] * M, fall[2], rtol=1e-13)
    T = 1300.0
    k0 = LOW[0] * T ** LOW[1] * math.exp(-LOW[2] / T)
    assert chem[1]["kf"][0] == pytest.approx(k0, rel=1e-14)            # the rate constant of the rates of progress is k_0
    assert chem[1]["c"][0] == pytest.approx(chem[1]["F"][0] / (1.0 + chem[1]["Pr"][0]), rel=1e-15)


def test_chem_activated_limits():
    """Pr -> 0: k -> k_0 (an elementary reaction with the low-pressure parameters); Pr -> inf: k [M] -> k_inf."""
    lo = _run(_two(type=mg.FALLOFF_LINDEMANN, low=LOW, chem_activated=True, A=4e43, beta=0.3, Ta=22000.0))   # k_inf huge
    elem = _run(_two(A=LOW[0], beta=LOW[1], Ta=LOW[2]))
    np.testing.assert_allclose(lo[2], elem[2], rtol=1e-12)
    np.testing.assert_allclose(lo[3], elem[3], rtol=1e-9, atol=1e-30 * np.abs(elem[3]).max())
    hi = _run(_two(type=mg.FALLOFF_LINDEMANN, low=(6e45, -1.0, 20000.0), chem_activated=True, **ARR))        # k_0 huge
    T = 1300.0
    kinf = ARR["A"] * T ** ARR["beta"] * math.exp(-ARR["Ta"] / T)
    assert hi[1]["c"][0] * hi[1]["kf"][0] * hi[1]["M"][0] == pytest.approx(kinf, rel=1e-12)


# ---- explicit reverse Arrhenius parameters (R9) ---------------------------------------------------------------
@pytest.mark.parametrize("extra", [dict(), dict(type=mg.THIRD_BODY, eff={0: 2.0}),
                                   dict(type=mg.FALLOFF_TROE, low=LOW, troe=(0.6, 200.0, 1800.0, 5000.0))])
def test_explicit_reverse_equals_equilibrium_constant_for_constant_cp(extra):
    """With constant c_p the Gibbs polynomial is g/RT = a0 (1 - ln T) + a5/T - a6, so K_c is itself of Arrhenius form:
    k_f / K_c = A_f e^{da0 - da6} (R/P_atm)^{sum nu} T^{beta_f - da0 + sum nu} exp(-(Ta_f - da5)/T).  An explicit reverse
    rate constant with exactly these parameters must reproduce the K_c-based source terms AND Jacobian."""
    a0 = [2.6, 3.0, 3.8]; a5 = [15000.0, 9000.0, 4000.0]; a6 = [5.0, 4.0, 6.0]          # species of _two(): A + B <=> C
    da0 = a0[2] - a0[0] - a0[1]; da5 = a5[2] - a5[0] - a5[1]; da6 = a6[2] - a6[0] - a6[1]; snu = -1
    Ar = ARR["A"] * math.exp(da0 - da6) * (R / PATM) ** snu
    rp = (Ar, ARR["beta"] - da0 + snu, ARR["Ta"] - da5)
    ref = _run(_two(**extra, **ARR))
    exp_ = _run(_two(rev_params=rp, **extra, **ARR))
    assert exp_[1]["kr"][0] == pytest.approx(ref[1]["kr"][0], rel=1e-12)
    np.testing.assert_allclose(exp_[2], ref[2], rtol=1e-11)
    np.testing.assert_allclose(exp_[3], ref[3], rtol=1e-9, atol=1e-12 * np.abs(ref[3]).max())


def test_explicit_reverse_value():
    """k_r is the Arrhenius expression itself, whatever the thermo says."""
    rp = (5.0e11, -0.2, 9000.0)
    r = _run(_two(rev_params=rp, **ARR))
    T = 1300.0
    assert r[1]["kr"][0] == pytest.approx(rp[0] * T ** rp[1] * math.exp(-rp[2] / T), rel=1e-14)


# ---- the blending functions BY VALUE (PAPER.md L143 / L430): the textbook Troe and SRI
# formulas are evaluated here in plain Python with the constants written out again (0.75, 1.27, 0.4, 0.67, 0.14) and
# compared with the oracle's F; c and q follow by closed form.  Non-degenerate parameters: F is far from 1. ----
def _troe_F(T, Pr, a, T3, T1, T2):
    Fc = (1.0 - a) * math.exp(-T / T3) + a * math.exp(-T / T1) + (math.exp(-T2 / T) if T2 is not None else 0.0)
    lc = math.log10(Fc)
    n = 0.75 - 1.27 * lc
    cc = -0.4 - 0.67 * lc
    x = (math.log10(Pr) + cc) / (n - 0.14 * (math.log10(Pr) + cc))
    return 10.0 ** (lc / (1.0 + x * x))


def _sri_F(T, Pr, a, b, c, d, e):
    X = 1.0 / (1.0 + math.log10(Pr) ** 2)
    return d * (a * math.exp(-b / T) + math.exp(-T / c)) ** X * T ** e


BLEND_CASES = [
    ("troe", (0.6, 250.0, 1800.0, None), (6e15, -1.0, 20000.0), dict(T=1300.0)),
    ("troe", (0.35, 90.0, 4200.0, 5200.0), (6e16, -1.2, 19000.0), dict(T=900.0, P=12 * PATM)),
    ("troe", (0.82, 700.0, 950.0, 2600.0), (2e14, -0.4, 21000.0), dict(T=2100.0, P=0.7 * PATM)),
    ("sri", (0.9, 350.0, 1200.0, 1.4, 0.0), (6e15, -1.0, 20000.0), dict(T=1300.0)),
    ("sri", (1.6, 800.0, 600.0, 0.8, 0.15), (6e16, -1.2, 19000.0), dict(T=1700.0, P=25 * PATM)),
    ("sri", (0.45, 150.0, 3000.0, 1.3, -0.1), (2e14, -0.4, 21000.0), dict(T=850.0, P=0.5 * PATM)),
]


@pytest.mark.parametrize("kind,par,low,st", BLEND_CASES)
def test_blend_value_against_textbook_formula(kind, par, low, st):
    if kind == "troe":
        m = _three(type=mg.FALLOFF_TROE, low=low, troe=par, **ARR)
    else:
        m = _three(type=mg.FALLOFF_SRI, low=low, sri=par, **ARR)
    o, it, f, _ = _run(m, **st)
    T = st.get("T", 1300.0); P = st.get("P", 3 * PATM)
    Ctot = P / (R * T)
    k0 = low[0] * T ** low[1] * math.exp(-low[2] / T)
    kinf = ARR["A"] * T ** ARR["beta"] * math.exp(-ARR["Ta"] / T)
    Pr = k0 * Ctot / kinf                                  # default efficiencies: [M] = C_tot
    assert it["Pr"][0] == pytest.approx(Pr, rel=1e-13)
    F = _troe_F(T, Pr, *par) if kind == "troe" else _sri_F(T, Pr, *par)
    assert abs(F - 1.0) > 0.02                             # a non-degenerate case
    assert it["F"][0] == pytest.approx(F, rel=1e-13)
    c = F * Pr / (1.0 + Pr)                                # c_i = F P_r / (1 + P_r)
    assert it["c"][0] == pytest.approx(c, rel=1e-13)
    CA = 0.3 * Ctot; CB = 0.2 * Ctot; CC = 0.1 * Ctot     # mole fractions of _state
    q = c * (kinf * CA - it["kr"][0] * CB * CC)            # q = c (k_inf C_A - k_r C_B C_C)
    assert it["q"][0] == pytest.approx(q, rel=1e-12)
    assert f[2] == pytest.approx(-0.05 * q, rel=1e-12)     # dn_A/dt = -V q (V = 0.05)


# ---- several P-Log entries per pressure (reading R10: the rates of equal-pressure entries are summed) ----
def test_plog_several_entries_per_pressure():
    T = 1300.0
    arr = lambda A, b, Ta: A * T ** b * math.exp(-Ta / T)
    e1a, e1b = (1e10, 0.0, 5000.0), (3e7, 0.9, 2500.0)
    e2a, e2b, e2c = (1e12, 0.5, 8000.0), (5e9, 0.2, 3000.0), (2e11, -0.3, 6000.0)
    pts = [(1.0 * PATM,) + e1a, (1.0 * PATM,) + e1b, (10.0 * PATM,) + e2a, (10.0 * PATM,) + e2b, (10.0 * PATM,) + e2c]
    m = _three(type=mg.PLOG, plog=pts)
    k1 = arr(*e1a) + arr(*e1b); k2 = arr(*e2a) + arr(*e2b) + arr(*e2c)
    # on the nodes and outside the table: the SUM at that pressure
    for P, k in ((1.0 * PATM, k1), (0.3 * PATM, k1), (10.0 * PATM, k2), (55.0 * PATM, k2)):
        _, it, _, _ = _run(m, P=P)
        assert it["kf"][0] == pytest.approx(k, rel=1e-13)
    # between the levels: log-log interpolation of the sums
    _, it, _, _ = _run(m, P=math.sqrt(10.0) * PATM)
    assert it["kf"][0] == pytest.approx(math.sqrt(k1 * k2), rel=1e-12)
    w = math.log(2.0) / math.log(10.0)
    _, it, _, _ = _run(m, P=2.0 * PATM)
    assert it["kf"][0] == pytest.approx(k1 ** (1 - w) * k2 ** w, rel=1e-12)
    # two identical entries = one entry with 2A: source terms and Jacobian, inside and outside the table
    twice = [(p * PATM, A, b, Ta) for (p, A, b, Ta) in ((1.0, 1e10, 0.0, 5000.0), (10.0, 1e12, 0.5, 8000.0)) for _ in range(2)]
    once = [(1.0 * PATM, 2e10, 0.0, 5000.0), (10.0 * PATM, 2e12, 0.5, 8000.0)]
    for P in (0.5 * PATM, 1.0 * PATM, 3.0 * PATM, 10.0 * PATM, 40.0 * PATM):
        a = _run(_three(type=mg.PLOG, plog=twice), P=P); b = _run(_three(type=mg.PLOG, plog=once), P=P)
        np.testing.assert_allclose(a[2], b[2], rtol=1e-13)
        np.testing.assert_allclose(a[3], b[3], rtol=1e-11, atol=1e-300)
    # the analytical Jacobian of the summed form against the complex step of the oracle's own source terms
    o = Oracle(m)
    for P in (0.3 * PATM, 2.0 * PATM, 10.0 * PATM, 70.0 * PATM):
        phi, Pp = _state(P=P)
        J = o.jacobian_dense(mg.CONP, phi, [Pp])[0]
        Jc = o.cs_jacobian(mg.CONP, phi, Pp)
        tol = np.maximum(1e-11 * np.abs(Jc), 1e-15 * np.abs(Jc).max(axis=1, keepdims=True))
        assert np.all(np.abs(J - Jc) <= tol)
