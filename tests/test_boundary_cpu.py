"""CPU-side checks of the product: the library loads, exports every symbol of include/pyjac.h, host
preprocessing (pattern, validation) works without a GPU, and compute calls fail loudly."""
import ctypes
import os
import re

import numpy as np
import pytest

import mechgen as mg
import paper_1809_01029_b200 as pj
from oracle import Oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "pyjac.h")).read()
    names = set(re.findall(r"\b(pyjac_[a-z_]+)\s*\(", hdr))
    assert {"pyjac_mech_create", "pyjac_mech_destroy", "pyjac_mech_dims", "pyjac_sparsity", "pyjac_source_terms",
            "pyjac_jacobian_sparse", "pyjac_jacobian_dense", "pyjac_jacobian_fd", "pyjac_eval_host", "pyjac_launch_info",
            "pyjac_last_error"} <= names
    lib = ctypes.CDLL(pj.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n


@pytest.mark.parametrize("name", ["four", "four_b", "all_types", "all_types_inert", "chem", "revx", "c1", "c2", "c3", "c4"])
def test_pattern_bit_exact_vs_oracle(name):
    m = {"four": lambda: mg.hand_four(), "four_b": lambda: mg.hand_four(order=(1, 2, 3, 0)), "chem": mg.hand_chem_activated, "revx": mg.hand_rev_explicit,
         "all_types": lambda: mg.hand_all_types(True, True), "all_types_inert": lambda: mg.hand_all_types(False, False)}.get(
        name, lambda: mg.config_mechanism(int(name[1:])))()
    M = pj.Mechanism(m, -1)
    o = Oracle(m)
    assert (M.ns, M.nr, M.nvar, M.nnz) == (o.ns, o.nr, o.nvar, o.nnz)
    for fmt in (mg.CSR, mg.CSC):
        p, i = M.sparsity(fmt); po, io = o.pattern(fmt)
        assert p.dtype == np.int32 and p.tobytes() == po.tobytes() and i.tobytes() == io.tobytes()


def test_equal_nondefault_efficiencies_are_structural_zeros():
    """alpha_ij == alpha_i,Ns (both non-default) cancels identically: not a pattern entry (rule R5)."""
    mb = mg.MechBuilder()
    cp = lambda a0: [a0, 0, 0, 0, 0, 100.0, 3.0]
    for W in (10.0, 10.0, 12.0, 28.0):
        mb.add_species(W, cp(3.0))
    mb.add_reaction({0: 1}, {1: 1}, A=1e6, rev=True, type=mg.THIRD_BODY, eff={2: 2.0, 3: 2.0})
    m = mb.build()
    M = pj.Mechanism(m, -1); o = Oracle(m)
    assert M.sparsity(0)[1].tobytes() == o.pattern(0)[1].tobytes()
    ptr, idx = M.sparsity(0)
    assert list(idx[ptr[2]:ptr[3]]) == [0, 1, 2, 3]          # row of species 0: T, E, n0, n1 -- NOT n2


def test_compute_fails_loudly_without_gpu():
    M = pj.Mechanism(mg.hand_ab(), -1)
    with pytest.raises(pj.PyjacError) as e:
        pj.pyjac_source_terms(M.h, 0, 1, 1, 1, 16, 16, 16)
    assert e.value.code == pj.PYJAC_ECUDA
    with pytest.raises(pj.PyjacError):
        pj.pyjac_eval_host(M.h, 0, 0, 0, 1, 1, 1, np.zeros(3), np.zeros(1), np.zeros(3))


def _bad(mut):
    m = dict(mg.hand_four())
    m = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in m.items()}
    mut(m)
    with pytest.raises(pj.PyjacError) as e:
        pj.Mechanism(m, -1)
    assert e.value.code == pj.PYJAC_EMECH
    return str(e.value)


def test_mechanism_validation_errors():
    assert "n_species" in _bad(lambda m: m.update(n_species=1))
    assert "out of range" in _bad(lambda m: m["reac_species"].__setitem__(0, 9))
    assert "coefficient" in _bad(lambda m: m["reac_nu"].__setitem__(0, 4))
    assert "A must be" in _bad(lambda m: m["A"].__setitem__(0, 0.0))
    assert "weight" in _bad(lambda m: m["mol_weight"].__setitem__(1, -1.0))
    assert "efficiency" in _bad(lambda m: m["eff_value"].__setitem__(0, -0.5))
    assert "type" in _bad(lambda m: m["type"].__setitem__(0, 9))
    assert "low-pressure" in _bad(lambda m: m["low_A"].__setitem__(2, 0.0))
    assert "chem_activated" in _bad(lambda m: m["chem_activated"].__setitem__(0, 1))       # reaction 0 is elementary
    assert "explicit reverse" in _bad(lambda m: m["rev_A"].__setitem__(0, -1.0))
    assert "explicit reverse" in _bad(lambda m: (m["rev_A"].__setitem__(0, 1.0), m["reversible"].__setitem__(0, 0)))

    def plog_bad(m):
        m["type"][0] = mg.PLOG
        m["plog_ptr"] = np.array([0, 2, 2, 2], np.int32)
        m["plog_P"] = np.array([2e5, 1e5]); m["plog_A"] = np.array([1.0, 1.0])
        m["plog_beta"] = np.zeros(2); m["plog_Ta"] = np.zeros(2)
    assert "ascending" in _bad(plog_bad)

    def cheb_bad(m):
        m["type"][0] = mg.CHEBYSHEV
    assert "Chebyshev" in _bad(cheb_bad)


def test_graft_entry_build_imports():
    import __graft_entry__ as g
    assert callable(g.build) and callable(g.smoke)


def test_validation_rejects_what_the_tables_cannot_hold():
    """|sum nu| > 7 does not fit the packed reaction word; NULL required arrays and decreasing pointer arrays."""
    from mechgen import MechBuilder
    cp = [3.5, 0, 0, 0, 0, 0.0, 1.0]
    mb = MechBuilder()
    for w in (90.0, 10.0, 10.0, 10.0, 28.0):
        mb.add_species(w, cp)
    mb.add_reaction({0: 1}, {1: 3, 2: 3, 3: 3}, 1e5, 0.0, 1000.0, rev=False)       # sum nu = +8
    with pytest.raises(pj.PyjacError) as ei:
        pj.Mechanism(mb.build(), -1)
    assert ei.value.code == pj.PYJAC_EMECH and "exceeds 7" in str(ei.value)
    m = dict(mg.config_mechanism(1))
    bad = dict(m); p = np.array(m["reac_ptr"]).copy(); p[3] = p[2] - 1; bad["reac_ptr"] = p
    with pytest.raises(pj.PyjacError) as ei:
        pj.Mechanism(bad, -1)
    assert ei.value.code == pj.PYJAC_EMECH
    d, keep = pj.make_desc(m)
    d.nasa_lo = None
    h = ctypes.c_void_p()
    rc = pj.lib().pyjac_mech_create(ctypes.byref(d), -1, ctypes.byref(h))
    assert rc == pj.PYJAC_EMECH and b"NULL" in pj.lib().pyjac_last_error()


def test_launch_info_is_the_one_launch_policy():
    M = pj.Mechanism(mg.config_mechanism(2), -1)
    S_big, nt, smem = pj.pyjac_launch_info(M.h, pj.WHAT_SPARSE)
    assert S_big == 8 and nt == 512 and 0 < smem <= 227 * 1024
    assert pj.pyjac_launch_info(M.h, pj.WHAT_SPARSE, 1 << 17, 4)[0] == 4          # never more states than the layout tile
    assert pj.pyjac_launch_info(M.h, pj.WHAT_SPARSE, 296 * 8, 8)[0] == 8          # two tiles per SM (148 on a host-only handle)
    assert pj.pyjac_launch_info(M.h, pj.WHAT_SPARSE, 296 * 8 - 8, 8)[0] == 4
    assert pj.pyjac_launch_info(M.h, pj.WHAT_SPARSE, 100, 1 << 20)[0] == 1
