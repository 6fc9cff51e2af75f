"""The paper's "approximate" Jacobian (R6): oracle pins (CPU) and GPU parity."""
import numpy as np
import pytest

import mechgen as mg
import paper_1809_01029_b200 as pj
from oracle import Oracle
from tests.util import jac_ok_dense, dense_from_sparse

CASES = {
    "c3": lambda: (mg.config_mechanism(3), mg.config_states(3, 6)),
    "all_types": lambda: (mg.hand_all_types(True, True), mg.make_states(6, 6, 31)),
    "all_types_eff_only": lambda: (mg.hand_all_types(False, True), mg.make_states(6, 6, 32)),
    "four_b": lambda: (mg.hand_four(order=(1, 2, 3, 0)), mg.make_states(4, 6, 33)),
}


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
def test_oracle_approx_equals_derivative_with_last_species_frozen_in_the_rates(name, mode):
    """Pin: the approximate Jacobian is the exact derivative of f when, for the species columns, the rate
    expressions see C_Ns as a constant and [M] = C_tot + sum (alpha_k - 1) C_k (complex step of that function)."""
    m, st = CASES[name]()
    o = Oracle(m, approx=True)
    phi, par = o.pack(st, mode)
    J = o.jacobian_dense(mode, phi, par)
    for s in range(phi.shape[0]):
        Jc = o.cs_jacobian(mode, phi[s], par[s])
        rowmax = np.abs(Jc).max(axis=1, keepdims=True)
        tol = np.maximum(np.maximum(1e-8 * np.abs(Jc), 1e-12 * rowmax), 1e-300)
        assert (np.abs(J[s] - Jc) / tol).max() < 1e-3


@pytest.mark.parametrize("c", [1, 2, 4])
def test_oracle_approx_is_exact_when_last_species_is_inert_with_default_efficiency(c):
    m = mg.config_mechanism(c)
    st = mg.config_states(c, 2)
    oa, oe = Oracle(m, approx=True), Oracle(m)
    assert oa.nnz == oe.nnz and oa.pattern(0)[1].tobytes() == oe.pattern(0)[1].tobytes()
    phi, par = oe.pack(st, mg.CONP)
    np.testing.assert_array_equal(oa.jacobian_dense(mg.CONP, phi, par), oe.jacobian_dense(mg.CONP, phi, par))


@pytest.mark.parametrize("name", list(CASES))
def test_approx_pattern_subset_T_E_columns_exact_and_brute_force(name):
    m, st = CASES[name]()
    oa, oe = Oracle(m, approx=True), Oracle(m)
    nvar = oa.nvar

    def mask(o):
        ptr, idx = o.pattern(mg.CSR)
        return dense_from_sparse(np.ones((1, o.nnz)), ptr, idx, mg.CSR, nvar)[0] != 0
    ma, me = mask(oa), mask(oe)
    assert np.all(me[ma]) and ma.sum() <= me.sum()                       # approximate pattern is a subset
    if name != "all_types_eff_only":
        assert ma.sum() < me.sum() or name == "all_types"
    nz = np.zeros((nvar, nvar), bool)
    for mode in (mg.CONP, mg.CONV):
        phi, par = oa.pack(st, mode)
        Ja, Je = oa.jacobian_dense(mode, phi, par), oe.jacobian_dense(mode, phi, par)
        np.testing.assert_allclose(Ja[:, :, :2], Je[:, :, :2], rtol=1e-13, atol=0)    # T and E columns unchanged
        assert np.all(Ja[:, ~ma] == 0.0)
        for s in range(phi.shape[0]):
            nz |= oa.cs_jacobian(mode, phi[s], par[s]) != 0.0
    assert np.array_equal(nz[2:, 2:], ma[2:, 2:])                        # rule == numerical nonzeros (frozen CS)
    # product pattern (host-only handle) is bit-exact
    M = pj.Mechanism(m, -1, pj.PYJAC_APPROX_JACOBIAN)
    for fmt in (mg.CSR, mg.CSC):
        p, i = M.sparsity(fmt); po, io = oa.pattern(fmt)
        assert p.tobytes() == po.tobytes() and i.tobytes() == io.tobytes()


def test_unknown_flag_rejected():
    with pytest.raises(pj.PyjacError) as e:
        pj.pyjac_mech_create_ex(mg.hand_ab(), -1, 8)
    assert e.value.code == pj.PYJAC_EINVAL


@pytest.mark.gpu
@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
def test_gpu_approx_parity(name, mode):
    import torch
    from mechgen.mechanism import pack_phi
    from tests.util import unpack
    m, _ = CASES[name]()
    n = 200 if name != "c3" else 96
    st = mg.config_states(3, n) if name == "c3" else mg.make_states(m["n_species"], n, 77)
    M = pj.Mechanism(m, 0, pj.PYJAC_APPROX_JACOBIAN)
    o = Oracle(m, approx=True)
    Jr = o.jacobian_dense(mode, *o.pack(st, mode))
    phi, par = pack_phi(st, mode)
    d_phi = torch.from_numpy(phi).cuda(); d_par = torch.from_numpy(par).cuda()
    for fmt in (mg.CSR, mg.CSC):
        out = torch.empty(M.nnz * n, dtype=torch.float64, device="cuda")
        pj.pyjac_jacobian_sparse(M.h, mode, fmt, n, n, n, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), 0)
        torch.cuda.synchronize()
        ptr, idx = M.sparsity(fmt)
        Jg = dense_from_sparse(unpack(out.cpu().numpy(), M.nnz, n, n, n), ptr, idx, fmt, M.nvar)
        assert not jac_ok_dense(Jg, Jr).any()
    out = torch.empty(M.nvar * M.nvar * n, dtype=torch.float64, device="cuda")
    pj.pyjac_jacobian_dense(M.h, mode, "C", n, n, n, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), 0)
    torch.cuda.synchronize()
    Jg = unpack(out.cpu().numpy(), M.nvar * M.nvar, n, n, n).reshape(n, M.nvar, M.nvar)
    assert not jac_ok_dense(Jg, Jr).any()
