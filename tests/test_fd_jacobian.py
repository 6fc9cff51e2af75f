"""First-order forward finite-difference Jacobian, the paper's comparison baseline (Fig. 12;
step rule DESIGN.md R7).

CPU part (pin P13): the oracle's fd1_jacobian against things it does not compute itself -- the analytical Jacobian
(itself pinned by complex step, P4) with the O(h) truncation error a forward difference must show, and a case where
the forward difference is exact.  GPU part: pyjac_jacobian_fd through the C ABI against the oracle, entry by entry,
with the tolerance the source-term tolerance implies for a difference quotient."""
import numpy as np
import pytest

import mechgen as mg
from mechgen.mechanism import pack_phi
from oracle import Oracle
from tests.util import unpack, dense_from_sparse

REL = 2.0 ** -26          # sqrt(eps)
ABS = 1e-14


def _states(name, n):
    if name == "all_types":
        return mg.hand_all_types(True, True), mg.make_states(6, n, 21)
    if name == "four":
        return mg.hand_four(), mg.make_states(4, n, 22)
    c = int(name[1:])
    return mg.config_mechanism(c), mg.config_states(c, n)


# ---------------------------------------------------------------------------------------------------------------
# CPU: pin P13
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["four", "all_types", "c1"])
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
def test_fd1_converges_to_analytical_at_first_order(name, mode):
    """||J_fd(h) - J|| = O(h): halving the step halves the error (a central or a wrong-sign difference would not),
    and at h = 1e-6 |phi| the two agree to truncation + rounding."""
    m, st = _states(name, 6)
    o = Oracle(m)
    phi, par = o.pack(st, mode)
    J = o.jacobian_dense(mode, phi, par)
    scale = np.abs(J).max(axis=1, keepdims=True) + 1e-300          # per column
    errs = []
    for rel in (4e-5, 2e-5, 1e-5):
        Jf = o.fd1_jacobian(mode, phi, par, rel, 0.0)
        errs.append(np.abs(Jf - J) / scale)
    e0, e1, e2 = errs
    big = e0 > 1e-7                                                # truncation well above rounding (eps/h ~ 1e-11)
    assert big.sum() > 10
    r01 = e0[big] / e1[big]; r12 = e1[big] / e2[big]
    assert np.median(r01) == pytest.approx(2.0, rel=0.05) and np.median(r12) == pytest.approx(2.0, rel=0.05)
    assert (np.abs(r01 - 2.0) < 0.1).mean() > 0.5      # the rest: entries where rounding eps |f| / h dominates
    # closeness: truncation O(rel) of the column scale plus the rounding of the quotient, eps |f_i| / h_c
    rel = 1e-6
    Jf = o.fd1_jacobian(mode, phi, par, rel, 0.0)
    f0 = np.abs(o.source(mode, phi, par))[:, :, None]
    h = (rel * np.abs(phi))[:, None, :]
    assert (np.abs(Jf - J) <= 300 * rel * scale + 64 * 2.2e-16 * f0 / h).all()


def test_fd1_exact_where_f_is_linear():
    """A -> B irreversible, beta = 0, Ta = 0 at constant volume: dn_A/dt = V k C_A = k n_A is LINEAR in n_A, so the
    forward difference equals -k up to rounding (eps |f| / h), whatever the step."""
    mb = mg.MechBuilder()
    cp = [3.5, 0, 0, 0, 0, 100.0, 3.0]
    for W in (20.0, 20.0, 28.0):
        mb.add_species(W, cp)
    k = 3.0e3
    mb.add_reaction({0: 1}, {1: 1}, A=k, beta=0.0, Ta=0.0, rev=False)
    o = Oracle(mb.build())
    st = mg.make_states(3, 4, 5)
    phi, par = o.pack(st, mg.CONV)
    for rel in (1e-3, 1e-6):
        J = o.fd1_jacobian(mg.CONV, phi, par, rel, 0.0)
        np.testing.assert_allclose(J[:, 2, 2], -k, rtol=1e-16 / rel * 50)
        np.testing.assert_allclose(J[:, 3, 2], +k, rtol=1e-16 / rel * 50)


def test_fd1_step_rule():
    """h_c = fl(phi_c + fma(rel, |phi_c|, abs)) - phi_c: with rel = 0 the step is the absolute one, and a column whose
    variable is exactly 0 still gets a step (abs)."""
    m = mg.hand_ab()
    o = Oracle(m)
    st = mg.make_states(2, 1, 3)
    phi, par = o.pack(st, mg.CONP)
    phi = phi.copy(); phi[0, 2] = 0.0
    J = o.fd1_jacobian(mg.CONP, phi, par, REL, 1e-9)
    assert np.isfinite(J).all()
    f0 = o.source(mg.CONP, phi, par)
    x = phi.copy(); x[0, 2] = 1e-9
    f1 = o.source(mg.CONP, x, par)
    np.testing.assert_array_equal(J[0, :, 2], (f1[0] - f0[0]) / 1e-9)


# ---------------------------------------------------------------------------------------------------------------
# GPU parity
# ---------------------------------------------------------------------------------------------------------------
def _fd_tol(o, mode, phi, par, Jref, rel, ab):
    """|dJ(i,c)| <= 1e-10 (|f_i(phi)| + |f_i(phi + h e_c)| + 2e-20) / h_c: the source-term tolerance of BASELINE.json
    applied to the two evaluations of the quotient (R7)."""
    f0 = o.source(mode, phi, par)                                   # [n, nvar]
    xp = phi + (rel * np.abs(phi) + ab)
    h = xp - phi                                                    # [n, nvar] (columns)
    f1 = np.abs(f0[:, :, None] + Jref * h[:, None, :])
    return 1e-10 * (np.abs(f0)[:, :, None] + f1 + 2e-20) / np.abs(h)[:, None, :]


def _run_fd(pj, torch, M, mode, fmt, states, rel, ab, ld=None, tile=None):
    N = states["T"].shape[0]
    ld = N if ld is None else ld
    tile = ld if tile is None else tile
    phi, par = pack_phi(states, mode, ld, tile)
    d_phi = torch.from_numpy(phi).cuda(); d_par = torch.from_numpy(par).cuda()
    n_e = M.nnz if fmt in (mg.CSR, mg.CSC) else M.nvar * M.nvar
    out = torch.full((n_e * ld,), float("nan"), dtype=torch.float64, device="cuda")
    pj.pyjac_jacobian_fd(M.h, mode, fmt, rel, ab, N, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(),
                         torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    full = out.cpu().numpy()
    if ld > N:
        pad = np.asarray(full).reshape(ld // tile, n_e, tile).transpose(0, 2, 1).reshape(ld, n_e)[N:]
        assert np.isnan(pad).all()
    return unpack(full, n_e, N, ld, tile)


_CACHE = {}


def _setup(pj, name):
    if name not in _CACHE:
        m, _ = _states(name, 1)
        _CACHE[name] = (m, pj.Mechanism(m, 0), Oracle(m))
    return _CACHE[name]


FD_CASES = [("four", 33), ("all_types", 40), ("c1", 100), ("c2", 24), ("c3", 6), ("c5", 3)]


@pytest.mark.gpu
@pytest.mark.parametrize("name,n", FD_CASES)
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
def test_fd_dense_and_sparse_vs_oracle(name, n, mode):
    torch = pytest.importorskip("torch")
    import paper_1809_01029_b200 as pj
    m, M, o = _setup(pj, name)
    _, st = _states(name, n)
    phi, par = o.pack(st, mode)
    ref = o.fd1_jacobian(mode, phi, par, REL, ABS)
    tol = _fd_tol(o, mode, phi, par, ref, REL, ABS)
    nvar = M.nvar
    got_c = _run_fd(pj, torch, M, mode, "C", st, REL, ABS).reshape(n, nvar, nvar)
    assert np.isfinite(got_c).all()
    assert (np.abs(got_c - ref) <= tol).all()
    got_f = _run_fd(pj, torch, M, mode, "F", st, REL, ABS).reshape(n, nvar, nvar).transpose(0, 2, 1)
    assert (np.abs(got_f - ref) <= tol).all()
    mask = np.zeros((nvar, nvar), bool)
    for fmt in (mg.CSR, mg.CSC):
        ptr, idx = M.sparsity(fmt)
        vals = _run_fd(pj, torch, M, mode, fmt, st, REL, ABS)
        assert np.isfinite(vals).all()
        Js = dense_from_sparse(vals, ptr, idx, fmt, nvar)
        major = np.repeat(np.arange(nvar), np.diff(ptr))
        mask[:] = False
        if fmt == mg.CSR:
            mask[major, idx] = True
        else:
            mask[idx, major] = True
        assert (np.abs(Js - ref) <= tol)[:, mask].all()
    # outside the exact pattern dJ is identically zero analytically; the quotient is 0 or rounding noise of the
    # cancelling terms (equal efficiencies, C_Ns), already inside tol in the dense comparison above
    assert (np.abs(ref[:, ~mask]) <= tol[:, ~mask]).all() and (np.abs(got_c[:, ~mask]) <= tol[:, ~mask]).all()


@pytest.mark.gpu
@pytest.mark.parametrize("ld,tile", [(64, 64), (64, 1), (64, 4), (56, 8)])
def test_fd_layouts_and_ragged_tail(ld, tile):
    torch = pytest.importorskip("torch")
    import paper_1809_01029_b200 as pj
    m, M, o = _setup(pj, "c1")
    n = 51
    _, st = _states("c1", n)
    phi, par = o.pack(st, mg.CONP)
    ref = o.fd1_jacobian(mg.CONP, phi, par, REL, ABS)
    tol = _fd_tol(o, mg.CONP, phi, par, ref, REL, ABS)
    got = _run_fd(pj, torch, M, mg.CONP, "C", st, REL, ABS, ld, tile).reshape(n, M.nvar, M.nvar)
    assert (np.abs(got - ref) <= tol).all()
    ptr, idx = M.sparsity(mg.CSR)
    vals = _run_fd(pj, torch, M, mg.CONP, mg.CSR, st, REL, ABS, ld, tile)
    major = np.repeat(np.arange(M.nvar), np.diff(ptr))
    assert (np.abs(vals - ref[:, major, idx]) <= tol[:, major, idx]).all()


@pytest.mark.gpu
def test_fd_argument_errors_and_empty():
    torch = pytest.importorskip("torch")
    import paper_1809_01029_b200 as pj
    m, M, o = _setup(pj, "c1")
    buf = torch.zeros(4096, dtype=torch.float64, device="cuda")
    p = buf.data_ptr()
    pj.pyjac_jacobian_fd(M.h, 0, "C", REL, ABS, 0, 0, 1, 0, 0, 0)       # empty batch: no-op
    for args in [(0, 7, REL, ABS), (0, "C", 0.0, 0.0), (0, "C", -1.0, 1.0), (0, "C", float("nan"), 1.0), (2, "C", REL, ABS)]:
        with pytest.raises(pj.PyjacError) as e:
            pj.pyjac_jacobian_fd(M.h, args[0], args[1], args[2], args[3], 1, 1, 1, p, p, p)
        assert e.value.code == pj.PYJAC_EINVAL


@pytest.mark.gpu
def test_fd_approaches_analytical_jacobian():
    """What Fig. 12 compares: the two routes to the same matrix.  At h ~ 1.5e-8 |phi| the GPU finite-difference
    Jacobian agrees with the GPU analytical one to truncation O(h) plus the rounding of the quotient."""
    torch = pytest.importorskip("torch")
    import paper_1809_01029_b200 as pj
    m, M, o = _setup(pj, "c2")
    n = 16
    _, st = _states("c2", n)
    fd = _run_fd(pj, torch, M, mg.CONP, "C", st, REL, 0.0).reshape(n, M.nvar, M.nvar)
    phi, par = pack_phi(st, mg.CONP, n, n)
    d_phi = torch.from_numpy(phi).cuda(); d_par = torch.from_numpy(par).cuda()
    out = torch.empty(M.nvar * M.nvar * n, dtype=torch.float64, device="cuda")
    pj.pyjac_jacobian_dense(M.h, mg.CONP, "C", n, n, n, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr())
    torch.cuda.synchronize()
    an = unpack(out.cpu().numpy(), M.nvar * M.nvar, n, n, n).reshape(n, M.nvar, M.nvar)
    scale = np.abs(an).max(axis=1, keepdims=True)
    phis, pars = o.pack(st, mg.CONP)
    f0 = np.abs(o.source(mg.CONP, phis, pars))[:, :, None]
    h = (REL * np.abs(phis))[:, None, :]
    assert (np.abs(fd - an) <= 300 * REL * scale + 64 * 2.2e-16 * f0 / h).all()      # truncation + rounding eps |f| / h
