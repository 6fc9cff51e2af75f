"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element."""
import numpy as np
import pytest

import mechgen as mg
from mechgen.mechanism import pack_phi
from tests.util import unpack, source_ok, jac_ok_dense, dense_from_sparse

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pj():
    import paper_1809_01029_b200 as pj_
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    pj_.lib()
    return pj_


_CACHE = {}


def setup(pj, name):
    if name not in _CACHE:
        from oracle import Oracle
        if name == "all_types":
            m = mg.hand_all_types(True, True); st = lambda n: mg.make_states(6, n, 21)
        elif name == "four":
            m = mg.hand_four(); st = lambda n: mg.make_states(4, n, 22)
        elif name == "chem":
            m = mg.hand_chem_activated(); st = lambda n: mg.make_states(5, n, 23)
        elif name == "revx":
            m = mg.hand_rev_explicit(); st = lambda n: mg.make_states(6, n, 24)
        else:
            c = int(name[1:]); m = mg.config_mechanism(c); st = lambda n, c=c: mg.config_states(c, n)
        _CACHE[name] = (m, pj.Mechanism(m, 0), Oracle(m), st)
    return _CACHE[name]


def run_gpu(pj, M, what, mode, fmt, states, ld=None, tile=None):
    N = states["T"].shape[0]
    ld = N if ld is None else ld
    tile = ld if tile is None else tile
    phi, par = pack_phi(states, mode, ld, tile)
    d_phi = torch.from_numpy(phi).cuda(); d_par = torch.from_numpy(par).cuda()
    n_e = M.n_elements(what)
    out = torch.full((n_e * ld,), float("nan"), dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    if what == pj.WHAT_SOURCE:
        pj.pyjac_source_terms(M.h, mode, N, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), st)
    elif what == pj.WHAT_SPARSE:
        pj.pyjac_jacobian_sparse(M.h, mode, fmt, N, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), st)
    else:
        pj.pyjac_jacobian_dense(M.h, mode, fmt, N, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), st)
    torch.cuda.synchronize()
    full = out.cpu().numpy()
    res = unpack(full, n_e, N, ld, tile)
    # slots of states >= n_states are never written
    if ld > N:
        pad = np.asarray(full).reshape(ld // tile, n_e, tile).transpose(0, 2, 1).reshape(ld, n_e)[N:]
        assert np.isnan(pad).all()
    return res


SRC_CASES = [("four", 64), ("all_types", 300), ("chem", 200), ("revx", 200), ("c1", 1024), ("c2", 1500), ("c3", 700), ("c4", 96), ("c5", 96)]


@pytest.mark.parametrize("name,n", SRC_CASES)
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
def test_source_terms(pj, name, n, mode):
    m, M, o, st = setup(pj, name)
    states = st(n)
    got = run_gpu(pj, M, pj.WHAT_SOURCE, mode, 0, states)
    ref = o.source(mode, *o.pack(states, mode))
    assert source_ok(got, ref) <= 1.0


JAC_CASES = [("four", 64), ("all_types", 300), ("chem", 200), ("revx", 200), ("c1", 1024), ("c2", 600), ("c3", 200), ("c4", 24), ("c5", 24)]


@pytest.mark.parametrize("name,n", JAC_CASES)
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
@pytest.mark.parametrize("fmt", [mg.CSR, mg.CSC])
def test_jacobian_sparse(pj, name, n, mode, fmt):
    m, M, o, st = setup(pj, name)
    states = st(n)
    ptr, idx = M.sparsity(fmt)
    optr, oidx = o.pattern(fmt)
    assert ptr.tobytes() == optr.tobytes() and idx.tobytes() == oidx.tobytes()      # bit-exact pattern
    got = run_gpu(pj, M, pj.WHAT_SPARSE, mode, fmt, states)
    Jg = dense_from_sparse(got, ptr, idx, fmt, M.nvar)
    Jr = o.jacobian_dense(mode, *o.pack(states, mode))
    bad = jac_ok_dense(Jg, Jr)
    assert not bad.any(), (np.argwhere(bad)[:5], Jg[bad][:5], Jr[bad][:5])


@pytest.mark.parametrize("name,n", JAC_CASES)
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
@pytest.mark.parametrize("order", ["C", "F"])
def test_jacobian_dense(pj, name, n, mode, order):
    m, M, o, st = setup(pj, name)
    states = st(n)
    got = run_gpu(pj, M, pj.WHAT_DENSE, mode, order, states).reshape(n, M.nvar, M.nvar)
    if order == "F":
        got = got.transpose(0, 2, 1)
    Jr = o.jacobian_dense(mode, *o.pack(states, mode))
    bad = jac_ok_dense(got, Jr)
    assert not bad.any(), (np.argwhere(bad)[:5], got[bad][:5], Jr[bad][:5])
    ptr, idx = M.sparsity(mg.CSR)
    pat = dense_from_sparse(np.ones((1, M.nnz)), ptr, idx, mg.CSR, M.nvar)[0] != 0
    assert np.all(got[:, ~pat] == 0.0)                 # structural zeros stored as exact 0.0


@pytest.mark.parametrize("name,n,ld,tile", [("c2", 1000, 1024, 1024), ("c2", 1000, 1024, 8), ("c2", 999, 1000, 1),
                                             ("c2", 37, 64, 4), ("c1", 1, 1, 1), ("c1", 5, 32, 32), ("c3", 130, 256, 2),
                                             ("c5", 19, 20, 1), ("c5", 19, 32, 4)])
def test_layouts_and_ragged_tails(pj, name, n, ld, tile):
    m, M, o, st = setup(pj, name)
    states = st(n)
    for mode in (mg.CONP, mg.CONV):
        ref = o.source(mode, *o.pack(states, mode))
        got = run_gpu(pj, M, pj.WHAT_SOURCE, mode, 0, states, ld, tile)
        assert source_ok(got, ref) <= 1.0
        Jr = o.jacobian_dense(mode, *o.pack(states, mode))
        ptr, idx = M.sparsity(mg.CSR)
        got = run_gpu(pj, M, pj.WHAT_SPARSE, mode, mg.CSR, states, ld, tile)
        assert not jac_ok_dense(dense_from_sparse(got, ptr, idx, mg.CSR, M.nvar), Jr).any()
        got = run_gpu(pj, M, pj.WHAT_DENSE, mode, "C", states, ld, tile).reshape(n, M.nvar, M.nvar)
        assert not jac_ok_dense(got, Jr).any()


def test_empty_and_errors(pj):
    m, M, o, st = setup(pj, "c1")
    buf = torch.zeros(4096, dtype=torch.float64, device="cuda")
    p = buf.data_ptr()
    pj.pyjac_source_terms(M.h, 0, 0, 0, 1, 0, 0, 0)                     # n_states = 0 is a no-op
    pj.pyjac_jacobian_sparse(M.h, 0, 0, 0, 16, 16, p, p, p)
    for bad in (lambda: pj.pyjac_source_terms(M.h, 2, 4, 4, 4, p, p, p),        # bad mode
                lambda: pj.pyjac_source_terms(M.h, 0, 8, 4, 4, p, p, p),        # ld < n
                lambda: pj.pyjac_source_terms(M.h, 0, 4, 12, 3, p, p, p),       # tile not pow2
                lambda: pj.pyjac_source_terms(M.h, 0, 4, 6, 4, p, p, p),        # ld % tile
                lambda: pj.pyjac_source_terms(M.h, 0, 4, 4, 4, p + 8, p, p),    # misaligned
                lambda: pj.pyjac_source_terms(M.h, 0, 4, 4, 4, 0, p, p),        # null
                lambda: pj.pyjac_jacobian_sparse(M.h, 0, 7, 4, 4, 4, p, p, p),  # bad fmt
                lambda: pj.pyjac_jacobian_dense(M.h, 0, "X", 4, 4, 4, p, p, p)):
        with pytest.raises(pj.PyjacError) as ei:
            bad()
        assert ei.value.code == pj.PYJAC_EINVAL


def test_eval_host_matches_device_path(pj):
    m, M, o, st = setup(pj, "c2")
    states = st(256)
    phi, par = pack_phi(states, mg.CONP, 256, 256)
    out = np.empty(M.nnz * 256)
    pj.pyjac_eval_host(M.h, pj.WHAT_SPARSE, mg.CONP, mg.CSR, 256, 256, 256, phi, par, out)
    got = run_gpu(pj, M, pj.WHAT_SPARSE, mg.CONP, mg.CSR, states)
    # not bitwise: warps take reaction chunks dynamically, so the order of the reaction sums varies run to run
    np.testing.assert_allclose(unpack(out, M.nnz, 256, 256, 256), got, rtol=1e-11, atol=0)


@pytest.mark.parametrize("c", [5, 4])
def test_full_size_bench_configuration_sampled(pj, c):
    """BASELINE.json's full sizes in the launch configuration bench.py times (tile = states per CTA): C5 2^18 states
    sparse CSR (26.8 GB of values), C4 2^14 states dense (17.1 GB); 48 states sampled across the batch (including the
    first and the last) are compared with the oracle one by one, and a checksum guards every state against NaN."""
    from mechgen.mechanism import CONFIGS
    m, M, o, st = setup(pj, "c%d" % c)
    cfg = CONFIGS[c]
    N, mode = cfg["n_states"], cfg["mode"]
    what = pj.WHAT_SPARSE if c == 5 else pj.WHAT_DENSE
    n_e = M.n_elements(what)
    free, _ = torch.cuda.mem_get_info()
    if free < n_e * N * 8 + (2 << 30):
        pytest.skip("not enough device memory for the full-size buffer")
    S, _, _ = pj.pyjac_launch_info(M.h, 1)
    tile = S
    states = st(N)
    phi, par = pack_phi(states, mode, N, tile)
    d_phi = torch.from_numpy(phi).cuda(); d_par = torch.from_numpy(par).cuda()
    out = torch.empty(n_e * N, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    if c == 5:
        pj.pyjac_jacobian_sparse(M.h, mode, mg.CSR, N, N, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), stream)
    else:
        pj.pyjac_jacobian_dense(M.h, mode, "C", N, N, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), stream)
    torch.cuda.synchronize()
    view = out.view(N // tile, n_e, tile)
    assert bool(torch.isfinite(view.sum(dim=1)).all())
    rng = np.random.default_rng(c)
    pick = np.unique(np.concatenate([[0, N - 1], rng.integers(0, N, 46)]))
    got = np.stack([view[s // tile, :, s % tile].cpu().numpy() for s in pick])
    sub = {k: (v[pick] if v.ndim == 1 else v[:, pick]) for k, v in states.items()}
    Jr = o.jacobian_dense(mode, *o.pack(sub, mode))
    if c == 5:
        ptr, idx = M.sparsity(mg.CSR)
        Jg = dense_from_sparse(got, ptr, idx, mg.CSR, M.nvar)
    else:
        Jg = got.reshape(len(pick), M.nvar, M.nvar)
    bad = jac_ok_dense(Jg, Jr)
    assert not bad.any(), (np.argwhere(bad)[:5], Jg[bad][:5], Jr[bad][:5])
    del out
    torch.cuda.empty_cache()
