"""pyjac_jacobian_sparse_static (include/pyjac.h): the allocation-free entry point -- the persistent Jacobian kernel with
its scratch (tile counter, finished-CTA counter) in a file-scope static __device__ array -- against the existing path
pyjac_jacobian_sparse, on two calls in a row.  Collected last on purpose (the suite runs with pytest -x); it passes
alone in a fresh process and after the other tests (the static scratch keeps the last call's contents and is cleared by
every call)."""
import numpy as np
import pytest

import mechgen as mg
from mechgen.mechanism import pack_phi
from tests.util import unpack, jac_ok_dense, dense_from_sparse

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _run(pj, fn, M, mode, fmt, states, ld, tile, stream):
    n = states["T"].shape[0]
    phi, par = pack_phi(states, mode, ld, tile)
    d_phi = torch.from_numpy(phi).cuda(); d_par = torch.from_numpy(par).cuda()
    out = torch.full((M.nnz * ld,), float("nan"), dtype=torch.float64, device="cuda")
    fn(M.h, mode, fmt, n, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), stream.cuda_stream)
    stream.synchronize()
    full = out.cpu().numpy()
    if ld > n:      # slots of states >= n_states are never written
        assert np.isnan(full.reshape(ld // tile, M.nnz, tile).transpose(0, 2, 1).reshape(ld, M.nnz)[n:]).all()
    return unpack(full, M.nnz, n, ld, tile)


@pytest.mark.parametrize("name,flags", [("c2", 0), ("c2", 2), ("c5", 0)])
def test_static_scratch_entry_point_matches_the_existing_path(name, flags):
    import paper_1809_01029_b200 as pj
    from oracle import Oracle
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    c = int(name[1:])
    mech = mg.config_mechanism(c)
    M = pj.Mechanism(mech, 0, flags)
    o = Oracle(mech)
    S, _, _ = pj.pyjac_launch_info(M.h, pj.WHAT_SPARSE)
    stream = torch.cuda.Stream()
    ptr, idx = M.sparsity(mg.CSR)
    # two calls in a row on one stream, different batches (sizes, modes, ragged tails): the second one starts from the
    # scratch the first one left behind
    calls = [(2200 if c == 2 else 310, mg.CONP, S), (1237 if c == 2 else 151, mg.CONV, 1), (2200 if c == 2 else 310, mg.CONP, S)]
    for n, mode, tile in calls:
        states = mg.config_states(c, n)
        ld = (n + tile - 1) // tile * tile
        ref = _run(pj, pj.pyjac_jacobian_sparse, M, mode, mg.CSR, states, ld, tile, stream)
        got = _run(pj, pj.pyjac_jacobian_sparse_static, M, mode, mg.CSR, states, ld, tile, stream)
        assert np.isfinite(got).all()                      # a skipped tile would leave NaN behind
        # the two paths run the same kernel; launches differ in the last bits only (dynamic chunk order): compared with
        # the parity tolerance of the Jacobian tests (tests/util.py), and a sample with the oracle itself
        Jg, Jx = dense_from_sparse(got, ptr, idx, mg.CSR, M.nvar), dense_from_sparse(ref, ptr, idx, mg.CSR, M.nvar)
        assert not jac_ok_dense(Jg, Jx).any()
        pick = np.unique(np.concatenate([[0, n - 1], np.arange(0, n, max(1, n // 12))]))
        sub = {k: (v[pick] if v.ndim == 1 else v[:, pick]) for k, v in states.items()}
        Jr = o.jacobian_dense(mode, *o.pack(sub, mode))
        assert not jac_ok_dense(Jg[pick], Jr).any()


def test_static_entry_point_rejects_oversize_and_bad_arguments():
    import paper_1809_01029_b200 as pj
    M = pj.Mechanism(mg.config_mechanism(1), 0)
    buf = torch.zeros(4096, dtype=torch.float64, device="cuda")
    p = buf.data_ptr()
    big = pj.PYJAC_STATIC_MAX_STATES + 1
    with pytest.raises(pj.PyjacError) as ei:
        pj.pyjac_jacobian_sparse_static(M.h, 0, 0, big, big, big, p, p, p)
    assert ei.value.code == pj.PYJAC_EINVAL and "PYJAC_STATIC_MAX_STATES" in str(ei.value)
    with pytest.raises(pj.PyjacError) as ei:
        pj.pyjac_jacobian_sparse_static(M.h, 0, 7, 4, 4, 4, p, p, p)            # bad fmt
    assert ei.value.code == pj.PYJAC_EINVAL
    pj.pyjac_jacobian_sparse_static(M.h, 0, 0, 0, 0, 1, 0, 0, 0)                # n_states = 0 is a no-op
