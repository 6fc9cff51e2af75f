"""The persistent Jacobian kernel: one CTA per SM takes tiles from a global counter that the last
CTA resets.  These tests exercise what the element-wise parity tests do not: many more tiles than CTAs with a ragged
tail, fewer tiles than CTAs, the scheduler words across more launches than the handle's ring holds, and launches of
one handle on two streams at once.  The reference is the oracle for a sample of states and, for the rest, the kernel's
own result on a batch small enough that every CTA owns exactly one tile (no scheduler involved, parity-tested)."""
import numpy as np
import pytest

import mechgen as mg
from mechgen.mechanism import pack_phi
from tests.util import unpack, jac_ok_dense, dense_from_sparse

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def env():
    import paper_1809_01029_b200 as pj
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    pj.lib()
    m = mg.config_mechanism(2)
    return pj, m, pj.Mechanism(m, 0)


def sparse(pj, M, states, mode, stream=None, ld=None, tile=None):
    N = states["T"].shape[0]
    ld = N if ld is None else ld
    tile = ld if tile is None else tile
    phi, par = pack_phi(states, mode, ld, tile)
    d_phi = torch.from_numpy(phi).cuda(); d_par = torch.from_numpy(par).cuda()
    n_e = M.n_elements(pj.WHAT_SPARSE)
    out = torch.full((n_e * ld,), float("nan"), dtype=torch.float64, device="cuda")
    st = (stream or torch.cuda.current_stream()).cuda_stream
    pj.pyjac_jacobian_sparse(M.h, mode, mg.CSR, N, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), st)
    return out, (d_phi, d_par), (n_e, N, ld, tile)


def host(out, shape):
    return unpack(out.cpu().numpy(), *shape)


def same(M, a, b):
    """Two results of the kernel for the same states.  Not bit-identical: the reaction chunks are handed to the warps
    dynamically, so the order of the reaction sums (and with it the last bits of the T and E rows) varies from run
    to run; the Jacobian tolerance of BASELINE.json is the criterion."""
    ptr, idx = M.sparsity(mg.CSR)
    return not jac_ok_dense(dense_from_sparse(a, ptr, idx, 0, M.nvar), dense_from_sparse(b, ptr, idx, 0, M.nvar)).any()


def test_many_tiles_ragged_tail_matches_oracle_and_small_batches(env):
    pj, m, M = env
    from oracle import Oracle
    N = 148 * 8 * 7 + 5                       # several tiles per CTA at any states-per-CTA, and a ragged last tile
    states = mg.config_states(2, N)
    out, _, shape = sparse(pj, M, states, mg.CONP, ld=N + 3, tile=8)
    torch.cuda.synchronize()
    big = host(out, shape)
    assert np.isfinite(big).all()
    # (i) oracle on a sample that includes the first, the last and tile-boundary states
    O = Oracle(m)
    pick = np.unique(np.r_[0, 1, 7, 8, 148 * 8 - 1, 148 * 8, N - 6, N - 5, N - 1, np.random.default_rng(3).integers(0, N, 40)])
    sub = {k: (v[..., pick] if k == "n" else v[pick]) for k, v in states.items()}
    ref = O.jacobian_dense(mg.CONP, *O.pack(sub, mg.CONP))
    ptr, idx = M.sparsity(mg.CSR)
    got = dense_from_sparse(big[pick], ptr, idx, 0, M.nvar)
    assert not jac_ok_dense(got, ref).any()
    # (ii) ALL states against the same kernel on batches of <= 148 states (one tile per CTA, one state per tile: no
    # scheduler involved; the summation order differs with the states per CTA, hence the Jacobian tolerance)
    for a in range(0, N, 148):
        sl = slice(a, min(a + 148, N))
        part = {k: (v[..., sl] if k == "n" else v[sl]) for k, v in states.items()}
        o2, _, sh2 = sparse(pj, M, part, mg.CONP)
        torch.cuda.synchronize()
        small = dense_from_sparse(host(o2, sh2), ptr, idx, 0, M.nvar)
        assert not jac_ok_dense(dense_from_sparse(big[sl], ptr, idx, 0, M.nvar), small).any(), a


def test_scheduler_words_survive_more_launches_than_the_ring(env):
    pj, m, M = env
    states = mg.config_states(2, 5000)
    first, keep, shape = sparse(pj, M, states, mg.CONV)
    torch.cuda.synchronize()
    ref = host(first, shape)
    for it in range(70):                      # the handle has 64 scheduler slots
        out, keep2, _ = sparse(pj, M, states, mg.CONV)
        if it % 23 == 0 or it == 69:
            torch.cuda.synchronize()
            assert same(M, host(out, shape), ref), it
    torch.cuda.synchronize()


def test_two_streams_one_handle(env):
    pj, m, M = env
    sa, sb = mg.config_states(2, 6000), mg.config_states(2, 4000, start=6000)
    ra, _, sha = sparse(pj, M, sa, mg.CONP); rb, _, shb = sparse(pj, M, sb, mg.CONP)
    torch.cuda.synchronize()
    ref_a, ref_b = host(ra, sha), host(rb, shb)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs = []
    for _ in range(6):
        with torch.cuda.stream(s1):
            outs.append((sparse(pj, M, sa, mg.CONP, s1), ref_a))
        with torch.cuda.stream(s2):
            outs.append((sparse(pj, M, sb, mg.CONP, s2), ref_b))
    torch.cuda.synchronize()
    for (out, _, shape), ref in outs:
        assert same(M, host(out, shape), ref)


def test_fewer_tiles_than_ctas(env):
    pj, m, M = env
    from oracle import Oracle
    states = mg.config_states(2, 3)
    out, _, shape = sparse(pj, M, states, mg.CONP)
    torch.cuda.synchronize()
    ptr, idx = M.sparsity(mg.CSR)
    got = dense_from_sparse(host(out, shape), ptr, idx, 0, M.nvar)
    O = Oracle(m)
    assert not jac_ok_dense(got, O.jacobian_dense(mg.CONP, *O.pack(states, mg.CONP))).any()
