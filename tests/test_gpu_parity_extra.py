"""More parity cases of the CUDA path against the oracle ("close the parity holes"): every
states-per-CTA instantiation of the tile kernel, the method's edge cases on the GPU, the BASELINE sizes of C2 and C3,
the pair kernel on every mechanism, and launches of one handle on two streams."""
import numpy as np
import pytest

import mechgen as mg
from mechgen.mechanism import CONFIGS, pack_phi
from tests.util import unpack, source_ok, source_violations, jac_ok_dense, dense_from_sparse
from tests.test_gpu_parity import setup, run_gpu, pj  # noqa: F401  (pj is the module fixture)

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

N_SM2 = 2 * 148      # the library keeps S states per CTA only while there are two tiles per SM


def _sub(states, pick):
    return {k: (v[pick] if v.ndim == 1 else v[:, pick]) for k, v in states.items()}


# ---- every instantiation jacobian_kernel<S> / source_kernel<S>: S = min(tile, largest that fits), given enough tiles --
@pytest.mark.parametrize("name,S", [("c1", 32), ("c1", 16), ("c2", 8), ("c3", 4), ("c3", 2), ("c2", 1)])
def test_every_states_per_cta(pj, name, S):
    m, M, o, st = setup(pj, name)
    smax, _, _ = pj.pyjac_launch_info(M.h, pj.WHAT_SPARSE)
    assert smax >= S, "mechanism does not fit %d states per CTA" % S
    n = N_SM2 * S + 2 * S + max(1, S // 2)            # >= 296 tiles and a ragged last tile
    ld = (n + S - 1) // S * S
    states = st(n)
    rng = np.random.default_rng(S)
    pick = np.unique(np.concatenate([[0, n - 1, n - 2], rng.integers(0, n, 40)]))
    sub = _sub(states, pick)
    for mode in (mg.CONP, mg.CONV):
        Jr = o.jacobian_dense(mode, *o.pack(sub, mode))
        fr = o.source(mode, *o.pack(sub, mode))
        got = run_gpu(pj, M, pj.WHAT_SOURCE, mode, 0, states, ld, S)
        assert source_ok(got[pick], fr) <= 10.0
        # all states, with the cancellation bound where the plain tolerance is not reachable (S12b)
        phi_o, par_o = o.pack(states, mode)
        viol, needed = source_violations(got, o.source(mode, phi_o, par_o), o, m, mode, phi_o, par_o)
        assert not viol and needed <= 3, (viol[:5], needed)
        for fmt in (mg.CSR, mg.CSC):
            ptr, idx = M.sparsity(fmt)
            got = run_gpu(pj, M, pj.WHAT_SPARSE, mode, fmt, states, ld, S)
            assert np.isfinite(got).all()
            assert not jac_ok_dense(dense_from_sparse(got[pick], ptr, idx, fmt, M.nvar), Jr).any()
        got = run_gpu(pj, M, pj.WHAT_DENSE, mode, "C", states, ld, S).reshape(n, M.nvar, M.nvar)
        assert not jac_ok_dense(got[pick], Jr).any()


# ---- edge cases of the method on the GPU (the oracle is pinned on them on the CPU, tests/test_oracle_rate_laws.py) ----
def _edge_states():
    """hand_all_types states with: P below the first P-Log node, above the last, exactly on nodes; C_k = 0 exactly;
    T exactly T_mid (S3, S4, S7)."""
    st = mg.make_states(6, 16, 77)
    T, P, V, n = st["T"].copy(), st["P"].copy(), st["V"].copy(), st["n"].copy()      # n: [species, state]
    nodes = [10132.5, 101325.0, 1013250.0, 10132500.0]
    P[0] = 5000.0; P[1] = 2.0e7; P[2:6] = nodes; P[6] = np.nextafter(nodes[1], 0.0); P[7] = np.nextafter(nodes[1], 1e9)
    T[8] = 1000.0; T[9] = np.nextafter(1000.0, 2000.0); T[10] = 1000.0; P[10] = nodes[2]
    n[0, 11] = 0.0; n[1, 12] = 0.0; n[2, 12] = 0.0; n[:3, 13] = 0.0
    return {"T": T, "P": P, "V": V, "n": n}


@pytest.mark.parametrize("flags", [0, 2])
def test_method_edge_cases_on_gpu(pj, flags):
    from oracle import Oracle
    m = mg.hand_all_types(True, True)
    M = pj.Mechanism(m, 0, flags)
    o = Oracle(m)
    states = _edge_states()
    n = states["T"].shape[0]
    for mode in (mg.CONP, mg.CONV):
        phi, par = o.pack(states, mode)
        fr = o.source(mode, phi, par); Jr = o.jacobian_dense(mode, phi, par)
        assert np.isfinite(fr).all() and np.isfinite(Jr).all()
        got = run_gpu(pj, M, pj.WHAT_SOURCE, mode, 0, states)
        assert source_ok(got, fr) <= 1.0
        ptr, idx = M.sparsity(mg.CSR)
        got = run_gpu(pj, M, pj.WHAT_SPARSE, mode, mg.CSR, states, n, 2)
        bad = jac_ok_dense(dense_from_sparse(got, ptr, idx, mg.CSR, M.nvar), Jr)
        assert not bad.any(), np.argwhere(bad)[:8]
        got = run_gpu(pj, M, pj.WHAT_DENSE, mode, "F", states).reshape(n, M.nvar, M.nvar).transpose(0, 2, 1)
        assert not jac_ok_dense(got, Jr).any()


# ---- the pair kernel (PYJAC_PAIR_KERNEL) on every mechanism: LS = 1, 2, 4 state pairs per item, odd tiles, tails ----
_PAIR = {}


def _pair_setup(pj, name):
    if name not in _PAIR:
        m, _, o, st = setup(pj, name)
        _PAIR[name] = (pj.Mechanism(m, 0, pj.PYJAC_PAIR_KERNEL), o, st)
    return _PAIR[name]


@pytest.mark.parametrize("name,n,tile", [("four", 64, 64), ("all_types", 301, 1), ("chem", 200, 2), ("revx", 199, 200),
                                         ("c1", 2500, 4), ("c1", 1300, 8), ("c2", 1201, 2), ("c3", 150, 2), ("c5", 25, 1),
                                         ("c5", 24, 2), ("c4", 11, 11)])
def test_pair_kernel_parity(pj, name, n, tile):
    M, o, st = _pair_setup(pj, name)
    states = st(n)
    ld = (n + tile - 1) // tile * tile
    for mode in (mg.CONP, mg.CONV):
        Jr = o.jacobian_dense(mode, *o.pack(states, mode))
        for fmt in (mg.CSR, mg.CSC):
            ptr, idx = M.sparsity(fmt)
            got = run_gpu(pj, M, pj.WHAT_SPARSE, mode, fmt, states, ld, tile)
            bad = jac_ok_dense(dense_from_sparse(got, ptr, idx, fmt, M.nvar), Jr)
            assert not bad.any(), (np.argwhere(bad)[:5])
        got = run_gpu(pj, M, pj.WHAT_DENSE, mode, "C", states, ld, tile).reshape(n, M.nvar, M.nvar)
        assert not jac_ok_dense(got, Jr).any()
        ptr, idx = M.sparsity(mg.CSR)
        pat = dense_from_sparse(np.ones((1, M.nnz)), ptr, idx, mg.CSR, M.nvar)[0] != 0
        assert np.all(got[:, ~pat] == 0.0)


def test_pair_kernel_is_the_path_where_the_tile_kernel_does_not_fit(pj):
    """A mechanism whose per-reaction partials exceed one SM's shared memory (C5 with every reaction reversible and
    third-body-like would; here: C5's reactions doubled) is evaluated by the pair kernel without the flag."""
    m = dict(mg.config_mechanism(5))
    nr = int(m["n_reactions"])

    def twice(key):
        a = np.asarray(m[key])
        return np.concatenate([a, a])

    ragged = {"reac": ("reac_ptr", ["reac_species", "reac_nu"]), "prod": ("prod_ptr", ["prod_species", "prod_nu"]),
              "eff": ("eff_ptr", ["eff_species", "eff_value"]), "plog": ("plog_ptr", ["plog_P", "plog_A", "plog_beta", "plog_Ta"]), "cheb": ("cheb_ptr", ["cheb_coef"])}
    out = dict(m)
    for _, (pk, vals) in ragged.items():
        p = np.asarray(m[pk]); out[pk] = np.concatenate([p, p[1:] + p[-1]]).astype(np.int32)
        for v in vals:
            out[v] = twice(v)
    for k in ("reversible", "type", "A", "beta", "Ta", "collider", "low_A", "low_beta", "low_Ta", "troe", "troe_has_T2", "sri",
              "cheb_nT", "cheb_nP", "cheb_Tmin", "cheb_Tmax", "cheb_Pmin", "cheb_Pmax", "chem_activated", "rev_A", "rev_beta", "rev_Ta"):
        if k in m:
            out[k] = twice(k)
    out["A"] = out["A"].copy(); out["A"][nr:] *= 0.5                       # the copies are not exact duplicates
    out["n_reactions"] = 2 * nr
    from oracle import Oracle
    M = pj.Mechanism(out, 0)
    info = pj.pyjac_plan_info(M.h)
    assert info["blocks"] >= 2
    o = Oracle(out)
    states = mg.config_states(5, 12)
    for mode in (mg.CONP, mg.CONV):
        Jr = o.jacobian_dense(mode, *o.pack(states, mode))
        ptr, idx = M.sparsity(mg.CSR)
        got = run_gpu(pj, M, pj.WHAT_SPARSE, mode, mg.CSR, states, 12, 2)
        assert not jac_ok_dense(dense_from_sparse(got, ptr, idx, mg.CSR, M.nvar), Jr).any()


# ---- BASELINE sizes of C2 (CONP and CONV, CSR) and C3 (CSC and dense) in the launch configuration bench.py times ----
@pytest.mark.parametrize("c,mode,what,fmt", [(2, mg.CONP, "sparse", mg.CSR), (2, mg.CONV, "sparse", mg.CSR),
                                             (3, mg.CONP, "sparse", mg.CSC), (3, mg.CONP, "dense", "C")])
def test_full_size_c2_c3_sampled(pj, c, mode, what, fmt):
    m, M, o, st = setup(pj, "c%d" % c)
    N = CONFIGS[c]["n_states"]
    w = pj.WHAT_SPARSE if what == "sparse" else pj.WHAT_DENSE
    n_e = M.n_elements(w)
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
    if what == "sparse":
        pj.pyjac_jacobian_sparse(M.h, mode, fmt, N, N, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), stream)
    else:
        pj.pyjac_jacobian_dense(M.h, mode, fmt, N, N, tile, d_phi.data_ptr(), d_par.data_ptr(), out.data_ptr(), stream)
    torch.cuda.synchronize()
    view = out.view(N // tile, n_e, tile)
    assert bool(torch.isfinite(view.sum(dim=1)).all())
    rng = np.random.default_rng(100 + c)
    pick = np.unique(np.concatenate([[0, N - 1], rng.integers(0, N, 62)]))
    got = np.stack([view[s // tile, :, s % tile].cpu().numpy() for s in pick])
    sub = _sub(states, pick)
    Jr = o.jacobian_dense(mode, *o.pack(sub, mode))
    if what == "sparse":
        ptr, idx = M.sparsity(fmt)
        Jg = dense_from_sparse(got, ptr, idx, fmt, M.nvar)
    else:
        Jg = got.reshape(len(pick), M.nvar, M.nvar)
    bad = jac_ok_dense(Jg, Jr)
    assert not bad.any(), (np.argwhere(bad)[:5], Jg[bad][:5], Jr[bad][:5])
    del out
    torch.cuda.empty_cache()


# ---- launches of one handle on two streams: stream A is held back while stream B issues more launches than the ring of
# scheduler words has slots (two kernels in flight must never share a tile counter) ----
@pytest.mark.parametrize("flags", [0, 2])
def test_held_back_stream_and_ring_wraparound(pj, flags):
    m, _, o, st = setup(pj, "c2")
    M = pj.Mechanism(m, 0, flags)
    n = 3000
    states = st(n)
    phi, par = pack_phi(states, mg.CONP, n, n)
    d_phi = torch.from_numpy(phi).cuda(); d_par = torch.from_numpy(par).cuda()
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    outs_a = [torch.full((M.nnz * n,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3)]
    outs_b = [torch.full((M.nnz * n,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(70)]
    torch.cuda.synchronize()
    with torch.cuda.stream(sa):
        torch.cuda._sleep(400_000_000)                        # ~0.2 s: everything queued on A stays pending meanwhile
        for t in outs_a:
            pj.pyjac_jacobian_sparse(M.h, mg.CONP, mg.CSR, n, n, n, d_phi.data_ptr(), d_par.data_ptr(), t.data_ptr(), sa.cuda_stream)
    for t in outs_b:
        pj.pyjac_jacobian_sparse(M.h, mg.CONP, mg.CSR, n, n, n, d_phi.data_ptr(), d_par.data_ptr(), t.data_ptr(), sb.cuda_stream)
    torch.cuda.synchronize()
    ref = unpack(outs_b[0].cpu().numpy(), M.nnz, n, n, n)
    ptr, idx = M.sparsity(mg.CSR)
    pick = np.arange(0, n, 97)
    Jr = o.jacobian_dense(mg.CONP, *o.pack(_sub(states, pick), mg.CONP))
    assert not jac_ok_dense(dense_from_sparse(ref[pick], ptr, idx, mg.CSR, M.nvar), Jr).any()
    for t in outs_a + outs_b[1:]:
        got = unpack(t.cpu().numpy(), M.nnz, n, n, n)
        assert np.isfinite(got).all()                         # a skipped tile would leave NaN behind
        # launches differ in the last bits (dynamic chunk order); entries that cancel may differ by more
        assert np.all(np.abs(got - ref) <= 1e-9 * np.abs(ref) + 1e-13 * np.abs(ref).max(axis=1, keepdims=True))


# ---- several P-Log entries per pressure (R10): summed rates, both Jacobian kernels and the source kernel ----
@pytest.mark.parametrize("flags", [0, 2])
def test_plog_several_entries_per_pressure_on_gpu(pj, flags):
    from mechgen import MechBuilder
    from oracle import Oracle
    PATM = 101325.0
    cp = lambda a0, a5, a6: [a0, 0, 0, 0, 0, a5, a6]
    mb = MechBuilder()
    mb.add_species(30.0, cp(4.0, 1000.0, 5.0)); mb.add_species(10.0, cp(3.0, 9000.0, 4.0))
    mb.add_species(20.0, cp(3.5, 4000.0, 6.0)); mb.add_species(28.0, cp(3.5, -1000.0, 6.5))
    pts = [(1.0 * PATM, 1e10, 0.0, 5000.0), (1.0 * PATM, 3e7, 0.9, 2500.0), (10.0 * PATM, 1e12, 0.5, 8000.0),
           (10.0 * PATM, 5e9, 0.2, 3000.0), (10.0 * PATM, 2e11, -0.3, 6000.0), (50.0 * PATM, 4e12, 0.1, 9000.0)]
    mb.add_reaction({0: 1}, {1: 1, 2: 1}, 1.0, 0.0, 0.0, rev=True, type=mg.PLOG, plog=pts)
    mb.add_reaction({1: 1, 2: 1}, {0: 1}, 3e9, 0.4, 1500.0, rev=False)
    mb.add_reaction({0: 2}, {1: 2, 2: 2}, 1.0, 0.0, 0.0, rev=False, type=mg.PLOG, plog=pts[2:4] + pts[5:])
    m = mb.build()
    M = pj.Mechanism(m, 0, flags)
    o = Oracle(m)
    states = mg.make_states(4, 24, 91)
    P = states["P"]
    P[:8] = np.array([0.3, 1.0, 2.0, 10.0, 30.0, 50.0, 90.0, 9.999999]) * PATM
    for mode in (mg.CONP, mg.CONV):
        phi, par = o.pack(states, mode)
        fr = o.source(mode, phi, par); Jr = o.jacobian_dense(mode, phi, par)
        assert source_ok(run_gpu(pj, M, pj.WHAT_SOURCE, mode, 0, states), fr) <= 1.0
        ptr, idx = M.sparsity(mg.CSR)
        got = run_gpu(pj, M, pj.WHAT_SPARSE, mode, mg.CSR, states, 24, 2)
        bad = jac_ok_dense(dense_from_sparse(got, ptr, idx, mg.CSR, M.nvar), Jr)
        assert not bad.any(), np.argwhere(bad)[:8]


# ---- fraction <-> state conversion kernels against the oracle, every layout kind ----
@pytest.mark.parametrize("name,n,ld,tile", [("c1", 1000, 1024, 1024), ("c3", 333, 336, 8), ("c2", 77, 77, 1), ("c5", 200, 200, 200)])
def test_fraction_conversions(pj, name, n, ld, tile):
    m, M, o, st = setup(pj, name)
    states = st(n)
    ns = M.ns

    def to_dev(a, n_e):          # [n][n_e] -> library layout
        full = np.zeros((ld, n_e)); full[:n] = a
        return torch.from_numpy(np.ascontiguousarray(full.reshape(ld // tile, tile, n_e).transpose(0, 2, 1)).reshape(-1)).cuda()

    def vec(a):
        v = np.ones(ld); v[:n] = a
        return torch.from_numpy(v).cuda()

    s_ = torch.cuda.current_stream().cuda_stream
    for mode in (mg.CONP, mg.CONV):
        phi0, par0 = o.pack(states, mode)
        for kind in (pj.PYJAC_MOLE_FRACTION, pj.PYJAC_MASS_FRACTION):
            ref = o.fractions_from_state(mode, kind, phi0, par0)
            d_phi = to_dev(phi0, M.nvar); d_par = vec(par0)
            d_f = torch.full((ns * ld,), float("nan"), dtype=torch.float64, device="cuda")
            pj.pyjac_fractions_from_state(M.h, mode, kind, n, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), d_f.data_ptr(), s_)
            torch.cuda.synchronize()
            got = unpack(d_f.cpu().numpy(), ns, n, ld, tile)
            assert np.all(np.abs(got - ref) <= 1e-12 * np.abs(ref) + 1e-15)      # X_Ns = 1 - sum X_k: absolute floor
            # and back: state from the fractions
            pref, parref = o.state_from_fractions(mode, kind, states["T"], states["P"], states["V"], ref)
            d_T, d_P, d_V = vec(states["T"]), vec(states["P"]), vec(states["V"])
            d_out = torch.full((M.nvar * ld,), float("nan"), dtype=torch.float64, device="cuda")
            d_po = torch.full((ld,), float("nan"), dtype=torch.float64, device="cuda")
            pj.pyjac_state_from_fractions(M.h, mode, kind, n, ld, tile, d_T.data_ptr(), d_P.data_ptr(), d_V.data_ptr(),
                                          to_dev(ref, ns).data_ptr(), d_out.data_ptr(), d_po.data_ptr(), s_)
            torch.cuda.synchronize()
            got = unpack(d_out.cpu().numpy(), M.nvar, n, ld, tile)
            np.testing.assert_allclose(got, pref, rtol=1e-13, atol=0)
            assert d_po.cpu().numpy()[:n].tobytes() == parref.tobytes()
            if ld > n:
                assert np.isnan(d_po.cpu().numpy()[n:]).all()
    with pytest.raises(pj.PyjacError):
        pj.pyjac_fractions_from_state(M.h, 0, 5, n, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), d_f.data_ptr(), s_)


# ---- many inert species: more than 128 empty gather lists in the T/E-row and source-term plans (their
# outputs -- an explicit 0 for dn_k/dt, the f_T (c_j - c_Ns) term of J[T][j] -- must still be stored) ----
def test_many_inert_species(pj):
    from mechgen import MechBuilder
    from oracle import Oracle
    rng = np.random.default_rng(5)
    mb = MechBuilder()
    ns = 340
    for k in range(ns):
        mb.add_species(10.0 + 0.1 * k, [3.0 + 0.002 * k, 1e-4, 0, 0, 0, -500.0 * (k % 7), 4.0])
    mb.add_reaction({0: 1, 1: 1}, {2: 1, 3: 1}, 4e9, 0.3, 4000.0, rev=True)
    mb.add_reaction({2: 1}, {0: 1}, 2e7, 0.0, 3000.0, rev=False)
    mb.add_reaction({3: 1, 4: 1}, {1: 1, 5: 1}, 6e9, -0.2, 2500.0, rev=True, type=mg.THIRD_BODY, eff={7: 2.5, 200: 0.4})
    m = mb.build()
    M = pj.Mechanism(m, 0); o = Oracle(m)
    states = mg.make_states(ns, 40, 17)
    for mode in (mg.CONP, mg.CONV):
        phi, par = o.pack(states, mode)
        fr = o.source(mode, phi, par); Jr = o.jacobian_dense(mode, phi, par)
        got = run_gpu(pj, M, pj.WHAT_SOURCE, mode, 0, states)
        assert np.isfinite(got).all() and source_ok(got, fr) <= 1.0
        assert np.all(got[:, 2 + 10:] == 0.0)                        # inert species: an explicit zero
        ptr, idx = M.sparsity(mg.CSR)
        got = run_gpu(pj, M, pj.WHAT_SPARSE, mode, mg.CSR, states, 40, 1)
        assert np.isfinite(got).all()
        assert not jac_ok_dense(dense_from_sparse(got, ptr, idx, mg.CSR, M.nvar), Jr).any()


# ---- dense by expansion (one state per CTA, state-major layout, n_var^2 >= 32768): more states than SMs, so that a CTA
# works through several tiles (the expansion of tile k runs inside tile k + 1; both scratch buffers; the last tile's
# expansion after the loop), both orders, odd and even alignment of a state's matrix (n_var^2 is odd for C4) ----
@pytest.mark.parametrize("order", ["C", "F"])
@pytest.mark.parametrize("mode", [mg.CONP, mg.CONV])
def test_dense_by_expansion_many_tiles(pj, order, mode):
    m, M, o, st = setup(pj, "c4")
    n = 3 * 148 + 5
    states = st(n)
    fmt = mg.CSR if order == "C" else mg.CSC
    sparse = run_gpu(pj, M, pj.WHAT_SPARSE, mode, fmt, states, n, 1)          # (its own parity: test_jacobian_sparse)
    dense = run_gpu(pj, M, pj.WHAT_DENSE, mode, order, states, n, 1)
    assert np.isfinite(dense).all()
    ptr, idx = M.sparsity(fmt)
    # every state, every element: the nonzeros are the sparse path's values (same arithmetic; the sums of a tile depend
    # on which warp took which chunk, so two launches agree to rounding, not to the bit), everything else is an exact zero
    expect = dense_from_sparse(sparse, ptr, idx, fmt, M.nvar)                 # [n, row, col]
    got = dense.reshape(n, M.nvar, M.nvar)
    if order == "F":
        got = got.transpose(0, 2, 1)
    pat = dense_from_sparse(np.ones((1, M.nnz)), ptr, idx, fmt, M.nvar)[0] != 0
    assert np.all(got[:, ~pat] == 0.0)
    scale = np.abs(expect).reshape(n, -1).max(axis=1)[:, None, None]
    assert np.all(np.abs(got - expect) <= 1e-9 * np.abs(expect) + 1e-13 * scale)
    # and against the oracle on a sample that has neighbours of both alignments, the first and the last state
    pick = np.array([0, 1, 2, 147, 148, 149, 295, 296, 297, n - 2, n - 1])
    Jr = o.jacobian_dense(mode, *o.pack(_sub(states, pick), mode))
    bad = jac_ok_dense(got[pick], Jr)
    assert not bad.any(), (np.argwhere(bad)[:5], got[pick][bad][:5], Jr[bad][:5])


# two dense-by-expansion launches of one handle on two streams share the handle's scratch buffers: the library orders the
# second behind the first (an event), so both results are those of a launch alone
def test_dense_by_expansion_two_streams(pj):
    m, M, o, st = setup(pj, "c4")
    n = 200
    sa, sb = st(n), _sub(st(2 * n), np.arange(n, 2 * n))
    ref_a = run_gpu(pj, M, pj.WHAT_DENSE, mg.CONP, "C", sa, n, 1)
    ref_b = run_gpu(pj, M, pj.WHAT_DENSE, mg.CONP, "C", sb, n, 1)
    n_e = M.nvar * M.nvar
    bufs = []
    for s_ in (sa, sb):
        phi, par = pack_phi(s_, mg.CONP, n, 1)
        bufs.append((torch.from_numpy(phi).cuda(), torch.from_numpy(par).cuda(),
                     torch.full((n_e * n,), float("nan"), dtype=torch.float64, device="cuda")))
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for (phi, par, out), s_ in zip(bufs, (s1, s2)):
        pj.pyjac_jacobian_dense(M.h, mg.CONP, "C", n, n, 1, phi.data_ptr(), par.data_ptr(), out.data_ptr(), s_.cuda_stream)
    torch.cuda.synchronize()
    for (_, _, out), ref in zip(bufs, (ref_a, ref_b)):
        got = out.cpu().numpy().reshape(n, n_e)
        assert np.array_equal(got == 0.0, ref == 0.0)
        assert np.all(np.abs(got - ref) <= 1e-9 * np.abs(ref) + 1e-13 * np.abs(ref).max(axis=1, keepdims=True))
