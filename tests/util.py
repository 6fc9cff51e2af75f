"""Helpers shared by the tests: layout packing and the parity tolerances of BASELINE.json."""
import numpy as np


def unpack(flat, n_e, n_states, ld, tile):
    """Library layout (include/pyjac.h) -> [n_states, n_e]."""
    a = np.asarray(flat).reshape(ld // tile, n_e, tile).transpose(0, 2, 1).reshape(ld, n_e)
    return a[:n_states]


def source_ok(got, ref):
    """max |d| <= 1e-10 (|ref| + 1e-20)  (BASELINE.json north_star)."""
    err = np.abs(got - ref) / (1e-10 * (np.abs(ref) + 1e-20))
    return err.max() if err.size else 0.0


def jac_ok_dense(got, ref):
    """<= 1e-8 relative with a 1e-12 max|row| absolute floor; got/ref [..., nvar, nvar]."""
    rowmax = np.abs(ref).max(axis=-1, keepdims=True)
    tol = np.maximum(1e-8 * np.abs(ref), 1e-12 * rowmax)
    bad = np.abs(got - ref) > tol
    bad |= ~np.isfinite(got)
    return bad


def dense_from_sparse(vals, ptr, idx, fmt, nvar):
    """[n, nnz] values in CSR (fmt 0) / CSC (fmt 1) order -> [n, nvar, nvar]."""
    n = vals.shape[0]
    J = np.zeros((n, nvar, nvar))
    major = np.repeat(np.arange(nvar), np.diff(ptr))
    if fmt == 0:
        J[:, major, idx] = vals
    else:
        J[:, idx, major] = vals
    return J


def net_stoichiometry(mech):
    """[n_species, n_reactions] net coefficients nu'' - nu' from the desc arrays (test helper, no rate law)."""
    ns, nr = int(mech["n_species"]), int(mech["n_reactions"])
    nu = np.zeros((ns, nr))
    for ptr, sp, co, sgn in ((mech["reac_ptr"], mech["reac_species"], mech["reac_nu"], -1.0),
                             (mech["prod_ptr"], mech["prod_species"], mech["prod_nu"], 1.0)):
        for i in range(nr):
            for j in range(ptr[i], ptr[i + 1]):
                nu[sp[j], i] += sgn * co[j]
    return nu


def source_violations(got, ref, oracle, mech, mode, phi, par):
    """Entries of dphi/dt outside the BASELINE tolerance 1e-10 (|ref| + 1e-20) AND outside the cancellation bound of
    DESIGN.md S12b.  Every source term is a sum over reactions of terms that cancel (3-9 digits are
    lost near partial equilibrium): dn_k/dt = V sum_i nu_ki q_i, N = sum_i dE~_i q_i (dT/dt = -N/D), S = sum_i dn~_i q_i.
    Two correct fp64 evaluations of q_i = c_i (R'_i - R''_i) differ by a few ulp each (exp, log, pow of different
    libraries), so 64 eps x (the same sum with |nu_ki| |c_i| (|R'_i| + |R''_i|) as terms) is the best any implementation
    can promise.  Returns (violations, n_entries_that_needed_the_bound)."""
    R = 8314.46261815324
    err = np.abs(got - ref) / (1e-10 * (np.abs(ref) + 1e-20))
    bad = np.argwhere(err > 1.0)
    nu = None
    out, needed = [], 0
    eps64 = 64 * np.finfo(float).eps
    for s, e in bad:
        if nu is None:
            nu = net_stoichiometry(mech)
            W = np.asarray(mech["mol_weight"], float); L = len(W) - 1
        it = oracle.intermediates(mode, phi[s], par[s])
        T = phi[s, 0]
        V, P = (phi[s, 1], par[s]) if mode == 0 else (par[s], phi[s, 1])
        aq = np.abs(it["c"]) * (np.abs(it["Rf"]) + np.abs(it["Rr"]))          # |q_i| without the cancellation
        if e >= 2:
            mag = V * np.sum(np.abs(nu[e - 2]) * aq)
        else:
            E = it["h"] if mode == 0 else it["h"] - R * T                      # H_k (CONP) or U_k (CONV), per kmol
            Et = E[:L] - W[:L] / W[L] * E[L]
            # dE~_i = sum_k nu_ki E~_k itself cancels for nearly thermoneutral reactions: terms taken by magnitude
            magT = np.sum((np.abs(Et) @ np.abs(nu[:L])) * aq) / it["D"]
            magS = np.sum((np.abs(1.0 - W[:L] / W[L]) @ np.abs(nu[:L])) * aq)
            mag = magT if e == 0 else (V * (T * R / P * magS + magT / T) if mode == 0 else T * R * magS + P / T * magT)
        if abs(got[s, e] - ref[s, e]) <= eps64 * mag:
            needed += 1
        else:
            out.append((int(s), int(e), float(err[s, e]), float(mag / max(abs(ref[s, e]), 1e-300))))
    return out, needed
