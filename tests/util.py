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
