"""ctypes binding of the oracle library (test infrastructure; see pyjac_oracle.cpp).

State-major numpy arrays in, numpy arrays out.  `Oracle(mech)` takes the desc-array dict produced by
`mechgen` (the only module shared with the CUDA product).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_D = C.POINTER(C.c_double)
_I = C.POINTER(C.c_int32)
_U = C.POINTER(C.c_uint8)

DESC_FIELDS = [
    ("mol_weight", _D), ("nasa_tmid", _D), ("nasa_lo", _D), ("nasa_hi", _D),
    ("reac_ptr", _I), ("reac_species", _I), ("reac_nu", _I), ("prod_ptr", _I), ("prod_species", _I), ("prod_nu", _I),
    ("reversible", _U), ("type", _I), ("A", _D), ("beta", _D), ("Ta", _D),
    ("eff_ptr", _I), ("eff_species", _I), ("eff_value", _D), ("collider", _I),
    ("low_A", _D), ("low_beta", _D), ("low_Ta", _D), ("troe", _D), ("troe_has_T2", _U), ("sri", _D),
    ("plog_ptr", _I), ("plog_P", _D), ("plog_A", _D), ("plog_beta", _D), ("plog_Ta", _D),
    ("cheb_ptr", _I), ("cheb_nT", _I), ("cheb_nP", _I),
    ("cheb_Tmin", _D), ("cheb_Tmax", _D), ("cheb_Pmin", _D), ("cheb_Pmax", _D), ("cheb_coef", _D),
    ("chem_activated", _U), ("rev_A", _D), ("rev_beta", _D), ("rev_Ta", _D),
]
_NP = {_D: np.float64, _I: np.int32, _U: np.uint8}


class _Desc(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_reactions", C.c_int32)] + DESC_FIELDS


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        lib.orc_create.restype = C.c_void_p
        lib.orc_create.argtypes = [C.POINTER(_Desc)]
        lib.orc_create2.restype = C.c_void_p
        lib.orc_create2.argtypes = [C.POINTER(_Desc), C.c_int]
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_nnz.restype = C.c_int64
        lib.orc_nnz.argtypes = [C.c_void_p]
        lib.orc_pattern.argtypes = [C.c_void_p, C.c_int, _I, _I]
        lib.orc_max_threads.restype = C.c_int
        lib.orc_source.argtypes = [C.c_void_p, C.c_int, C.c_int64, _D, _D, _D]
        lib.orc_jacobian_dense.argtypes = [C.c_void_p, C.c_int, C.c_int64, _D, _D, _D]
        lib.orc_jacobian_sparse.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int64, _D, _D, _D]
        lib.orc_intermediates.argtypes = [C.c_void_p, C.c_int, _D, C.c_double] + [_D] * 17
        lib.orc_fd_jacobian.argtypes = [C.c_void_p, C.c_int, _D, C.c_double, C.c_double, _D, _D]
        lib.orc_cs_jacobian.argtypes = [C.c_void_p, C.c_int, _D, C.c_double, C.c_double, _D, _D]
        lib.orc_state_from_fractions.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int64, _D, _D, _D, _D, _D, _D]
        lib.orc_fractions_from_state.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int64, _D, _D, _D]
        lib.orc_fd1_jacobian.argtypes = [C.c_void_p, C.c_int, C.c_int64, _D, _D, C.c_double, C.c_double, _D]
        _lib = lib
    return _lib


def _p(a, t=_D):
    return a.ctypes.data_as(t)


class Oracle:
    def __init__(self, mech, approx=False):
        """approx=True: the paper's "approximate" Jacobian and its sparser pattern."""
        lib = _load()
        self._keep = []
        d = _Desc()
        d.n_species = int(mech["n_species"]); d.n_reactions = int(mech["n_reactions"])
        for name, ct in DESC_FIELDS:
            a = np.ascontiguousarray(mech[name], dtype=_NP[ct])
            if a.size == 0:
                a = np.zeros(1, dtype=_NP[ct])
            self._keep.append(a)
            setattr(d, name, _p(a, ct))
        self.ns = d.n_species; self.nr = d.n_reactions; self.nvar = self.ns + 1
        self._h = C.c_void_p(lib.orc_create2(C.byref(d), 1 if approx else 0))
        self.nnz = int(lib.orc_nnz(self._h))
        self.threads = int(lib.orc_max_threads())

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.orc_destroy(self._h); self._h = None

    # ---- helpers -----------------------------------------------------------------------------
    @staticmethod
    def pack(states, mode):
        """(phi [n][nvar], param [n]) state-major from a mechgen states dict."""
        T, P, V, n = states["T"], states["P"], states["V"], states["n"]
        phi = np.empty((T.shape[0], n.shape[0] + 2))
        phi[:, 0] = T; phi[:, 1] = V if mode == 0 else P; phi[:, 2:] = n.T
        return np.ascontiguousarray(phi), np.ascontiguousarray(P if mode == 0 else V)

    def pattern(self, fmt):
        ptr = np.empty(self.nvar + 1, np.int32); idx = np.empty(self.nnz, np.int32)
        _lib.orc_pattern(self._h, fmt, _p(ptr, _I), _p(idx, _I))
        return ptr, idx

    def source(self, mode, phi, param):
        phi = np.ascontiguousarray(phi, np.float64).reshape(-1, self.nvar)
        param = np.ascontiguousarray(param, np.float64).reshape(-1)
        f = np.empty_like(phi)
        _lib.orc_source(self._h, mode, phi.shape[0], _p(phi), _p(param), _p(f))
        return f

    def jacobian_dense(self, mode, phi, param):
        phi = np.ascontiguousarray(phi, np.float64).reshape(-1, self.nvar)
        param = np.ascontiguousarray(param, np.float64).reshape(-1)
        J = np.empty((phi.shape[0], self.nvar, self.nvar))
        _lib.orc_jacobian_dense(self._h, mode, phi.shape[0], _p(phi), _p(param), _p(J))
        return J

    def jacobian_sparse(self, mode, fmt, phi, param):
        phi = np.ascontiguousarray(phi, np.float64).reshape(-1, self.nvar)
        param = np.ascontiguousarray(param, np.float64).reshape(-1)
        v = np.empty((phi.shape[0], self.nnz))
        _lib.orc_jacobian_sparse(self._h, mode, fmt, phi.shape[0], _p(phi), _p(param), _p(v))
        return v

    def state_from_fractions(self, mode, kind, T, P, V, frac):
        """kind 0: mole fractions, 1: mass fractions; frac [n][ns] -> (phi [n][nvar], param [n])."""
        T, P, V = (np.ascontiguousarray(a, np.float64).reshape(-1) for a in (T, P, V))
        frac = np.ascontiguousarray(frac, np.float64).reshape(-1, self.ns)
        phi = np.empty((T.shape[0], self.nvar)); param = np.empty(T.shape[0])
        _lib.orc_state_from_fractions(self._h, mode, kind, T.shape[0], _p(T), _p(P), _p(V), _p(frac), _p(phi), _p(param))
        return phi, param

    def fractions_from_state(self, mode, kind, phi, param):
        phi = np.ascontiguousarray(phi, np.float64).reshape(-1, self.nvar)
        param = np.ascontiguousarray(param, np.float64).reshape(-1)
        frac = np.empty((phi.shape[0], self.ns))
        _lib.orc_fractions_from_state(self._h, mode, kind, phi.shape[0], _p(phi), _p(param), _p(frac))
        return frac

    def intermediates(self, mode, phi, param):
        phi = np.ascontiguousarray(phi, np.float64).reshape(self.nvar)
        names_s = ["C", "cp", "h", "s", "g"]
        names_r = ["kf", "kr", "Kc", "M", "Pr", "F", "c", "Rf", "Rr", "q"]
        out = {k: np.empty(self.ns) for k in names_s}
        out.update({k: np.empty(self.nr) for k in names_r})
        out["wdot"] = np.empty(self.ns); scal = np.empty(4)
        args = [_p(out[k]) for k in names_s + names_r] + [_p(out["wdot"]), _p(scal)]
        _lib.orc_intermediates(self._h, mode, _p(phi), float(param), *args)
        out.update(Ctot=scal[0], D=scal[1], N=scal[2], S=scal[3])
        return out

    def _floor(self, phi, floor):
        if floor is None:
            ntot = np.abs(phi[2:]).sum()
            floor = np.concatenate([[1.0, 1e-30], np.full(self.nvar - 2, 1e-3 * ntot)])
        return np.ascontiguousarray(floor, np.float64)

    def fd1_jacobian(self, mode, phi, param, rel_step, abs_step):
        """First-order forward finite-difference Jacobian (step rule DESIGN.md R7), dense [n, nvar, nvar]."""
        phi = np.ascontiguousarray(phi, np.float64).reshape(-1, self.nvar)
        param = np.ascontiguousarray(param, np.float64).reshape(-1)
        J = np.empty((phi.shape[0], self.nvar, self.nvar))
        _lib.orc_fd1_jacobian(self._h, mode, phi.shape[0], _p(phi), _p(param), float(rel_step), float(abs_step), _p(J))
        return J

    def fd_jacobian(self, mode, phi, param, rel=1e-4, floor=None):
        phi = np.ascontiguousarray(phi, np.float64).reshape(self.nvar)
        J = np.empty((self.nvar, self.nvar)); fl = self._floor(phi, floor)
        _lib.orc_fd_jacobian(self._h, mode, _p(phi), float(param), rel, _p(fl), _p(J))
        return J

    def cs_jacobian(self, mode, phi, param, rel=1e-30, floor=None):
        phi = np.ascontiguousarray(phi, np.float64).reshape(self.nvar)
        J = np.empty((self.nvar, self.nvar)); fl = self._floor(phi, floor)
        _lib.orc_cs_jacobian(self._h, mode, _p(phi), float(param), rel, _p(fl), _p(J))
        return J
