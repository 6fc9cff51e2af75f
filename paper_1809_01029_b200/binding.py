"""Thin ctypes binding of include/pyjac.h: argument marshalling only, same names as the C ABI.

Every step of the path runs in the CUDA kernels of libpyjac_b200.so; there is no Python or CPU
fallback: a missing library raises, a missing GPU makes `pyjac_mech_create` fail with PYJAC_ECUDA.
Device buffers are passed as integer addresses (`tensor.data_ptr()`), streams as
`torch.cuda.current_stream().cuda_stream` (or 0).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

PYJAC_OK, PYJAC_EINVAL, PYJAC_EMECH, PYJAC_ECUDA, PYJAC_ENOMEM = range(5)
PYJAC_CONP, PYJAC_CONV = 0, 1
PYJAC_CSR, PYJAC_CSC = 0, 1
PYJAC_APPROX_JACOBIAN = 1
PYJAC_PAIR_KERNEL = 2
WHAT_SOURCE, WHAT_SPARSE, WHAT_DENSE = 0, 1, 2

_D = C.POINTER(C.c_double)
_I = C.POINTER(C.c_int32)
_U = C.POINTER(C.c_uint8)
_FIELDS = [
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


class pyjac_mech_desc(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_reactions", C.c_int32)] + _FIELDS


class PyjacError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("pyjac error %d: %s" % (code, msg))
        self.code = code


LIB_PATH = os.environ.get("PYJAC_LIB") or os.path.join(os.path.dirname(os.path.abspath(__file__)), "libpyjac_b200.so")
_lib = None


def lib():
    """Loads libpyjac_b200.so (building it first if the sources are newer and nvcc is present)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            from . import build as _b
            _b.build()
        L = C.CDLL(LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int, C.c_int64
        L.pyjac_last_error.restype = C.c_char_p
        L.pyjac_mech_create.argtypes = [C.POINTER(pyjac_mech_desc), i32, C.POINTER(vp)]
        L.pyjac_mech_create_ex.argtypes = [C.POINTER(pyjac_mech_desc), i32, C.c_uint32, C.POINTER(vp)]
        L.pyjac_mech_destroy.argtypes = [vp]
        L.pyjac_mech_destroy.restype = None
        L.pyjac_mech_dims.argtypes = [vp, _I, _I, _I, C.POINTER(i64)]
        L.pyjac_sparsity.argtypes = [vp, i32, C.POINTER(_I), C.POINTER(_I)]
        L.pyjac_source_terms.argtypes = [vp, i32, i64, i64, i64, vp, vp, vp, vp]
        L.pyjac_jacobian_sparse.argtypes = [vp, i32, i32, i64, i64, i64, vp, vp, vp, vp]
        L.pyjac_jacobian_sparse_static.argtypes = [vp, i32, i32, i64, i64, i64, vp, vp, vp, vp]
        L.pyjac_jacobian_dense.argtypes = [vp, i32, C.c_char, i64, i64, i64, vp, vp, vp, vp]
        L.pyjac_state_from_fractions.argtypes = [vp, i32, i32, i64, i64, i64, vp, vp, vp, vp, vp, vp, vp]
        L.pyjac_fractions_from_state.argtypes = [vp, i32, i32, i64, i64, i64, vp, vp, vp, vp]
        L.pyjac_jacobian_fd.argtypes = [vp, i32, i32, C.c_double, C.c_double, i64, i64, i64, vp, vp, vp, vp]
        L.pyjac_eval_host.argtypes = [vp, i32, i32, i32, i64, i64, i64, vp, vp, vp]
        L.pyjac_launch_info.argtypes = [vp, i32, i64, i64, _I, _I, C.POINTER(i64)]
        L.pyjac_measure_peak.argtypes = [i32, i32, i32, _D]
        L.pyjac_plan_info.argtypes = [vp, C.POINTER(i64)]
        _lib = L
    return _lib


def _check(rc):
    if rc != PYJAC_OK:
        raise PyjacError(rc, lib().pyjac_last_error().decode())


def make_desc(mech):
    """pyjac_mech_desc from a dict of numpy arrays; returns (desc, keepalive list)."""
    d = pyjac_mech_desc()
    keep = []
    d.n_species = int(mech["n_species"]); d.n_reactions = int(mech["n_reactions"])
    for name, ct in _FIELDS:
        if name in ("chem_activated", "rev_A", "rev_beta", "rev_Ta") and name not in mech:
            continue                                     # optional fields: NULL = none
        a = np.ascontiguousarray(mech[name], dtype=_NP[ct])
        if a.size == 0:
            a = np.zeros(1, dtype=_NP[ct])
        keep.append(a)
        setattr(d, name, a.ctypes.data_as(ct))
    return d, keep


def pyjac_mech_create(mech, cuda_device=0):
    d, keep = make_desc(mech)
    h = C.c_void_p()
    _check(lib().pyjac_mech_create(C.byref(d), int(cuda_device), C.byref(h)))
    return h


def pyjac_mech_create_ex(mech, cuda_device=0, flags=0):
    d, keep = make_desc(mech)
    h = C.c_void_p()
    _check(lib().pyjac_mech_create_ex(C.byref(d), int(cuda_device), int(flags), C.byref(h)))
    return h


def pyjac_mech_destroy(h):
    lib().pyjac_mech_destroy(h)


def pyjac_mech_dims(h):
    ns, nr, nvar, nnz = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int64()
    _check(lib().pyjac_mech_dims(h, C.byref(ns), C.byref(nr), C.byref(nvar), C.byref(nnz)))
    return ns.value, nr.value, nvar.value, nnz.value


def pyjac_sparsity(h, fmt):
    _, _, nvar, nnz = pyjac_mech_dims(h)
    ptr, idx = _I(), _I()
    _check(lib().pyjac_sparsity(h, int(fmt), C.byref(ptr), C.byref(idx)))
    return (np.ctypeslib.as_array(ptr, shape=(nvar + 1,)).copy(), np.ctypeslib.as_array(idx, shape=(nnz,)).copy())


def pyjac_source_terms(h, mode, n_states, ld, tile, d_phi, d_param, d_dphi, stream=0):
    _check(lib().pyjac_source_terms(h, mode, n_states, ld, tile, d_phi, d_param, d_dphi, stream))


def pyjac_jacobian_sparse(h, mode, fmt, n_states, ld, tile, d_phi, d_param, d_vals, stream=0):
    _check(lib().pyjac_jacobian_sparse(h, mode, fmt, n_states, ld, tile, d_phi, d_param, d_vals, stream))


PYJAC_STATIC_MAX_STATES = 1 << 22


def pyjac_jacobian_sparse_static(h, mode, fmt, n_states, ld, tile, d_phi, d_param, d_vals, stream=0):
    """pyjac_jacobian_sparse with the kernel's scratch in a static device array: allocates nothing (include/pyjac.h)."""
    _check(lib().pyjac_jacobian_sparse_static(h, mode, fmt, n_states, ld, tile, d_phi, d_param, d_vals, stream))


def pyjac_jacobian_dense(h, mode, order, n_states, ld, tile, d_phi, d_param, d_J, stream=0):
    _check(lib().pyjac_jacobian_dense(h, mode, order.encode() if isinstance(order, str) else order, n_states, ld, tile,
                                      d_phi, d_param, d_J, stream))


PYJAC_MOLE_FRACTION, PYJAC_MASS_FRACTION = 0, 1


def pyjac_state_from_fractions(h, mode, kind, n_states, ld, tile, d_T, d_P, d_V, d_frac, d_phi, d_param, stream=0):
    _check(lib().pyjac_state_from_fractions(h, mode, kind, n_states, ld, tile, d_T, d_P, d_V, d_frac, d_phi, d_param, stream))


def pyjac_fractions_from_state(h, mode, kind, n_states, ld, tile, d_phi, d_param, d_frac, stream=0):
    _check(lib().pyjac_fractions_from_state(h, mode, kind, n_states, ld, tile, d_phi, d_param, d_frac, stream))


def pyjac_jacobian_fd(h, mode, fmt, rel_step, abs_step, n_states, ld, tile, d_phi, d_param, d_out, stream=0):
    """fmt: CSR / CSC (the handle's pattern) or 'C' / 'F' (dense)."""
    _check(lib().pyjac_jacobian_fd(h, mode, ord(fmt) if isinstance(fmt, str) else fmt, rel_step, abs_step, n_states, ld,
                                   tile, d_phi, d_param, d_out, stream))


def pyjac_eval_host(h, what, mode, fmt, n_states, ld, tile, h_phi, h_param, h_out):
    """Host numpy buffers in / out (copies inside the call)."""
    if isinstance(fmt, str):
        fmt = ord(fmt)
    for a in (h_phi, h_param, h_out):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    _check(lib().pyjac_eval_host(h, what, mode, fmt, n_states, ld, tile, h_phi.ctypes.data, h_param.ctypes.data,
                                 h_out.ctypes.data))


def pyjac_launch_info(h, what, n_states=0, tile=0):
    """(states per CTA, threads, shared-memory bytes) the library uses for a call with these n_states and tile."""
    S, nt, sm = C.c_int32(), C.c_int32(), C.c_int64()
    _check(lib().pyjac_launch_info(h, what, int(n_states), int(tile), C.byref(S), C.byref(nt), C.byref(sm)))
    return S.value, nt.value, sm.value


def pyjac_plan_info(h):
    """dict with the shape of the Jacobian kernel's gather plan (reporting only)."""
    a = (C.c_int64 * 8)()
    _check(lib().pyjac_plan_info(h, a))
    return dict(zip(("blocks", "slots_per_block", "partial_slots", "entries", "stored_entries", "groups", "piece_slots",
                     "split_lists"), [int(x) for x in a]))


PEAK_DFMA, PEAK_HBM_WRITE, PEAK_HBM_READ, PEAK_HBM_COPY, PEAK_L2_READ, PEAK_LDS = range(6)


def pyjac_measure_peak(kind, cuda_device=0, reps=5):
    """DFMA/s (PEAK_DFMA) or bytes/s of the machine, measured with the library's own microbenchmarks."""
    v = C.c_double()
    _check(lib().pyjac_measure_peak(int(kind), int(cuda_device), int(reps), C.byref(v)))
    return v.value


class Mechanism:
    """RAII convenience around the handle; methods forward to the C ABI."""

    def __init__(self, mech, cuda_device=0, flags=0):
        self.h = pyjac_mech_create_ex(mech, cuda_device, flags) if flags else pyjac_mech_create(mech, cuda_device)
        self.ns, self.nr, self.nvar, self.nnz = pyjac_mech_dims(self.h)

    def close(self):
        if getattr(self, "h", None) is not None:
            pyjac_mech_destroy(self.h); self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sparsity(self, fmt):
        return pyjac_sparsity(self.h, fmt)

    def n_elements(self, what):
        return {WHAT_SOURCE: self.nvar, WHAT_SPARSE: self.nnz, WHAT_DENSE: self.nvar * self.nvar}[what]
