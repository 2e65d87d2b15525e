"""ctypes binding of oracle/forcefield.c -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

O2 (neighbours under PBC) and O3 (Eq. 4, 5, 8).  Argument marshalling only.
"""
import ctypes

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = ctypes.CDLL(path)
        c_int, c_dbl = ctypes.c_int, ctypes.c_double
        dp = ctypes.POINTER(c_dbl)
        ip = ctypes.POINTER(c_int)
        for name in ("oracle_neighbors_brute", "oracle_neighbors_cells"):
            fn = getattr(_lib, name)
            fn.restype = c_int
            fn.argtypes = [c_int, dp, dp, dp, c_dbl, c_int, ip, ip, ip]
        _lib.oracle_energy_force_virial.restype = c_int
        _lib.oracle_energy_force_virial.argtypes = [c_int, dp, dp, dp, c_int, dp, c_int, ip, ip, ip, dp, dp, dp, dp, dp]
        _lib.oracle_eval_images.restype = c_int
        _lib.oracle_eval_images.argtypes = [c_int, c_int, dp, dp, dp, c_int, dp, c_dbl, c_int, c_int, dp, dp, dp]
        _lib.oracle_set_types.restype = None
        _lib.oracle_set_types.argtypes = [ip, c_int]
        _lib.oracle_max_threads.restype = c_int
        _lib.oracle_set_threads.restype = None
        _lib.oracle_set_threads.argtypes = [c_int]
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _i(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__("oracle error %d" % code)
        self.code = code


def set_types(types):
    """Atom types (0 / 1) of the NEP-shaped potential (kind 4) for all later evaluations; None = all 0."""
    if types is None:
        lib().oracle_set_types(None, 0)
        return
    t = np.ascontiguousarray(types, dtype=np.int32)
    lib().oracle_set_types(_i(t), int(t.size))


def max_threads():
    return int(lib().oracle_max_threads())


def neighbors(Rt, h0, h, r_list, cap, brute=False):
    """Neighbour list of one image: count[N], list[N,cap], shift[N,cap,3] (int32).

    Entry (i; j, n) iff |(s_j - s_i + n) h| < r_list strictly, (j, n) != (i, 0); s = Rt h0^-1 unwrapped.
    """
    Rt, pR = _d(Rt)
    h0, ph0 = _d(h0)
    h, ph = _d(h)
    N = Rt.shape[0]
    count = np.zeros(N, dtype=np.int32)
    lst = np.full((N, cap), -1, dtype=np.int32)
    shift = np.zeros((N, cap, 3), dtype=np.int32)
    fn = lib().oracle_neighbors_brute if brute else lib().oracle_neighbors_cells
    rc = fn(N, pR, ph0, ph, float(r_list), int(cap), _i(count), _i(lst), _i(shift))
    if rc:
        raise OracleError(rc)
    return count, lst, shift


def energy_force_virial(Rt, h0, h, kind, pot, nbr, per_atom=False):
    """E, F[N,3], V[3,3] (and U_i[N], rho[N] if per_atom) of one image from its neighbour list."""
    Rt, pR = _d(Rt)
    h0, ph0 = _d(h0)
    h, ph = _d(h)
    pot, pp = _d(pot)
    count, lst, shift = nbr
    N = Rt.shape[0]
    cap = lst.shape[1]
    E = ctypes.c_double(0.0)
    F = np.zeros((N, 3))
    V = np.zeros((3, 3))
    Ui = np.zeros(N)
    rho = np.zeros(N)
    dp = ctypes.POINTER(ctypes.c_double)
    rc = lib().oracle_energy_force_virial(
        N, pR, ph0, ph, int(kind), pp, cap, _i(count), _i(lst), _i(shift), ctypes.byref(E),
        F.ctypes.data_as(dp), V.ctypes.data_as(dp), Ui.ctypes.data_as(dp), rho.ctypes.data_as(dp))
    if rc:
        raise OracleError(rc)
    if per_atom:
        return E.value, F, V, Ui, rho
    return E.value, F, V


def eval_images(Rt, h0, h, kind, pot, r_list, cap, brute=False, threads=None):
    """Batch: Rt[P,N,3], h[P,3,3] -> E[P], F[P,N,3], V[P,3,3] (own neighbour search per image)."""
    Rt, pR = _d(Rt)
    h0, ph0 = _d(h0)
    h, ph = _d(h)
    pot, pp = _d(pot)
    P, N = Rt.shape[0], Rt.shape[1]
    E = np.zeros(P)
    F = np.zeros((P, N, 3))
    V = np.zeros((P, 3, 3))
    dp = ctypes.POINTER(ctypes.c_double)
    if threads is not None:
        lib().oracle_set_threads(int(threads))
    rc = lib().oracle_eval_images(P, N, pR, ph0, ph, int(kind), pp, float(r_list), int(cap), int(bool(brute)),
                                  E.ctypes.data_as(dp), F.ctypes.data_as(dp), V.ctypes.data_as(dp))
    if rc:
        raise OracleError(rc)
    return E, F, V
