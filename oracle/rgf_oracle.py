"""ctypes loader for the CPU oracle (oracle/rgf_oracle.c).  TEST INFRASTRUCTURE ONLY.

Argument marshalling only; every formula lives in rgf_oracle.c, each citing the passage of
PAPER.md / BASELINE.json it follows.  Function names mirror the C exports (orc_*).
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None

LEAD_CELL = 0    # Sancho-Rubio on the 2M x 2M two-slice cell (north_star's wording)
LEAD_BLOCK = 1   # same chain, non-surface slice eliminated first (M x M); pinned == LEAD_CELL


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__("oracle %s failed with code %d" % (what, code))
        self.code = code


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, ip, u8p = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_uint8)
        L.orc_num_threads.restype = C.c_int
        L.orc_inverse.argtypes = [C.c_int, dp, dp]
        L.orc_matmul.argtypes = [C.c_int, dp, dp, dp]
        L.orc_lead_surface.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, dp, ip]
        L.orc_lead_self_energy.argtypes = [C.c_int, C.c_int, u8p, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, dp, ip]
        L.orc_transmission.argtypes = [C.c_int, C.c_int, dp, u8p, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, dp, dp, ip]
        L.orc_sweep_state.argtypes = [C.c_int, C.c_int, dp, u8p, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, dp, dp]
        L.orc_transmission_batch.argtypes = [C.c_int, C.c_int, dp, u8p, C.c_double, dp, C.c_int, C.c_double, C.c_int, C.c_int, dp, ip]
        L.orc_transmission_eq4_batch.argtypes = [C.c_int, C.c_int, dp, u8p, C.c_double, dp, C.c_int, C.c_double, C.c_int, C.c_int, C.c_int, dp, ip]
        L.orc_ldos_batch.argtypes = [C.c_int, C.c_int, dp, u8p, C.c_double, dp, C.c_int, C.c_double, C.c_int, C.c_int, dp]
        L.orc_transmission_brute.argtypes = [C.c_int, C.c_int, dp, u8p, C.c_double, C.c_double, C.c_double, C.c_int, dp, dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _onsite(onsite, vacancy):
    onsite = np.ascontiguousarray(onsite, dtype=np.float64)
    assert onsite.ndim == 2
    L, M = onsite.shape
    if vacancy is None:
        vp = None
        vac = None
    else:
        vac = np.ascontiguousarray(vacancy, dtype=np.uint8)
        assert vac.shape == (L, M)
        vp = vac.ctypes.data_as(C.POINTER(C.c_uint8))
    return onsite, vac, vp, M, L


def num_threads():
    return lib().orc_num_threads()


def inverse(A):
    A = np.ascontiguousarray(A, dtype=np.complex128)
    n = A.shape[0]
    out = np.empty_like(A)
    rc = lib().orc_inverse(n, _dp(A), _dp(out))
    if rc:
        raise OracleError(rc, "inverse")
    return out


def matmul(A, B):
    A = np.ascontiguousarray(A, dtype=np.complex128)
    B = np.ascontiguousarray(B, dtype=np.complex128)
    out = np.empty_like(A)
    rc = lib().orc_matmul(A.shape[0], _dp(A), _dp(B), _dp(out))
    if rc:
        raise OracleError(rc, "matmul")
    return out


def lead_surface(M, L, t, E, eta, side, method=LEAD_CELL):
    g = np.empty((M, M), dtype=np.complex128)
    it = C.c_int(0)
    rc = lib().orc_lead_surface(M, L, t, E, eta, side, method, _dp(g), C.byref(it))
    if rc:
        raise OracleError(rc, "lead_surface")
    return g, it.value


def lead_self_energy(M, L, vacancy, t, E, eta, side, method=LEAD_CELL):
    vp = None
    if vacancy is not None:
        vac = np.ascontiguousarray(vacancy, dtype=np.uint8)
        vp = vac.ctypes.data_as(C.POINTER(C.c_uint8))
    S = np.empty((M, M), dtype=np.complex128)
    it = C.c_int(0)
    rc = lib().orc_lead_self_energy(M, L, vp, t, E, eta, side, method, _dp(S), C.byref(it))
    if rc:
        raise OracleError(rc, "lead_self_energy")
    return S, it.value


def transmission(onsite, vacancy, t, E, eta, direction=0, method=LEAD_CELL, full=False):
    onsite, vac, vp, M, L = _onsite(onsite, vacancy)
    T, im = C.c_double(0), C.c_double(0)
    its = (C.c_int * 2)()
    rc = lib().orc_transmission(M, L, _dp(onsite), vp, t, E, eta, direction, method, C.byref(T), C.byref(im), its)
    if rc:
        raise OracleError(rc, "transmission")
    if full:
        return T.value, im.value, (its[0], its[1])
    return T.value


def sweep_state(onsite, vacancy, t, E, eta, nslices, method=LEAD_CELL):
    onsite, vac, vp, M, L = _onsite(onsite, vacancy)
    g = np.empty((M, M), dtype=np.complex128)
    P = np.empty((M, M), dtype=np.complex128)
    rc = lib().orc_sweep_state(M, L, _dp(onsite), vp, t, E, eta, method, nslices, _dp(g), _dp(P))
    if rc:
        raise OracleError(rc, "sweep_state")
    return g, P


def transmission_batch(onsite, vacancy, t, energies, eta, method=LEAD_CELL, nthreads=0, return_status=False):
    onsite, vac, vp, M, L = _onsite(onsite, vacancy)
    energies = np.ascontiguousarray(energies, dtype=np.float64)
    n_E = energies.shape[0]
    T = np.empty(n_E, dtype=np.float64)
    st = np.zeros(n_E, dtype=np.int32)
    rc = lib().orc_transmission_batch(M, L, _dp(onsite), vp, t, _dp(energies), n_E, eta, method, nthreads,
                                      _dp(T), st.ctypes.data_as(C.POINTER(C.c_int)))
    if return_status:
        return T, st
    if rc:
        raise OracleError(rc, "transmission_batch")
    return T


def transmission_brute(onsite, vacancy, t, E, eta, method=LEAD_CELL):
    onsite, vac, vp, M, L = _onsite(onsite, vacancy)
    a, b = C.c_double(0), C.c_double(0)
    rc = lib().orc_transmission_brute(M, L, _dp(onsite), vp, t, E, eta, method, C.byref(a), C.byref(b))
    if rc:
        raise OracleError(rc, "transmission_brute")
    return a.value, b.value


def ldos_batch(onsite, vacancy, t, energies, eta, method=LEAD_CELL, nthreads=0):
    """LDOS[n_E][L][M] = -(1/pi) Im G_ii[j][j] of the connected device (orc_ldos_batch, O9)."""
    onsite, vac, vp, M, L = _onsite(onsite, vacancy)
    E = np.ascontiguousarray(energies, dtype=np.float64)
    out = np.empty((E.shape[0], L, M), dtype=np.float64)
    rc = lib().orc_ldos_batch(M, L, _dp(onsite), vp, t, _dp(E), E.shape[0], eta, method, nthreads, _dp(out))
    if rc:
        raise OracleError(rc, "ldos_batch")
    return out


def transmission_eq4_batch(onsite, vacancy, t, energies, eta, use_float, method=LEAD_CELL, nthreads=0):
    """T(E) by the paper's own Eq. 4 form (O10), double or single precision; a failed energy is NaN."""
    onsite, vac, vp, M, L = _onsite(onsite, vacancy)
    E = np.ascontiguousarray(energies, dtype=np.float64)
    T = np.empty(E.shape[0], dtype=np.float64)
    st = np.zeros(E.shape[0], dtype=np.int32)
    lib().orc_transmission_eq4_batch(M, L, _dp(onsite), vp, t, _dp(E), E.shape[0], eta, 1 if use_float else 0, method, nthreads, _dp(T),
                                     st.ctypes.data_as(C.POINTER(C.c_int)))
    return T
