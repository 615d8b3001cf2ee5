"""Thin ctypes binding of the C ABI in include/rgf.h -- argument marshalling only.

Every function has the name and argument order of its C counterpart; arrays may be numpy
arrays (host pointers) or torch CUDA tensors (device pointers).  All computation happens in
the CUDA kernels of librgf_b200.so; importing this module fails loudly if the library has
not been built (python -m paper_1107_5300_b200.build) -- there is no CPU fallback.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librgf_b200.so")

RGF_C128, RGF_C64 = 0, 1
RGF_FORM_DENSE, RGF_FORM_HALF, RGF_FORM_HALF_STEPWISE = 0, 1, 2
RGF_LEAD_CELL_DENSE, RGF_LEAD_CELL_SCHUR, RGF_LEAD_MODE_SPACE = 0, 1, 2
RGF_OK, RGF_EINVAL, RGF_ECUDA, RGF_ENOMEM, RGF_ENOCONV, RGF_ESINGULAR, RGF_ESTATE, RGF_EUNSUPPORTED = 0, -1, -2, -3, -4, -5, -6, -7

if not os.path.exists(LIB_PATH):
    raise ImportError("%s is missing: build it with `python -m paper_1107_5300_b200.build` "
                      "(the RGF path has no CPU fallback)" % LIB_PATH)
_lib = C.CDLL(LIB_PATH)


class rgf_stats(C.Structure):
    _fields_ = [("ms_total", C.c_double), ("ms_leads", C.c_double), ("ms_sweep", C.c_double), ("ms_trace", C.c_double),
                ("ms_inverse_update", C.c_double), ("launches", C.c_longlong), ("launches_inverse_update", C.c_longlong), ("launches_leads", C.c_longlong),
                ("lead_iterations", C.c_int), ("cohort", C.c_int), ("guard_redone", C.c_int), ("reserved", C.c_int), ("ms_guard", C.c_double)]


_vp = C.c_void_p
_lib.rgf_plan_create.argtypes = [C.POINTER(_vp), C.c_int, _vp]
_lib.rgf_set_device.argtypes = [_vp, C.c_int, C.c_int, _vp, C.c_double, _vp]
_lib.rgf_set_device_batch.argtypes = [_vp, C.c_int, C.c_int, C.c_int, _vp, C.c_double, _vp]
_lib.rgf_transmission.argtypes = [_vp, _vp, C.c_int, C.c_double, C.c_int, _vp]
_lib.rgf_destroy.argtypes = [_vp]
_lib.rgf_last_error.argtypes = [_vp]
_lib.rgf_last_error.restype = C.c_char_p
_lib.rgf_get_stats.argtypes = [_vp, C.POINTER(rgf_stats)]
_lib.rgf_set_profiling.argtypes = [_vp, C.c_int]
_lib.rgf_set_cohort.argtypes = [_vp, C.c_int]
_lib.rgf_set_formulation.argtypes = [_vp, C.c_int]
_lib.rgf_set_lead_method.argtypes = [_vp, C.c_int]
_lib.rgf_set_guard.argtypes = [_vp, C.c_double]
_lib.rgf_get_guard_indicators.argtypes = [_vp, _vp, _vp, C.c_int]
_lib.rgf_fp64_peak_tflops.argtypes = [_vp, C.POINTER(C.c_double)]
_lib.rgf_inverse_batched.argtypes = [_vp, C.c_int, C.c_int, _vp, _vp]
_lib.rgf_lead_self_energy.argtypes = [_vp, C.c_int, _vp, C.c_int, C.c_double, C.c_int, _vp, C.POINTER(C.c_int)]
_lib.rgf_sweep_state.argtypes = [_vp, C.c_int, _vp, C.c_int, C.c_double, C.c_int, C.c_int, _vp, _vp]
_lib.rgf_shard_count.argtypes = [C.c_int, C.c_int, C.c_int]
_lib.rgf_shard_energies.argtypes = [_vp, C.c_int, C.c_int, C.c_int, _vp]
_lib.rgf_unshard.argtypes = [_vp, C.c_int, C.c_int, C.c_int, C.c_int, _vp]
_lib.rgf_ldos.argtypes = [_vp, _vp, C.c_int, C.c_double, _vp]
_lib.rgf_inverse_batched_static.argtypes = [C.c_int, _vp, C.c_int, C.c_int, _vp, _vp, _vp]
_lib.rgf_static_last_error.restype = C.c_char_p


class RgfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("rgf error %d: %s" % (code, msg))
        self.code = code


def _addr(a, dtype=None):
    """Pointer of a numpy array (host) or a torch CUDA/CPU tensor; None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"], "array must be C-contiguous"
        if dtype is not None:
            assert a.dtype == dtype, (a.dtype, dtype)
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        assert a.is_contiguous()
        return a.data_ptr()
    raise TypeError(type(a))


def _check(plan, rc, ok=()):
    if rc != RGF_OK and rc not in ok:
        raise RgfError(rc, rgf_last_error(plan))
    return rc


def rgf_plan_create(cuda_device=0, cuda_stream=None):
    out = _vp()
    rc = _lib.rgf_plan_create(C.byref(out), cuda_device, cuda_stream)
    if rc != RGF_OK:
        raise RgfError(rc, "rgf_plan_create failed")
    return out


def rgf_last_error(plan):
    return _lib.rgf_last_error(plan).decode()


def rgf_set_device(plan, M, L, onsite, t, vacancy=None):
    return _check(plan, _lib.rgf_set_device(plan, M, L, _addr(onsite), t, _addr(vacancy)))


def rgf_set_device_batch(plan, n_dev, M, L, onsite, t, vacancy=None):
    return _check(plan, _lib.rgf_set_device_batch(plan, n_dev, M, L, _addr(onsite), t, _addr(vacancy)))


def rgf_transmission(plan, energies, n_E, eta, precision, T_out, ok=()):
    return _check(plan, _lib.rgf_transmission(plan, _addr(energies), n_E, eta, precision, _addr(T_out)), ok)


def rgf_destroy(plan):
    return _lib.rgf_destroy(plan)


def rgf_get_stats(plan):
    s = rgf_stats()
    _lib.rgf_get_stats(plan, C.byref(s))
    return {k: getattr(s, k) for k, _ in rgf_stats._fields_}


def rgf_set_profiling(plan, level):
    return _check(plan, _lib.rgf_set_profiling(plan, level))


def rgf_set_formulation(plan, formulation):
    return _check(plan, _lib.rgf_set_formulation(plan, formulation))


def rgf_set_lead_method(plan, method):
    return _check(plan, _lib.rgf_set_lead_method(plan, method))


def rgf_set_cohort(plan, cohort):
    return _check(plan, _lib.rgf_set_cohort(plan, cohort))


def rgf_set_guard(plan, tol):
    return _check(plan, _lib.rgf_set_guard(plan, tol))


def rgf_get_guard_indicators(plan, Grms_out, Gmax_out, n):
    return _check(plan, _lib.rgf_get_guard_indicators(plan, _addr(Grms_out, np.float64), _addr(Gmax_out, np.float64), n))


def rgf_fp64_peak_tflops(plan):
    out = C.c_double(0.0)
    _check(plan, _lib.rgf_fp64_peak_tflops(plan, C.byref(out)))
    return out.value


def rgf_inverse_batched(plan, n, batch, A, Ainv):
    return _check(plan, _lib.rgf_inverse_batched(plan, n, batch, _addr(A), _addr(Ainv)))


def rgf_lead_self_energy(plan, dev, energies, n_E, eta, side, Sigma_out):
    it = C.c_int(0)
    _check(plan, _lib.rgf_lead_self_energy(plan, dev, _addr(energies), n_E, eta, side, _addr(Sigma_out), C.byref(it)))
    return it.value


def rgf_sweep_state(plan, dev, energies, n_E, eta, precision, nslices, g_out, P_out):
    return _check(plan, _lib.rgf_sweep_state(plan, dev, _addr(energies), n_E, eta, precision, nslices, _addr(g_out), _addr(P_out)))


def rgf_shard_count(n_E, world, rank):
    return _lib.rgf_shard_count(n_E, world, rank)


def rgf_shard_energies(energies, n_E, world, rank, shard_out):
    """Host numpy arrays; returns the number of energies written."""
    return _lib.rgf_shard_energies(_addr(energies, np.float64), n_E, world, rank, _addr(shard_out, np.float64))


def rgf_unshard(T_shard, n_dev, n_E, world, rank, T_full):
    rc = _lib.rgf_unshard(_addr(T_shard, np.float64), n_dev, n_E, world, rank, _addr(T_full, np.float64))
    if rc != RGF_OK:
        raise RgfError(rc, "rgf_unshard: bad argument")
    return rc


def rgf_ldos(plan, energies, n_E, eta, ldos_out):
    return _check(plan, _lib.rgf_ldos(plan, _addr(energies), n_E, eta, _addr(ldos_out)))


def rgf_static_last_error():
    return _lib.rgf_static_last_error().decode()


def rgf_inverse_batched_static(cuda_device, cuda_stream, n, batch, A_dev, Ainv_dev, status_dev=None):
    """Allocation-free inverse (include/rgf.h): device tensors in and out, scratch in the library's static array."""
    rc = _lib.rgf_inverse_batched_static(cuda_device, cuda_stream, n, batch, _addr(A_dev), _addr(Ainv_dev), _addr(status_dev))
    if rc != RGF_OK:
        raise RgfError(rc, rgf_static_last_error())
    return rc


class Plan:
    """Context manager around rgf_plan_create / rgf_destroy (no arithmetic, marshalling only)."""

    def __init__(self, cuda_device=0, cuda_stream=None):
        self.handle = rgf_plan_create(cuda_device, cuda_stream)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def close(self):
        if self.handle is not None:
            rgf_destroy(self.handle)
            self.handle = None

    def set_device(self, onsite, t, vacancy=None):
        """onsite [L][M] or [n_dev][L][M] float64 (numpy)."""
        onsite = np.ascontiguousarray(onsite, dtype=np.float64)
        if onsite.ndim == 2:
            onsite = onsite[None]
        n_dev, L, M = onsite.shape
        vac = None if vacancy is None else np.ascontiguousarray(vacancy, dtype=np.uint8).reshape(n_dev, L, M)
        self.n_dev, self.L, self.M = n_dev, L, M
        rgf_set_device_batch(self.handle, n_dev, M, L, onsite, t, vac)

    def transmission(self, energies, eta, precision=RGF_C128, ok=()):
        """Host convenience: numpy energies in, numpy T[n_dev][n_E] out."""
        energies = np.ascontiguousarray(energies, dtype=np.float64)
        T = np.empty((self.n_dev, energies.shape[0]), dtype=np.float64)
        rgf_transmission(self.handle, energies, energies.shape[0], eta, precision, T, ok)
        return T

    def ldos(self, energies, eta):
        """Host convenience: numpy energies in, numpy LDOS[n_dev][n_E][L][M] out."""
        energies = np.ascontiguousarray(energies, dtype=np.float64)
        out = np.empty((self.n_dev, energies.shape[0], self.L, self.M), dtype=np.float64)
        rgf_ldos(self.handle, energies, energies.shape[0], eta, out)
        return out

    def stats(self):
        return rgf_get_stats(self.handle)
