"""Thin ctypes binding of liberf_b200.so (include/erf_b200.h): argument marshalling only.

Every step of the RK3 dycore path runs inside the CUDA library; PyTorch supplies device
memory (``tensor.data_ptr()``) and the stream (``torch.cuda.current_stream().cuda_stream``)
and does nothing else.  There is no CPU fallback: importing works without a GPU (so the
symbol table can be checked), but creating a context without the built library or without a
CUDA device raises.

The module-level functions carry the C names (erf_create, erf_set_state, erf_rk3_step,
erf_get_state, erf_destroy, ...); :class:`Dycore` wraps one context for convenience.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liberf_b200.so")

ERF_OK, ERF_EINVAL, ERF_EUNSUPPORTED, ERF_ENOMEM, ERF_ECUDA, ERF_ETOOLARGE = 0, -1, -2, -3, -4, -5
ERF_NOALLOC_MAX_VALUES = 1048576  # erf_poisson_modes_noalloc: nx*ny*nz limit (doubles of built-in work space)
ERF_PATH_AUTO, ERF_PATH_GENERAL = 0, 1
# erf_set_option keys and ERF_OPT_VARIANT bits (include/erf_b200.h, diagnostics block)
ERF_OPT_VARIANT, ERF_OPT_GRAPH = 1, 2
ERF_VARIANT_DIFF_SPLIT = 1024
ERF_VARIANT_FORCE_COLUMN, ERF_VARIANT_SPLIT_SLOW_RHS, ERF_VARIANT_FORCE_TILE = 4096, 8192, 16384

EXPORTS = ["erf_create", "erf_set_state", "erf_rk3_step", "erf_get_state", "erf_destroy",
           "erf_strerror", "erf_set_scalar", "erf_get_scalar", "erf_anelastic_step", "erf_get_pprime", "erf_project", "erf_slow_rhs", "erf_acoustic", "erf_set_path", "erf_set_option", "erf_launch_count",
           "erf_device_bytes", "erf_set_timing", "erf_get_timing", "erf_reset_timing", "erf_timing_name",
           "erf_measure_fp64_peak", "erf_poisson_modes_noalloc"]
ERF_TIMING_CLASSES = 8

_dp = C.c_void_p


class erf_grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("dx", C.c_double),
                ("dy", C.c_double), ("periodic_x", C.c_int), ("periodic_y", C.c_int)]


class erf_metrics(C.Structure):
    _fields_ = [("z_nodes", _dp), ("z_levels", _dp), ("rho0", _dp), ("rhotheta0", _dp),
                ("base_is_1d", C.c_int)]


class erf_params(C.Structure):
    _fields_ = [("Rd", C.c_double), ("cp", C.c_double), ("g", C.c_double), ("p00", C.c_double),
                ("adv_order_h", C.c_int), ("adv_order_v", C.c_int), ("diffusion", C.c_int),
                ("nu", C.c_double), ("alpha_theta", C.c_double), ("Cs", C.c_double),
                ("Pr_t", C.c_double), ("beta_s", C.c_double), ("beta_d", C.c_double),
                ("substep_mode", C.c_int), ("scalar_adv", C.c_int),
                ("ray_depth", C.c_double), ("ray_coef", C.c_double), ("ray_fields", C.c_int),
                ("ray_uref", C.c_double), ("ray_vref", C.c_double)]


class ErfError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = _lib.erf_strerror(code).decode() if _lib is not None else "?"
        super().__init__(f"{where}: {msg} ({code})")


_lib = None


def load(path: str | None = None):
    """Load the C-ABI library (fails loudly if it has not been built)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise FileNotFoundError(
            f"{p} is missing: build it with `python -m paper_2412_04395_b200.build` "
            "(nvcc, sm_100a). There is no CPU fallback.")
    L = C.CDLL(p)
    L.erf_create.argtypes = [C.POINTER(erf_grid), C.POINTER(erf_metrics), C.POINTER(erf_params),
                             C.c_void_p, C.POINTER(C.c_void_p)]
    L.erf_set_state.argtypes = [C.c_void_p] + [_dp] * 5 + [C.c_void_p]
    L.erf_get_state.argtypes = [C.c_void_p] + [_dp] * 5 + [C.c_void_p]
    L.erf_rk3_step.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_void_p]
    L.erf_destroy.argtypes = [C.c_void_p]
    L.erf_destroy.restype = None
    L.erf_strerror.argtypes = [C.c_int]
    L.erf_strerror.restype = C.c_char_p
    L.erf_slow_rhs.argtypes = [C.c_void_p] + [_dp] * 5 + [C.c_void_p]
    L.erf_acoustic.argtypes = [C.c_void_p, C.c_double, C.c_int] + [_dp] * 10 + [C.c_void_p]
    L.erf_set_scalar.argtypes = [C.c_void_p, _dp, C.c_void_p]
    L.erf_get_scalar.argtypes = [C.c_void_p, _dp, C.c_void_p]
    L.erf_anelastic_step.argtypes = [C.c_void_p, C.c_double, C.c_void_p]
    L.erf_project.argtypes = [C.c_void_p, C.c_double, C.c_void_p]
    L.erf_get_pprime.argtypes = [C.c_void_p, _dp, C.c_void_p]
    L.erf_set_path.argtypes = [C.c_void_p, C.c_int]
    L.erf_set_option.argtypes = [C.c_void_p, C.c_int, C.c_longlong]
    L.erf_launch_count.argtypes = [C.c_void_p]
    L.erf_launch_count.restype = C.c_longlong
    L.erf_device_bytes.argtypes = [C.c_void_p]
    L.erf_device_bytes.restype = C.c_longlong
    L.erf_set_timing.argtypes = [C.c_void_p, C.c_int]
    L.erf_reset_timing.argtypes = [C.c_void_p]
    L.erf_get_timing.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_longlong), C.POINTER(C.c_double)]
    L.erf_timing_name.argtypes = [C.c_int]
    L.erf_timing_name.restype = C.c_char_p
    L.erf_measure_fp64_peak.argtypes = [C.POINTER(C.c_double), C.c_void_p]
    L.erf_poisson_modes_noalloc.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [_dp] * 4 + [C.c_void_p]
    _lib = L
    return L


def _ptr(t):
    """Device pointer of a contiguous fp64 CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("expected a contiguous float64 CUDA tensor")
    return t.data_ptr()


def _stream(stream):
    if stream is not None:
        return C.c_void_p(int(stream))
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ck(rc, where):
    if rc != ERF_OK:
        raise ErfError(rc, where)


# ---- functions with the C names -------------------------------------------------------

def erf_create(grid: erf_grid, metrics: erf_metrics, params: erf_params, stream=None):
    h = C.c_void_p()
    _ck(load().erf_create(C.byref(grid), C.byref(metrics), C.byref(params), _stream(stream), C.byref(h)),
        "erf_create")
    return h


def erf_set_state(h, rho, rhou, rhov, rhow, rhotheta, stream=None):
    _ck(load().erf_set_state(h, _ptr(rho), _ptr(rhou), _ptr(rhov), _ptr(rhow), _ptr(rhotheta),
                             _stream(stream)), "erf_set_state")


def erf_rk3_step(h, dt, n_acoustic, stream=None):
    _ck(load().erf_rk3_step(h, float(dt), int(n_acoustic), _stream(stream)), "erf_rk3_step")


def erf_get_state(h, rho, rhou, rhov, rhow, rhotheta, stream=None):
    _ck(load().erf_get_state(h, _ptr(rho), _ptr(rhou), _ptr(rhov), _ptr(rhow), _ptr(rhotheta),
                             _stream(stream)), "erf_get_state")


def erf_set_scalar(h, rhophi, stream=None):
    _ck(load().erf_set_scalar(h, _ptr(rhophi), _stream(stream)), "erf_set_scalar")


def erf_get_scalar(h, rhophi, stream=None):
    _ck(load().erf_get_scalar(h, _ptr(rhophi), _stream(stream)), "erf_get_scalar")


def erf_anelastic_step(h, dt, stream=None):
    _ck(load().erf_anelastic_step(h, float(dt), _stream(stream)), "erf_anelastic_step")


def erf_project(h, dt, stream=None):
    _ck(load().erf_project(h, float(dt), _stream(stream)), "erf_project")


def erf_get_pprime(h, pprime, stream=None):
    _ck(load().erf_get_pprime(h, _ptr(pprime), _stream(stream)), "erf_get_pprime")


def erf_poisson_modes_noalloc(nx, ny, nz, dx, dy, dt, dz, dzw, hat_re, hat_im, stream=None):
    """Eq. 16's tridiagonal solve per horizontal mode, in place in (hat_re, hat_im), for callers that may not allocate
    device memory (include/erf_b200.h): no context, the work space is a fixed array inside the library, so
    nx*ny*nz <= ERF_NOALLOC_MAX_VALUES and calls on one GPU must not overlap.  All four arrays are float64 CUDA tensors."""
    _ck(load().erf_poisson_modes_noalloc(int(nx), int(ny), int(nz), float(dx), float(dy), float(dt), _ptr(dz),
                                         _ptr(dzw), _ptr(hat_re), _ptr(hat_im), _stream(stream)),
        "erf_poisson_modes_noalloc")


def erf_destroy(h):
    if h:
        load().erf_destroy(h)


def erf_slow_rhs(h, R_rho, R_U, R_V, R_W, R_Theta, stream=None):
    _ck(load().erf_slow_rhs(h, _ptr(R_rho), _ptr(R_U), _ptr(R_V), _ptr(R_W), _ptr(R_Theta),
                            _stream(stream)), "erf_slow_rhs")


def erf_acoustic(h, dtau, n, R, P, stream=None):
    _ck(load().erf_acoustic(h, float(dtau), int(n), *[_ptr(x) for x in R], *[_ptr(x) for x in P],
                            _stream(stream)), "erf_acoustic")


def erf_set_path(h, path):
    _ck(load().erf_set_path(h, int(path)), "erf_set_path")


def erf_set_option(h, key, value):
    _ck(load().erf_set_option(h, int(key), int(value)), "erf_set_option")


def erf_launch_count(h):
    return int(load().erf_launch_count(h))


def erf_device_bytes(h):
    return int(load().erf_device_bytes(h))


def erf_measure_fp64_peak(stream=None):
    """Measured fp64 FMA peak of the current device in TFLOP/s (FMA = 2 flop)."""
    v = C.c_double(0.0)
    _ck(load().erf_measure_fp64_peak(C.byref(v), _stream(stream)), "erf_measure_fp64_peak")
    return v.value


def erf_set_timing(h, on):
    _ck(load().erf_set_timing(h, int(bool(on))), "erf_set_timing")


def erf_reset_timing(h):
    _ck(load().erf_reset_timing(h), "erf_reset_timing")


def erf_get_timing(h, idx):
    n, ms = C.c_longlong(), C.c_double()
    _ck(load().erf_get_timing(h, int(idx), C.byref(n), C.byref(ms)), "erf_get_timing")
    return n.value, ms.value


def erf_timing_name(idx):
    return load().erf_timing_name(int(idx)).decode()


def make_params(par: dict) -> erf_params:
    return erf_params(par["Rd"], par["cp"], par["g"], par["p00"], par["adv_order_h"],
                      par["adv_order_v"], par["diffusion"], par["nu"], par["alpha_theta"], par["Cs"],
                      par["Pr_t"], par["beta_s"], par["beta_d"], par["substep_mode"], par.get("scalar_adv", 0),
                      par.get("ray_depth", 0.0), par.get("ray_coef", 0.0), par.get("ray_fields", 0),
                      par.get("ray_uref", 0.0), par.get("ray_vref", 0.0))


# ---- convenience wrapper ---------------------------------------------------------------

class Dycore:
    """One context built from a workload dict (paper_2412_04395_b200.workloads.make_case)."""

    def __init__(self, case: dict, device="cuda:0", stream=None):
        import numpy as np
        import torch
        load()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: liberf_b200 has no CPU fallback")
        self.device = torch.device(device)
        self.nx, self.ny, self.nz = case["nx"], case["ny"], case["nz"]
        g = erf_grid(self.nx, self.ny, self.nz, case["dx"], case["dy"], int(case.get("periodic_x", 1)),
                     int(case.get("periodic_y", 1)))
        m = erf_metrics()
        keep = []

        def dev(a):
            t = torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).to(self.device)
            keep.append(t)
            return t

        with torch.cuda.device(self.device):
            if case.get("z_nodes") is not None:
                zn = dev(case["z_nodes"])
                assert tuple(zn.shape) == (self.nz + 1, self.ny + 1, self.nx + 1)
                m.z_nodes = zn.data_ptr()
            else:
                zl = np.ascontiguousarray(case["z_levels"], dtype=np.float64)
                assert zl.shape == (self.nz + 1,)
                keep.append(zl)
                m.z_levels = zl.ctypes.data
            r0, t0 = dev(case["rho0"]), dev(case["rhotheta0"])
            m.rho0, m.rhotheta0 = r0.data_ptr(), t0.data_ptr()
            m.base_is_1d = 1 if r0.dim() == 1 else 0
            self._h = erf_create(g, m, make_params(case["params"]), stream)
        del keep  # erf_create has synchronised: the library holds its own copies
        self._torch = torch

    # shapes
    @property
    def shape_c(self):
        return (self.nz, self.ny, self.nx)

    @property
    def shape_w(self):
        return (self.nz + 1, self.ny, self.nx)

    def empty_state(self):
        t = self._torch
        return [t.empty(self.shape_w if f == 3 else self.shape_c, dtype=t.float64, device=self.device)
                for f in range(5)]

    def close(self):
        if getattr(self, "_h", None):
            erf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, rho, U, V, W, Th, stream=None):
        erf_set_state(self._h, rho, U, V, W, Th, stream)

    def set_scalar(self, rhophi, stream=None):
        erf_set_scalar(self._h, rhophi, stream)

    def anelastic_step(self, dt, stream=None):
        erf_anelastic_step(self._h, dt, stream)

    def project(self, dt, stream=None):
        erf_project(self._h, dt, stream)

    def pprime(self, stream=None):
        out = self.empty_state()[0]
        erf_get_pprime(self._h, out, stream)
        return out

    def get_scalar(self, stream=None):
        out = self.empty_state()[0]
        erf_get_scalar(self._h, out, stream)
        return out

    def get_state(self, out=None, stream=None):
        out = out if out is not None else self.empty_state()
        erf_get_state(self._h, *out, stream=stream)
        return out

    def rk3_step(self, dt, n_acoustic, stream=None):
        erf_rk3_step(self._h, dt, n_acoustic, stream)

    def slow_rhs(self, stream=None):
        out = self.empty_state()
        erf_slow_rhs(self._h, *out, stream=stream)
        return out

    def acoustic(self, dtau, n, R, P, stream=None):
        P = [p.clone() for p in P]
        erf_acoustic(self._h, dtau, n, R, P, stream)
        return P

    def set_path(self, path):
        erf_set_path(self._h, path)

    def set_option(self, key, value):
        erf_set_option(self._h, key, value)

    def set_timing(self, on):
        erf_set_timing(self._h, on)

    def reset_timing(self):
        erf_reset_timing(self._h)

    def timing(self):
        """{class name: (launch groups, total device ms)} since the last reset."""
        out = {}
        for i in range(ERF_TIMING_CLASSES):
            n, ms = erf_get_timing(self._h, i)
            if n:
                out[erf_timing_name(i)] = (n, ms)
        return out

    @property
    def launch_count(self):
        return erf_launch_count(self._h)

    @property
    def device_bytes(self):
        return erf_device_bytes(self._h)
