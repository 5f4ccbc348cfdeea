"""ctypes front end of the CPU ORACLE (test infrastructure, NOT the product).

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this module.  It loads
``oracle/liberf_oracle.so`` (built by :func:`build` with
``gcc -O2 -ffp-contract=off``) and marshals numpy arrays; no arithmetic of the
method lives here.  See erf_oracle.h / erf_oracle.c for the citations.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liberf_oracle.so")
_SRC = os.path.join(_HERE, "erf_oracle.c")
_HDR = os.path.join(_HERE, "erf_oracle.h")

_dp = C.POINTER(C.c_double)


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("dx", C.c_double),
                ("dy", C.c_double), ("periodic_x", C.c_int), ("periodic_y", C.c_int)]


class Metrics(C.Structure):
    _fields_ = [("z_nodes", _dp), ("z_levels", _dp), ("rho0", _dp), ("rhotheta0", _dp),
                ("base_is_1d", C.c_int)]


class Params(C.Structure):
    _fields_ = [("Rd", C.c_double), ("cp", C.c_double), ("g", C.c_double), ("p00", C.c_double),
                ("adv_order_h", C.c_int), ("adv_order_v", C.c_int), ("diffusion", C.c_int),
                ("nu", C.c_double), ("alpha_theta", C.c_double), ("Cs", C.c_double),
                ("Pr_t", C.c_double), ("beta_s", C.c_double), ("beta_d", C.c_double),
                ("substep_mode", C.c_int), ("scalar_adv", C.c_int),
                ("ray_depth", C.c_double), ("ray_coef", C.c_double), ("ray_fields", C.c_int),
                ("ray_uref", C.c_double), ("ray_vref", C.c_double)]


_SO_OMP = os.path.join(_HERE, "liberf_oracle_omp.so")
_use_omp = False


def build(force: bool = False, omp: bool = False) -> str:
    """Compile the oracle (plain C, no FMA contraction) if stale.  ``omp``: the same source with -fopenmp
    (bitwise-identical results, see erf_oracle.c; for the long parity runs only)."""
    so = _SO_OMP if omp else _SO
    if (not force and os.path.exists(so)
            and os.path.getmtime(so) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return so
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c99", "-Wall", "-Wno-unknown-pragmas"]
    if omp:
        cmd.append("-fopenmp")
    subprocess.check_call(cmd + ["-o", so, _SRC, "-lm"])
    return so


def use_openmp(on: bool):
    """Switch every Oracle created from now on to the OpenMP build (False: back to the serial build)."""
    global _lib, _use_omp
    if on != _use_omp:
        _use_omp = on
        _lib = None


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build(omp=_use_omp))
        L.erfo_create.argtypes = [C.POINTER(Grid), C.POINTER(Metrics), C.POINTER(Params),
                                  C.POINTER(C.c_void_p)]
        L.erfo_set_state.argtypes = [C.c_void_p] + [_dp] * 5
        L.erfo_get_state.argtypes = [C.c_void_p] + [_dp] * 5
        L.erfo_rk3_step.argtypes = [C.c_void_p, C.c_double, C.c_int]
        L.erfo_set_scalar.argtypes = [C.c_void_p, _dp]
        L.erfo_get_scalar.argtypes = [C.c_void_p, _dp]
        L.erfo_anelastic_step.argtypes = [C.c_void_p, C.c_double]
        L.erfo_get_pprime.argtypes = [C.c_void_p, _dp]
        L.erfo_project.argtypes = [C.c_void_p, C.c_double]
        L.erfo_divergence.argtypes = [C.c_void_p, _dp]
        L.erfo_destroy.argtypes = [C.c_void_p]
        L.erfo_destroy.restype = None
        L.erfo_interp.argtypes = [C.c_int, C.c_double, _dp]
        L.erfo_interp.restype = C.c_double
        L.erfo_vertical_order.argtypes = [C.c_int, C.c_int]
        L.erfo_eos.argtypes = [C.c_double] * 5 + [_dp, _dp]
        L.erfo_eos.restype = None
        L.erfo_slow_rhs.argtypes = [C.c_void_p] + [_dp] * 5
        L.erfo_viscosity.argtypes = [C.c_void_p, _dp]
        L.erfo_get_geometry.argtypes = [C.c_void_p, C.c_char_p, _dp]
        L.erfo_acoustic.argtypes = [C.c_void_p, C.c_double, C.c_int] + [_dp] * 10
        L.erfo_tridiag_rows.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int, _dp, _dp, _dp]
        L.erfo_schedule.argtypes = [C.c_int, C.c_double, C.c_int, C.POINTER(C.c_int), _dp, _dp]
        L.erfo_schedule.restype = None
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def make_params(par: dict) -> Params:
    return Params(par["Rd"], par["cp"], par["g"], par["p00"], par["adv_order_h"],
                  par["adv_order_v"], par["diffusion"], par["nu"], par["alpha_theta"], par["Cs"],
                  par["Pr_t"], par["beta_s"], par["beta_d"], par["substep_mode"], par.get("scalar_adv", 0),
                  par.get("ray_depth", 0.0), par.get("ray_coef", 0.0), par.get("ray_fields", 0),
                  par.get("ray_uref", 0.0), par.get("ray_vref", 0.0))


class Oracle:
    """One oracle context.  ``case`` is a dict as produced by
    paper_2412_04395_b200.workloads (plain data: grid, metrics, params)."""

    def __init__(self, case: dict):
        L = lib()
        self.nx, self.ny, self.nz = case["nx"], case["ny"], case["nz"]
        g = Grid(self.nx, self.ny, self.nz, case["dx"], case["dy"], int(case.get("periodic_x", 1)),
                 int(case.get("periodic_y", 1)))
        self._keep = []
        m = Metrics()
        if case.get("z_nodes") is not None:
            zn = _c(case["z_nodes"])
            assert zn.shape == (self.nz + 1, self.ny + 1, self.nx + 1)
            self._keep.append(zn)
            m.z_nodes = _p(zn)
        else:
            zl = _c(case["z_levels"])
            assert zl.shape == (self.nz + 1,)
            self._keep.append(zl)
            m.z_levels = _p(zl)
        r0, t0 = _c(case["rho0"]), _c(case["rhotheta0"])
        self._keep += [r0, t0]
        m.rho0, m.rhotheta0 = _p(r0), _p(t0)
        m.base_is_1d = 1 if r0.ndim == 1 else 0
        p = make_params(case["params"])
        h = C.c_void_p()
        rc = L.erfo_create(C.byref(g), C.byref(m), C.byref(p), C.byref(h))
        if rc != 0:
            raise RuntimeError(f"erfo_create failed: {rc}")
        self._h = h
        self._L = L

    def close(self):
        if self._h:
            self._L.erfo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def shape_c(self):
        return (self.nz, self.ny, self.nx)

    @property
    def shape_w(self):
        return (self.nz + 1, self.ny, self.nx)

    def set_state(self, rho, U, V, W, Th):
        a = [_c(rho), _c(U), _c(V), _c(W), _c(Th)]
        assert a[0].shape == self.shape_c and a[3].shape == self.shape_w
        rc = self._L.erfo_set_state(self._h, *[_p(x) for x in a])
        assert rc == 0

    def get_state(self):
        out = [np.empty(self.shape_c), np.empty(self.shape_c), np.empty(self.shape_c),
               np.empty(self.shape_w), np.empty(self.shape_c)]
        rc = self._L.erfo_get_state(self._h, *[_p(x) for x in out])
        assert rc == 0
        return out

    def set_scalar(self, rhophi):
        a = _c(rhophi)
        assert a.shape == self.shape_c
        assert self._L.erfo_set_scalar(self._h, _p(a)) == 0

    def get_scalar(self):
        out = np.empty(self.shape_c)
        assert self._L.erfo_get_scalar(self._h, _p(out)) == 0
        return out

    def step(self, dt, n_acoustic):
        rc = self._L.erfo_rk3_step(self._h, float(dt), int(n_acoustic))
        if rc != 0:
            raise RuntimeError(f"erfo_rk3_step failed: {rc}")

    def anelastic_step(self, dt):
        rc = self._L.erfo_anelastic_step(self._h, float(dt))
        if rc != 0:
            raise RuntimeError(f"erfo_anelastic_step failed: {rc}")

    def project(self, dt):
        assert self._L.erfo_project(self._h, float(dt)) == 0

    def divergence(self):
        out = np.empty(self.shape_c)
        assert self._L.erfo_divergence(self._h, _p(out)) == 0
        return out

    def pprime(self):
        out = np.empty(self.shape_c)
        assert self._L.erfo_get_pprime(self._h, _p(out)) == 0
        return out

    def slow_rhs(self):
        out = [np.empty(self.shape_c), np.empty(self.shape_c), np.empty(self.shape_c),
               np.empty(self.shape_w), np.empty(self.shape_c)]
        rc = self._L.erfo_slow_rhs(self._h, *[_p(x) for x in out])
        assert rc == 0
        return out

    def viscosity(self):
        mu = np.empty(self.shape_c)
        assert self._L.erfo_viscosity(self._h, _p(mu)) == 0
        return mu

    def geometry(self, name):
        out = np.empty(self.shape_w)
        assert self._L.erfo_get_geometry(self._h, name.encode(), _p(out)) == 0
        return out

    def acoustic(self, dtau, n, R, P):
        """R, P: lists (rho, U, V, W, Theta); returns the new S''."""
        Rc = [_c(x) for x in R]
        Pc = [_c(x).copy() for x in P]
        rc = self._L.erfo_acoustic(self._h, float(dtau), int(n), *[_p(x) for x in Rc],
                                   *[_p(x) for x in Pc])
        assert rc == 0
        return Pc

    def tridiag_rows(self, dtau, i, j):
        A, D, Cc = (np.zeros(self.nz + 1) for _ in range(3))
        assert self._L.erfo_tridiag_rows(self._h, float(dtau), i, j, _p(A), _p(D), _p(Cc)) == 0
        return A, D, Cc


def interp(order, sgn, q):
    q = _c(q)
    assert q.shape == (6,)
    return lib().erfo_interp(int(order), float(sgn), _p(q))


def vertical_order(requested, r):
    return lib().erfo_vertical_order(int(requested), int(r))


def eos(Rd, cp, p00, Theta, Theta0):
    pp, pi = C.c_double(), C.c_double()
    lib().erfo_eos(Rd, cp, p00, Theta, Theta0, C.byref(pp), C.byref(pi))
    return pp.value, pi.value


def schedule(stage, dt, ns):
    n, dtau, dts = C.c_int(), C.c_double(), C.c_double()
    lib().erfo_schedule(stage, dt, ns, C.byref(n), C.byref(dtau), C.byref(dts))
    return n.value, dtau.value, dts.value
