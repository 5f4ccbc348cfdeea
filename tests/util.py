"""Helpers for the oracle pin tests: simple hand-built cases (plain data)."""
import numpy as np

from paper_2412_04395_b200 import workloads as wl


def uniform_case(nx, ny, nz, dx, dy, dz, theta0=300.0, rho0=1.0, g=0.0, **par):
    """Uniform base state (no gravity unless asked), flat uniform grid."""
    p = dict(wl.DEFAULT_PARAMS)
    p.update(g=g)
    p.update(par)
    zl = np.arange(nz + 1, dtype=np.float64) * dz
    return dict(name="uniform", nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, z_nodes=None, z_levels=zl,
                rho0=np.full(nz, rho0), rhotheta0=np.full(nz, rho0 * theta0), params=p)


def zeros_state(case):
    nx, ny, nz = case["nx"], case["ny"], case["nz"]
    c = (nz, ny, nx)
    return [np.zeros(c), np.zeros(c), np.zeros(c), np.zeros((nz + 1, ny, nx)), np.zeros(c)]


def base_state_fields(case):
    """(rho0, Theta0) broadcast to [nz][ny][nx]."""
    nx, ny, nz = case["nx"], case["ny"], case["nz"]
    r0, t0 = case["rho0"], case["rhotheta0"]
    if r0.ndim == 1:
        r0 = np.broadcast_to(r0[:, None, None], (nz, ny, nx))
        t0 = np.broadcast_to(t0[:, None, None], (nz, ny, nx))
    return np.array(r0), np.array(t0)


def rel_err(a, b, scale=None):
    s = scale if scale is not None else max(np.abs(b).max(), 1e-300)
    return float(np.abs(a - b).max() / s)


def field_errors(got, ref):
    """Max relative field error per field (reading G24): |got-ref|_max / scale with
    scale_rho = max|rho|, scale_Theta = max|Theta| and ONE shared scale max(|U|,|V|,|W|) for the
    three momenta.  Order (rho, U, V, W, Theta)."""
    got = [np.asarray(a) for a in got]
    ref = [np.asarray(a) for a in ref]
    tiny = 1e-300
    sm = max(max(float(np.abs(ref[f]).max()) for f in (1, 2, 3)), tiny)
    scale = [max(float(np.abs(ref[0]).max()), tiny), sm, sm, sm, max(float(np.abs(ref[4]).max()), tiny)]
    return [float(np.abs(got[f] - ref[f]).max() / scale[f]) for f in range(5)]


def perturbation_errors(got, ref, case):
    """A stricter companion of G24 (reported beside it): the error of each field relative to what
    actually moves -- rho - rho0 and Theta - Theta0 against the largest perturbation, W against max|W| alone (not
    the shared momentum scale), U and V against their largest departure from the horizontal mean of each level.
    Order (rho', U', V', W, Theta')."""
    got = [np.asarray(a) for a in got]
    ref = [np.asarray(a) for a in ref]
    r0, t0 = base_state_fields(case)
    tiny = 1e-300

    def dev(a):
        return a - a.mean(axis=(1, 2), keepdims=True)

    scale = [max(float(np.abs(ref[0] - r0).max()), tiny), max(float(np.abs(dev(ref[1])).max()), tiny),
             max(float(np.abs(dev(ref[2])).max()), tiny), max(float(np.abs(ref[3]).max()), tiny),
             max(float(np.abs(ref[4] - t0).max()), tiny)]
    return [float(np.abs(got[f] - ref[f]).max() / scale[f]) for f in range(5)]
