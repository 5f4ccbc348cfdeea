"""Pins of the oracle's transported scalar (Eq. 4), advanced in every RK stage after the acoustic
substeps with the stage-time-averaged normal momenta (L138).  Closed forms and invariants only."""
import math
import os

import numpy as np
import pytest

from oracle import erfo
from paper_2412_04395_b200 import workloads as wl
from util import uniform_case, zeros_state


def _fsum(a):
    return math.fsum(a.ravel().tolist())


def _hill(nx=28, ny=10, nz=20, height=250.0, **par):
    """Config 4 shrunk: fewer (stretched) levels reach ~540 m only, so the hill is lowered to stay below the top."""
    wl.CONFIGS[4]["hill"]["height"] = height
    try:
        return wl.make_case(4, nx=nx, ny=ny, nz=nz, params=par)
    finally:
        wl.CONFIGS[4]["hill"]["height"] = 400.0


@pytest.mark.parametrize("cfg,kw", [(1, dict(nx=12, ny=10, nz=12)), (2, dict(nx=12, ny=12, nz=14)),
                                    (3, dict(nx=10, ny=12, nz=14)), (4, None)])
def test_constant_scalar_stays_constant_and_mass_is_conserved(cfg, kw):
    """L138: the scalar is advected by the time average of the very momenta that advanced rho in the substeps.
    Then (rho phi) with phi = const obeys the substepped continuity equation exactly: phi stays constant to
    round-off -- with substeps, off-centring, divergence damping, diffusion and terrain.  Any other choice of
    momenta (stage momenta alone, only the new or only the old Omega'') breaks this at 1e-4 .. 1e-8.
    A non-constant scalar keeps sum(rho phi * cell volume) (flux form, L69)."""
    case = _hill() if cfg == 4 else wl.make_case(cfg, **kw)
    o = erfo.Oracle(case)
    o.set_state(*case["state"])
    hc = o.geometry("hc")[:-1]
    rho0 = case["state"][0]
    o.set_scalar(3.7 * rho0)
    for _ in range(3):
        o.step(case["dt"], case["ns"])
    rho = o.get_state()[0]
    assert np.abs(rho - rho0).max() > 1e-9 * rho0.max()           # the density did change
    phi = o.get_scalar() / rho
    assert np.abs(phi - 3.7).max() < 2e-13 * 3.7, np.abs(phi - 3.7).max()
    # conservation of a structured scalar
    rng = np.random.default_rng(5)
    q0 = rho0 * (1.0 + 0.3 * rng.random(rho0.shape))
    o2 = erfo.Oracle(case)
    o2.set_state(*case["state"])
    o2.set_scalar(q0)
    for _ in range(3):
        o2.step(case["dt"], case["ns"])
    q1 = o2.get_scalar()
    assert np.abs(q1 - q0).max() > 1e-6
    assert abs(_fsum((q1 - q0) * hc)) < 3e-15 * _fsum(q0 * hc)


def test_scalar_without_substepping_uses_the_stage_momenta():
    """L140 mode (no substepping): constant phi still stays constant (momenta = the stage momenta)."""
    case = wl.make_case(2, nx=10, ny=8, nz=10, params=dict(substep_mode=0))
    o = erfo.Oracle(case)
    o.set_state(*case["state"])
    o.set_scalar(2.5 * case["state"][0])
    for _ in range(2):
        o.step(0.02, 6)
    phi = o.get_scalar() / o.get_state()[0]
    assert np.abs(phi - 2.5).max() < 1e-13 * 2.5


@pytest.mark.parametrize("axis", ["x", "y", "z"])
def test_scalar_pure_diffusion_rk3_polynomial(axis):
    """State at rest in balance (f(S) = 0 exactly), constant K = rho alpha: the scalar obeys
    dQ/dt = -alpha khat^2 Q' per mode, and Eq. 11-13 applied to it (every stage restarts from Q^n) multiply the
    mode by 1 + z + z^2/2 + z^3/6, z = -alpha khat^2 dt."""
    nx, ny, nz, dx, dy, dz = 16, 12, 10, 40.0, 25.0, 15.0
    alpha = 400.0
    case = uniform_case(nx, ny, nz, dx, dy, dz, diffusion=1, nu=0.0, alpha_theta=alpha)
    st = zeros_state(case)
    st[0][:] = 1.0
    st[4][:] = 300.0
    H = nz * dz
    k = dict(x=2 * np.pi / (nx * dx), y=2 * np.pi * 2 / (ny * dy), z=3 * np.pi / H)[axis]
    h = dict(x=dx, y=dy, z=dz)[axis]
    xc = ((np.arange(nx) + 0.5) * dx)[None, None, :]
    yc = ((np.arange(ny) + 0.5) * dy)[None, :, None]
    zc = ((np.arange(nz) + 0.5) * dz)[:, None, None]
    mode = dict(x=np.sin(k * xc), y=np.sin(k * yc), z=np.cos(k * zc))[axis] * np.ones((nz, ny, nx))
    o = erfo.Oracle(case)
    o.set_state(*st)
    o.set_scalar(2.0 + 0.5 * mode)
    dt = 1.5
    o.step(dt, 4)
    z = -alpha * ((2.0 / h) * np.sin(0.5 * k * h)) ** 2 * dt
    amp = 1 + z + z * z / 2 + z ** 3 / 6
    assert abs(z) > 0.05
    got = o.get_scalar()
    assert np.array_equal(o.get_state()[0], st[0])                # the flow really stayed at rest
    assert np.abs(got - (2.0 + 0.5 * amp * mode)).max() < 1e-13


def _weights(order):
    """Face weights of Eq. 17-21 for positive flux, from the golden table (the paper's printed stencils)."""
    path = os.path.join(os.path.dirname(__file__), "golden", "stencil_weights.txt")
    for line in open(path):
        t = line.split()
        if t and not line.startswith("#") and t[0] == str(order) and t[1] in ("0", "1"):   # centred, or sgn = +1
            return np.array([float(x) for x in t[3:9]]) / float(t[2])
    raise AssertionError(f"no weights for order {order} in {path}")


@pytest.mark.parametrize("order", [2, 3, 5, 6])
@pytest.mark.parametrize("direction", ["x", "y"])
def test_scalar_linear_advection_symbol(order, direction):
    """Uniform flow, uniform rho and theta, g = 0: f(S) = 0, the flow stays uniform and the scalar is linearly
    advected.  One RK3 step multiplies the Fourier mode exp(i k x) by P(z) = 1 + z + z^2/2 + z^3/6 with
    z = -c (1 - exp(-i k h)) sum_n w_n exp(i k h (n - 2)) -- the symbol of the flux difference built from the
    paper's printed face weights w (tests/golden/stencil_weights.txt), c = u dt / h."""
    n, h = 24, 100.0
    dims = dict(x=2, y=2, z=3)
    dims[direction] = n
    case = uniform_case(dims["x"], dims["y"], dims["z"], h, h, h, adv_order_h=order, adv_order_v=order)
    st = zeros_state(case)
    st[0][:] = 1.0
    st[4][:] = 300.0
    u0 = 12.0
    st[1 if direction == "x" else 2][:] = u0
    nz, ny, nx = st[0].shape
    kk, jj, ii = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    m = {"x": ii, "y": jj}[direction]
    kw = 2 * np.pi * 3 / (n * h)
    xcen = (m + 0.5) * h
    o = erfo.Oracle(case)
    o.set_state(*st)
    o.set_scalar(1.0 + 0.25 * np.cos(kw * xcen))
    dt = 2.0
    o.step(dt, 4)
    for a, b in zip(o.get_state(), st):
        assert np.abs(a - b).max() < 1e-12 * max(np.abs(b).max(), 1.0)     # uniform flow stays uniform
    w = _weights(order)          # q_{m-3} .. q_{m+2} -> value at the face between q_{m-1} and q_m
    th = kw * h
    # face value at the LEFT face of cell m for mode exp(i k x_m): sum_n w_n exp(i th (n - 3))
    face = sum(w[nn] * np.exp(1j * th * (nn - 3)) for nn in range(6))
    z = -(u0 * dt / h) * (np.exp(1j * th) - 1.0) * face     # -(F_{m+1} - F_m)/h * dt
    P = 1 + z + z * z / 2 + z ** 3 / 6
    expect = 1.0 + 0.25 * np.real(P * np.exp(1j * kw * xcen))
    assert np.abs(o.get_scalar() - expect).max() < 2e-13
