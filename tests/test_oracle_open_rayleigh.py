"""Pins of the oracle's open lateral boundary ("periodic, inflow, outflow, or open"; reading G27:
ghost = nearest interior value) and of the Rayleigh damping layer (L219; Appendix C: sine-squared ramp of an
inverse time scale from 0 at the bottom of the layer to the stated value at the top; Table C1: damped fields; reading
G28).  Each expected value below is written from the paper's sentence or from the telescoping of the flux form, not
from the oracle's code."""
import numpy as np
import pytest

from oracle import erfo
from paper_2412_04395_b200 import workloads as wl
from util import base_state_fields, uniform_case


@pytest.fixture(scope="module", autouse=True)
def _build():
    erfo.build()


def _state(case, u=0.0, v=0.0, dtheta=None, rng=None, noise=0.0):
    r0, t0 = base_state_fields(case)
    nz, ny, nx = r0.shape
    th = t0 / r0 + (dtheta if dtheta is not None else 0.0)
    U = r0 * u
    V = r0 * v
    if rng is not None and noise:
        U = U + noise * rng.standard_normal(r0.shape)
        V = V + noise * rng.standard_normal(r0.shape)
    return [r0.copy(), U, V, np.zeros((nz + 1, ny, nx)), r0 * th]


# ------------------------------------------------------------------ open lateral boundaries
@pytest.mark.parametrize("per", [(0, 1), (1, 0), (0, 0)])
@pytest.mark.parametrize("order", [2, 3, 5, 6])
def test_uniform_flow_is_steady_through_open_boundaries(per, order):
    """A uniform wind over a flat grid has no gradient anywhere, so a zero-gradient boundary changes nothing: f(S) = 0
    in every cell, boundary cells included, and the state does not move."""
    case = uniform_case(12, 9, 6, 100.0, 80.0, 50.0, adv_order_h=order, adv_order_v=order, diffusion=1, nu=2.0,
                        alpha_theta=2.0)
    case["periodic_x"], case["periodic_y"] = per
    st = _state(case, u=7.0, v=-3.0)
    o = erfo.Oracle(case)
    o.set_state(*st)
    R = o.slow_rhs()
    for f, r in enumerate(R):
        assert np.abs(r).max() <= 1e-12, (f, np.abs(r).max())
    for _ in range(3):
        o.step(0.5, 4)
    out = o.get_state()
    for a, b in zip(out, st):
        assert np.abs(a - b).max() <= 1e-11 * max(np.abs(b).max(), 1.0)


def test_mass_budget_of_an_open_domain_is_the_boundary_flux():
    """Flux form (Eq. 1): the x-differences of rho u telescope, so the total mass tendency is the flux through the
    first face minus the flux through the face beyond the last cell -- which under G27 is the copy of the last stored
    face.  (On a periodic domain the same sum is zero: this test tells the two closures apart.)"""
    rng = np.random.default_rng(5)
    case = uniform_case(10, 7, 5, 100.0, 100.0, 40.0, adv_order_h=2, adv_order_v=2)
    st = _state(case, u=5.0, v=1.0, rng=rng, noise=0.5)
    dz, dx, dy = 40.0, case["dx"], case["dy"]
    got = {}
    for per in ((1, 1), (0, 1), (1, 0)):
        case["periodic_x"], case["periodic_y"] = per
        o = erfo.Oracle(case)
        o.set_state(*st)
        got[per] = float(np.sum(o.slow_rhs()[0]) * dx * dy * dz)
    U, V = st[1], st[2]
    assert abs(got[(1, 1)]) <= 1e-9
    exp_x = -float(np.sum(U[:, :, -1] - U[:, :, 0])) * dy * dz
    exp_y = -float(np.sum(V[:, -1, :] - V[:, 0, :])) * dx * dz
    assert abs(exp_x) > 1.0 and abs(exp_y) > 1.0
    assert got[(0, 1)] == pytest.approx(exp_x, rel=1e-11)
    assert got[(1, 0)] == pytest.approx(exp_y, rel=1e-11)


def test_a_warm_blob_leaves_through_the_open_boundary_and_does_not_come_back():
    """Open = what reaches the boundary leaves.  A theta anomaly carried by a uniform wind crosses the downstream
    boundary; afterwards the domain holds (almost) none of it, while the periodic closure of the same problem still
    holds all of it (it re-enters upstream)."""
    nx, dx, u0 = 48, 100.0, 20.0
    case = uniform_case(nx, 2, 6, dx, dx, 100.0, adv_order_h=5, adv_order_v=5)
    x = (np.arange(nx) + 0.5) * dx
    bump = 0.5 * np.exp(-((x - 0.75 * nx * dx) / (3 * dx)) ** 2)[None, None, :] * np.ones((6, 2, 1))
    st = _state(case, u=u0, dtheta=bump)
    r0, t0 = base_state_fields(case)
    steps = int(round((0.25 * nx * dx + 14 * dx) / u0))  # dt = 1 s: centre 14 cells beyond the boundary
    left = {}
    for per in (1, 0):
        case["periodic_x"] = per
        o = erfo.Oracle(case)
        o.set_state(*st)
        for _ in range(steps):
            o.step(1.0, 6)
        rho, _, _, _, Th = o.get_state()
        assert np.isfinite(Th).all()
        left[per] = float(np.abs(Th / rho - t0 / r0).max())
    assert left[1] > 0.35          # periodic: the blob is still there (5th-order upwind damps it a little)
    assert left[0] < 0.02          # open: gone, up to the weak reflection of a zero-gradient boundary


# ------------------------------------------------------------------ Rayleigh damping layer
def _tau_paper(z, ztop, depth, coef):
    """L622 as a sentence: sine squared, 0 at the bottom of the layer, `coef` at the top."""
    zb = ztop - depth
    return np.where(z > zb, coef * np.sin(0.5 * np.pi * (z - zb) / depth) ** 2, 0.0)


def test_rayleigh_profile_and_tendencies():
    """f(S) with the layer minus f(S) without it, on the same state, is -tau(z) * (variable - reference) for the
    masked fields and exactly 0 for the others; tau is the paper's sine-squared ramp at the height of each point."""
    rng = np.random.default_rng(11)
    case = wl.make_case(3, nx=6, ny=5, nz=24)
    nz, ny, nx = 24, 5, 6
    zl = case["z_levels"]
    ztop, depth, coef, uref, vref = zl[-1], 90.0, 0.2, 10.0, -2.0
    st = [a.copy() for a in case["state"]]
    st[3][1:-1] = 0.3 * rng.standard_normal((nz - 1, ny, nx))
    st[2] += 0.5 * rng.standard_normal(st[2].shape)
    o = erfo.Oracle(case)
    o.set_state(*st)
    base = o.slow_rhs()
    for mask in (1, 2, 4, 8, 15):
        c2 = dict(case)
        c2["params"] = dict(case["params"], ray_depth=depth, ray_coef=coef, ray_fields=mask, ray_uref=uref,
                            ray_vref=vref)
        o2 = erfo.Oracle(c2)
        o2.set_state(*st)
        d = [a - b for a, b in zip(o2.slow_rhs(), base)]
        zc = 0.5 * (zl[:-1] + zl[1:])
        tc = _tau_paper(zc, ztop, depth, coef)[:, None, None]
        tw = _tau_paper(zl, ztop, depth, coef)[:, None, None]
        rho, U, V, W, Th = st
        r0, t0 = base_state_fields(case)
        exp = [np.zeros_like(a) for a in d]
        if mask & 1:
            exp[1] = -tc * (U - 0.5 * (rho + np.roll(rho, 1, axis=2)) * uref)
        if mask & 2:
            exp[2] = -tc * (V - 0.5 * (rho + np.roll(rho, 1, axis=1)) * vref)
        if mask & 4:
            exp[3] = -tw * W
            exp[3][0] = exp[3][-1] = 0.0
        if mask & 8:
            exp[4] = -tc * (Th - rho * t0 / r0)
        for f in range(5):
            scale = max(np.abs(exp[f]).max(), np.abs(base[f]).max(), 1e-30)
            assert np.abs(d[f] - exp[f]).max() <= 1e-12 * scale, (mask, f)
        assert tc.max() > 0.9 * coef * np.sin(0.5 * np.pi * (depth - 5.0) / depth) ** 2  # the layer is resolved
        assert (tc[zc <= ztop - depth] == 0).all()


def test_rayleigh_layer_damps_w_at_the_stated_rate():
    """A horizontally varying w' on one face inside the layer, one RK3 step without substepping, with the layer and
    without it (same state, so the acoustic response of the step is common to both): the ratio of the two results is
    the RK3 polynomial of z = -tau dt (Eq. 11-13 applied to dW/dt = -tau W), cross terms being O(z (c k dt)^2)."""
    case = uniform_case(8, 8, 20, 200.0, 200.0, 50.0, adv_order_h=2, adv_order_v=2)
    case["params"].update(substep_mode=0)
    nz, ny, nx = 20, 8, 8
    st = _state(case)
    x = np.arange(nx)
    k = 16                                          # a face inside the layer: z = 800 m, layer 600..1000 m
    st[3][k] = 1e-6 * np.cos(2 * np.pi * x / nx)[None, :] * np.ones((ny, 1))
    dt = 1e-3
    W = {}
    for on in (0, 1):
        c2 = dict(case)
        c2["params"] = dict(case["params"], ray_depth=400.0, ray_coef=0.5, ray_fields=4 * on)
        o = erfo.Oracle(c2)
        o.set_state(*st)
        o.step(dt, 2)
        W[on] = o.get_state()[3]
    tau = float(_tau_paper(np.array([800.0]), 1000.0, 400.0, 0.5)[0])
    assert tau == pytest.approx(0.25)               # half-way up the ramp: sin^2(pi/4) = 1/2 of 0.5
    z = -tau * dt
    assert W[1][k, 0, 0] / W[0][k, 0, 0] == pytest.approx(1 + z + z * z / 2 + z ** 3 / 6, rel=1e-7)
    assert abs(W[1][k, 0, 0] / W[0][k, 0, 0] - 1.0) > 1e-4
    assert np.array_equal(W[1][10], W[0][10])       # below the layer nothing is damped


# ------------------------------------------------------------------ inflow (reading G30: a Dirichlet column of cells)
def test_inflow_column_is_held_and_feeds_the_domain():
    """periodic_x = 2: the first column of cells keeps the values it was given, exactly, whatever happens inside; what
    it holds is carried into the domain by the wind.  A column 1 K warmer than the rest at a 20 m/s inflow: after 60 s
    the warm air has reached x = u t = 1200 m (cell 12) -- warm well behind the front, untouched well ahead of it.  With
    the open closure (periodic_x = 0) nothing holds the boundary column: its value floats with the flow."""
    nx, dx, u0 = 48, 100.0, 20.0
    case = uniform_case(nx, 3, 6, dx, dx, 100.0, adv_order_h=3, adv_order_v=3)
    dth = np.zeros((6, 3, nx))
    dth[:, :, 0] = 1.0
    st = _state(case, u=u0, dtheta=dth)
    r0, t0 = base_state_fields(case)
    res = {}
    for code in (2, 0):
        case["periodic_x"] = code
        o = erfo.Oracle(case)
        o.set_state(*st)
        for _ in range(60):
            o.step(1.0, 6)
        got = o.get_state()
        res[code] = got[4] / got[0] - t0 / r0
        if code == 2:
            for f in range(5):
                assert np.array_equal(got[f][..., 0], st[f][..., 0]), f     # the Dirichlet column, bitwise
    th = res[2][2, 1]
    assert th[1:7].min() > 0.9 and th[1:7].max() < 1.1        # behind the front: the inflow value
    assert abs(th[12] - 0.5) < 0.35                           # the front is where u t says
    assert np.abs(th[24:]).max() < 1e-3                       # ahead of it: nothing yet
    assert abs(res[0][2, 1][0] - 1.0) > 0.05                  # open closure: the boundary value is not held, it floats


@pytest.mark.parametrize("code", [(2, 1), (1, 2), (2, 2), (2, 0)])
def test_uniform_flow_is_steady_with_inflow(code):
    case = uniform_case(12, 9, 6, 100.0, 80.0, 50.0, adv_order_h=5, adv_order_v=5, diffusion=1, nu=2.0, alpha_theta=2.0)
    case["periodic_x"], case["periodic_y"] = code
    st = _state(case, u=7.0, v=3.0)
    o = erfo.Oracle(case)
    o.set_state(*st)
    for _ in range(3):
        o.step(0.5, 4)
    for a, b in zip(o.get_state(), st):
        assert np.abs(a - b).max() <= 1e-11 * max(np.abs(b).max(), 1.0)
