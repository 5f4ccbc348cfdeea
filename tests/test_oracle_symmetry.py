"""Symmetry pins of the oracle's discretisation D0.

Most of D0's two- and four-point means and metric factors are readings ([R]): no number in the paper fixes them.  The
mathematics does: on a laterally periodic grid the discrete operators must commute with the reflections x -> -x and
y -> -y, with the exchange of x and y, and -- on a flat, uniformly spaced column between two rigid lids -- with z -> -z
together with g -> -g.  A one-sided replacement of a mean (own cell instead of the face average, level k instead of the
mean of k-1 and k, hx where hy belongs) breaks one of them.  Each test builds the transformed problem from the same
arrays (fields, node heights, base state), runs the oracle on both, and requires the results to be the transformed
images of one another to round-off.

How the staggered fields transform (L178: rho*u on low-x faces, rho*v on low-y faces, rho*w on low-z faces):
  x-reflection:  cell fields, V, W: i -> nx-1-i;   U(i) -> -U((nx-i) mod nx);   nodes: i -> nx-i
  exchange:      every array transposed in (y, x); U <-> V; dx <-> dy
  z-reflection:  cell fields, U, V: k -> nz-1-k;   W(k) -> -W(nz-k);   g -> -g;   base state reversed
Seeded states with non-uniform rho, theta and all three momenta; 3rd-, 5th- and 6th-order stencils (upwind parts flip with
the velocity); Smagorinsky diffusion; flat stretched levels, and config 4's levels over a smooth periodic terrain that has no symmetry of its own."""
import numpy as np
import pytest

from paper_2412_04395_b200 import workloads as wl

TOL = 2e-12  # of the field's maximum: sums are formed in another order on the image, nothing else differs


# ------------------------------------------------------------------ the three maps (involutions on arrays)
def _mx_cell(a):
    return a[..., ::-1]


def _mx_face(a):  # U on low-x faces
    return -np.roll(a[..., ::-1], 1, axis=-1)


def _my_cell(a):
    return a[..., ::-1, :]


def _my_face(a):
    return -np.roll(a[..., ::-1, :], 1, axis=-2)


def _t(a):
    return np.swapaxes(a, -1, -2)


def _mz_cell(a):
    return a[::-1]


def _mz_face(a):  # W on low-z faces, nz+1 levels
    return -a[::-1]


def map_fields(F, kind):
    """Image of a list (rho, U, V, W, Theta)-like (state, tendencies or perturbation)."""
    r, U, V, W, T = F
    if kind == "x":
        out = [_mx_cell(r), _mx_face(U), _mx_cell(V), _mx_cell(W), _mx_cell(T)]
    elif kind == "y":
        out = [_my_cell(r), _my_cell(U), _my_face(V), _my_cell(W), _my_cell(T)]
    elif kind == "xy":
        out = [_t(r), _t(V), _t(U), _t(W), _t(T)]
    else:
        out = [_mz_cell(r), _mz_cell(U), _mz_cell(V), _mz_face(W), _mz_cell(T)]
    return [np.ascontiguousarray(a) for a in out]


def map_case(case, kind):
    c = dict(case)
    c["params"] = dict(case["params"])
    cell = {"x": _mx_cell, "y": _my_cell, "xy": _t, "z": _mz_cell}[kind]
    if kind == "xy":
        c["nx"], c["ny"], c["dx"], c["dy"] = case["ny"], case["nx"], case["dy"], case["dx"]
    if case.get("z_nodes") is not None:
        zn = case["z_nodes"]
        assert kind != "z"
        c["z_nodes"] = np.ascontiguousarray({"x": zn[..., ::-1], "y": zn[..., ::-1, :], "xy": _t(zn)}[kind])
    elif kind == "z":
        zl = case["z_levels"]
        c["z_levels"] = np.ascontiguousarray(zl[-1] - zl[::-1])
        c["params"]["g"] = -case["params"]["g"]
    for key in ("rho0", "rhotheta0"):
        a = case[key]
        c[key] = np.ascontiguousarray(a[::-1] if (a.ndim == 1 and kind == "z") else a if a.ndim == 1 else cell(a))
    return c


# ------------------------------------------------------------------ problems
def _problem(terrain, order, seed, diffusion=2):
    if terrain:
        # config 4's levels, base-state recipe and parameters over a smooth periodic terrain with no symmetry of its own
        # (slopes up to about 0.25 in x and y): z = zeta + h(x, y) (1 - zeta / z_top), L180
        case = wl.make_case(4, nx=12, ny=10, nz=14, params=dict(adv_order_h=order, adv_order_v=order, diffusion=diffusion))
        nx, ny, zl = case["nx"], case["ny"], case["z_nodes"][:, 0, 0].copy()
        zl -= zl[0]
        x = 2.0 * np.pi * np.arange(nx + 1)[None, :] / nx
        y = 2.0 * np.pi * np.arange(ny + 1)[:, None] / ny
        h = 40.0 * (1.0 + 0.5 * np.sin(x + 0.7) * np.cos(y + 0.3) + 0.3 * np.sin(2.0 * x + 1.1) + 0.2 * np.cos(y - 0.4))
        h[:, -1], h[-1, :] = h[:, 0], h[0, :]  # the periodic closure, exactly
        case["z_nodes"] = zl[:, None, None] + h[None] * (1.0 - zl[:, None, None] / zl[-1])
        theta0, rho0 = wl.hydrostatic_base(wl.cell_centre_heights(case["z_nodes"]), wl.CONFIGS[4]["layers"])
        case["rho0"], case["rhotheta0"] = rho0, rho0 * theta0
    else:
        case = wl.make_case(5, nx=12, ny=10, nz=14, params=dict(adv_order_h=order, adv_order_v=order, diffusion=diffusion))
        dz = np.diff(case["z_levels"])[0] * 1.07 ** np.arange(case["nz"])
        case["z_levels"] = np.concatenate([[0.0], np.cumsum(dz)])
    return case, _state(case, seed)


def _state(case, seed):
    nz, ny, nx = case["nz"], case["ny"], case["nx"]
    rng = np.random.default_rng(seed)
    r0 = case["rho0"] if case["rho0"].ndim == 3 else np.broadcast_to(case["rho0"][:, None, None], (nz, ny, nx))
    t0 = case["rhotheta0"] if case["rhotheta0"].ndim == 3 else np.broadcast_to(case["rhotheta0"][:, None, None], (nz, ny, nx))
    rho = r0 * (1.0 + 0.02 * rng.standard_normal((nz, ny, nx)))
    Th = t0 * (1.0 + 0.003 * rng.standard_normal((nz, ny, nx)))
    U = rho * (3.0 + 4.0 * rng.standard_normal((nz, ny, nx)))
    V = rho * (-2.0 + 4.0 * rng.standard_normal((nz, ny, nx)))
    W = np.zeros((nz + 1, ny, nx))
    W[1:-1] = 2.0 * rng.standard_normal((nz - 1, ny, nx))
    return [rho, U, V, W, Th]


def _uniform_column_problem(order, seed):
    """Flat, uniformly spaced levels, uniform base state (so that the reversed base state is the same physical column)."""
    case = wl.make_case(5, nx=10, ny=8, nz=12, params=dict(adv_order_h=order, adv_order_v=order, diffusion=2))
    nz = case["nz"]
    case["rho0"] = np.full(nz, 1.1)
    case["rhotheta0"] = np.full(nz, 1.1 * 295.0)
    return case, _state(case, seed)


def _close(a, b, what):
    scale = max(np.abs(b).max(), 1e-300)
    err = np.abs(a - b).max() / scale
    assert err <= TOL, (what, err)


CASES = [(False, 3), (False, 5), (False, 6), (False, 2), (True, 3), (True, 5), (True, 4)]


@pytest.mark.parametrize("kind", ["x", "y", "xy"])
@pytest.mark.parametrize("terrain,order", CASES)
def test_reflections_and_exchange_commute_with_every_operator(oracle_lib, terrain, order, kind):
    erfo = oracle_lib
    case, st = _problem(terrain, order, seed=40 + order)
    imcase, imst = map_case(case, kind), map_fields(st, kind)
    P0 = [0.01 * a for a in _state(case, seed=77)]  # a perturbation S'' of the same shape (scaled state-like noise)
    P0[3][0] = P0[3][-1] = 0.0
    res = []
    for c, s, P in ((case, st, P0), (imcase, imst, map_fields(P0, kind))):
        o = erfo.Oracle(c)
        o.set_state(*s)
        R = o.slow_rhs()
        A = o.acoustic(c["dt"] / c["ns"], 2, R, P)
        o.step(c["dt"], c["ns"])
        res.append((R, A, o.get_state()))
        o.close()
    names = ("rho", "U", "V", "W", "Theta")
    for what, a, b in zip(("slow_rhs", "acoustic", "rk3_step"), res[1], [map_fields(x, kind) for x in res[0]]):
        for n, x, y in zip(names, a, b):
            _close(x, y, (what, n, kind, terrain, order))


@pytest.mark.parametrize("order", [2, 3, 5, 6])
def test_vertical_reflection_with_reversed_gravity_on_a_uniform_column(oracle_lib, order):
    erfo = oracle_lib
    case, st = _uniform_column_problem(order, seed=60 + order)
    imcase, imst = map_case(case, "z"), map_fields(st, "z")
    P0 = [0.01 * a for a in _state(case, seed=78)]
    P0[3][0] = P0[3][-1] = 0.0
    res = []
    for c, s, P in ((case, st, P0), (imcase, imst, map_fields(P0, "z"))):
        o = erfo.Oracle(c)
        o.set_state(*s)
        R = o.slow_rhs()
        A = o.acoustic(c["dt"] / c["ns"], 2, R, P)
        o.step(c["dt"], c["ns"])
        res.append((R, A, o.get_state()))
        o.close()
    names = ("rho", "U", "V", "W", "Theta")
    for what, a, b in zip(("slow_rhs", "acoustic", "rk3_step"), res[1], [map_fields(x, "z") for x in res[0]]):
        for n, x, y in zip(names, a, b):
            _close(x, y, (what, n, order))


def test_the_maps_are_involutions_and_the_state_is_not_symmetric():
    """Guards the test itself: applying a map twice is the identity, and the seeded state is far from its own image (a
    symmetric state would make every assertion above empty)."""
    case, st = _problem(True, 5, seed=45)
    for kind in ("x", "y", "xy"):
        back = map_fields(map_fields(st, kind), kind)
        assert all(np.array_equal(a, b) for a, b in zip(st, back))
        assert np.array_equal(map_case(map_case(case, kind), kind)["z_nodes"], case["z_nodes"])
    im = map_fields(st, "x")
    assert np.abs(im[1] - st[1]).max() > 1.0 and np.abs(im[0] - st[0]).max() > 1e-3
    zn = case["z_nodes"]
    assert np.abs(zn[0, :, ::-1] - zn[0]).max() > 10.0 and np.abs(zn[0, ::-1, :] - zn[0]).max() > 10.0  # no symmetry of its own
    case, st = _uniform_column_problem(5, seed=65)
    back = map_fields(map_fields(st, "z"), "z")
    assert all(np.array_equal(a, b) for a, b in zip(st, back))
