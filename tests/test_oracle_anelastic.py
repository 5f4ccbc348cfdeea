"""Pins of the oracle's anelastic mode (Sec. 2.2 Eq. 8; Sec. 3.2 Eq. 14-16): RK2 with a
projection after each stage, buoyancy rho0 (theta - theta0)/theta0 g, p' from the Poisson equation only.  Expected values
come from the paper's equations written out densely in numpy (brute force on tiny grids), from closed forms, or from
invariants -- never from the oracle's own routines."""
import numpy as np
import pytest

from oracle import erfo
from paper_2412_04395_b200 import workloads as wl
from util import base_state_fields, uniform_case


@pytest.fixture(scope="module", autouse=True)
def _build():
    erfo.build()


def _stretched(case, ratio=1.15):
    nz = case["nz"]
    dz = 40.0 * ratio ** np.arange(nz)
    case["z_levels"] = np.concatenate([[0.0], np.cumsum(dz)])
    return case


def _random_momenta(case, rng, amp=1.0):
    r0, t0 = base_state_fields(case)
    nz, ny, nx = r0.shape
    W = amp * rng.standard_normal((nz + 1, ny, nx))
    W[0] = W[-1] = 0.0
    return [r0.copy(), amp * rng.standard_normal(r0.shape), amp * rng.standard_normal(r0.shape), W, t0.copy()]


def _dense_operators(case):
    """Eq. 16's two operators from their definitions, as dense matrices: D (divergence of face momenta at cell
    centres, rigid lids) and G (gradient of a cell-centred psi at the U, V and interior W faces)."""
    nx, ny, nz, dx, dy = case["nx"], case["ny"], case["nz"], case["dx"], case["dy"]
    zl = case["z_levels"]
    dz = np.diff(zl)
    zc = 0.5 * (zl[:-1] + zl[1:])
    N = nx * ny * nz
    nW = nx * ny * (nz - 1)

    def c(i, j, k):
        return (k * ny + j % ny) * nx + i % nx

    def w(i, j, k):  # interior w-face k = 1..nz-1
        return 2 * N + ((k - 1) * ny + j) * nx + i

    D = np.zeros((N, 2 * N + nW))
    G = np.zeros((2 * N + nW, N))
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                r = c(i, j, k)
                D[r, c(i + 1, j, k)] += 1 / dx
                D[r, c(i, j, k)] -= 1 / dx
                D[r, N + c(i, j + 1, k)] += 1 / dy
                D[r, N + c(i, j, k)] -= 1 / dy
                if k + 1 <= nz - 1:
                    D[r, w(i, j, k + 1)] += 1 / dz[k]
                if k >= 1:
                    D[r, w(i, j, k)] -= 1 / dz[k]
                G[c(i, j, k), c(i, j, k)] += 1 / dx
                G[c(i, j, k), c(i - 1, j, k)] -= 1 / dx
                G[N + c(i, j, k), c(i, j, k)] += 1 / dy
                G[N + c(i, j, k), c(i, j - 1, k)] -= 1 / dy
                if k >= 1:
                    hw = zc[k] - zc[k - 1]
                    G[w(i, j, k), c(i, j, k)] += 1 / hw
                    G[w(i, j, k), c(i, j, k - 1)] -= 1 / hw
    return D, G


def _pack(st):
    return np.concatenate([st[1].ravel(), st[2].ravel(), st[3][1:-1].ravel()])


def test_projection_against_a_dense_solve_of_eq16():
    """Brute force on a 4 x 3 x 5 stretched grid: dt D G psi = D M, M* = M - dt G psi, solved densely (least squares:
    the constants are the null space).  The projected momenta are unique; psi is unique up to a constant."""
    rng = np.random.default_rng(3)
    case = _stretched(uniform_case(4, 3, 5, 70.0, 110.0, 1.0))
    st = _random_momenta(case, rng)
    dt = 0.7
    D, G = _dense_operators(case)
    M = _pack(st)
    psi = np.linalg.lstsq(dt * D @ G, D @ M, rcond=None)[0]
    Mstar = M - dt * G @ psi
    assert np.abs(D @ Mstar).max() <= 1e-12
    o = erfo.Oracle(case)
    o.set_state(*st)
    o.project(dt)
    got = o.get_state()
    assert np.abs(_pack(got) - Mstar).max() <= 1e-11 * np.abs(M).max()
    assert np.abs(Mstar - M).max() > 0.1          # the projection did something
    pp = o.pprime().ravel()
    assert np.abs((pp - pp.mean()) - (psi - psi.mean())).max() <= 1e-10 * np.abs(psi - psi.mean()).max()
    assert np.array_equal(got[0], st[0]) and np.array_equal(got[4], st[4])  # rho, Theta untouched


@pytest.mark.parametrize("shape", [(12, 10, 9), (16, 5, 14), (7, 9, 6)])
def test_projection_gives_a_divergence_free_field_and_is_idempotent(shape):
    """Eq. 8: after the projection div(rho0 u) = 0 in every cell to round-off; projecting again changes nothing."""
    nx, ny, nz = shape
    rng = np.random.default_rng(nx)
    case = _stretched(uniform_case(nx, ny, nz, 50.0, 80.0, 1.0))
    st = _random_momenta(case, rng)
    o = erfo.Oracle(case)
    o.set_state(*st)
    d0 = np.abs(o.divergence()).max()
    o.project(0.3)
    a = o.get_state()
    assert np.abs(o.divergence()).max() <= 1e-12 * d0
    o.project(0.3)
    b = o.get_state()
    for f in (1, 2, 3):
        assert np.abs(a[f] - b[f]).max() <= 1e-12
    assert np.all(b[3][0] == 0.0) and np.all(b[3][-1] == 0.0)  # rigid lids


def test_rest_state_stays_at_rest():
    case = wl.make_case(3, nx=8, ny=6, nz=20)
    r0, t0 = base_state_fields(case)
    z = np.zeros_like(r0)
    st = [r0.copy(), z, z.copy(), np.zeros((21, 6, 8)), t0.copy()]
    o = erfo.Oracle(case)
    o.set_state(*st)
    for _ in range(3):
        o.anelastic_step(0.5)
    for a, b in zip(o.get_state(), st):
        assert np.array_equal(a, b)
    assert np.all(o.pprime() == 0.0)


def test_horizontally_uniform_buoyancy_is_balanced_by_the_pressure_not_by_motion():
    """A warm LAYER (no horizontal structure) cannot move a fluid between rigid lids: the projection must return
    W = 0 exactly and put the force into p'.  Discretely: after the first projection grad_z psi = g B_face (B = rho0
    (theta - theta0)/theta0, L96).  With p' += psi after EACH of the two projections, as printed (L160), the lagged p'
    after one step is 3/2 of that balance, and approaches it like (-1/2)^n over the following steps."""
    case = _stretched(uniform_case(6, 5, 12, 100.0, 100.0, 1.0, g=9.81, rho0=1.1), ratio=1.08)
    r0, t0 = base_state_fields(case)
    nz = 12
    th0 = t0 / r0
    dth = np.zeros(nz)
    dth[3:7] = [0.5, 1.5, 1.0, 0.25]
    th = th0 + dth[:, None, None]
    st = [r0.copy(), np.zeros_like(r0), np.zeros_like(r0), np.zeros((nz + 1, 5, 6)), r0 * th]
    zl = case["z_levels"]
    zc = 0.5 * (zl[:-1] + zl[1:])
    hw = zc[1:] - zc[:-1]
    B = 1.1 * dth / 300.0
    balance = 9.81 * 0.5 * (B[1:] + B[:-1])          # g B at the interior w-faces
    o = erfo.Oracle(case)
    o.set_state(*st)
    fac = 0.0
    for n in range(1, 13):
        o.anelastic_step(2.0)
        got = o.get_state()
        for f in (1, 2, 3):
            assert np.abs(got[f]).max() <= 1e-12
        assert np.array_equal(got[4], st[4])
        pp = o.pprime()
        grad = (pp[1:, 2, 3] - pp[:-1, 2, 3]) / hw
        fac = 1.0 - (-0.5) ** n                      # 3/2, 3/4, 9/8, ...
        assert np.abs(grad - fac * balance).max() <= 1e-11 * np.abs(balance).max(), n
        assert np.abs(pp - pp[:, :1, :1]).max() <= 1e-10 * np.abs(pp).max()   # no horizontal structure
    assert abs(fac - 1.0) < 3e-4


def test_rk2_polynomial():
    """Eq. 14-15 on dTheta'/dt = -tau Theta' (a theta-only Rayleigh layer spanning the whole depth, no gravity, no
    wind: nothing else acts): one step multiplies theta' by 1 + z + z^2/2, z = -tau(z_k) dt, level by level."""
    case = uniform_case(5, 4, 10, 100.0, 100.0, 50.0)
    case["params"].update(ray_depth=500.0, ray_coef=0.4, ray_fields=8)
    r0, t0 = base_state_fields(case)
    rng = np.random.default_rng(2)
    thp = 0.3 * rng.standard_normal(r0.shape)
    st = [r0.copy(), np.zeros_like(r0), np.zeros_like(r0), np.zeros((11, 4, 5)), t0 + r0 * thp]
    o = erfo.Oracle(case)
    o.set_state(*st)
    dt = 0.8
    o.anelastic_step(dt)
    got = o.get_state()[4]
    zc = (np.arange(10) + 0.5) * 50.0
    z = -0.4 * np.sin(0.5 * np.pi * zc / 500.0) ** 2 * dt
    amp = (1 + z + z * z / 2)[:, None, None]
    assert np.abs((got - t0) - amp * (r0 * thp)).max() <= 1e-12
    assert np.abs(z).max() > 0.2                     # the quadratic term matters: RK2, not forward Euler


def test_warm_bubble_rises_with_the_constraint_and_the_invariants_held():
    """A warm bubble (L96 buoyancy) in a neutral atmosphere: it accelerates upward, div(rho0 u) stays 0 after every
    step, rho stays rho0 (L94), and the flux-form theta equation conserves sum(rho0 theta dz)."""
    case = wl.make_case(1, nx=16, ny=4, nz=16, params=dict(adv_order_h=3, adv_order_v=3))
    r0, t0 = base_state_fields(case)
    nz, ny, nx = r0.shape
    x = (np.arange(nx) + 0.5) * case["dx"]
    zc = 0.5 * (case["z_levels"][:-1] + case["z_levels"][1:])
    rr = np.sqrt(((x[None, :] - 800.0) / 300.0) ** 2 + ((zc[:, None] - 500.0) / 300.0) ** 2)
    dth = np.where(rr < 1, 2.0 * np.cos(0.5 * np.pi * rr) ** 2, 0.0)[:, None, :] * np.ones((1, ny, 1))
    th = t0 / r0 + dth
    st = [r0.copy(), np.zeros_like(r0), np.zeros_like(r0), np.zeros((nz + 1, ny, nx)), r0 * th]
    dz = np.diff(case["z_levels"])[:, None, None]
    o = erfo.Oracle(case)
    o.set_state(*st)
    m0 = float((st[4] * dz).sum())
    wc = []
    for _ in range(8):
        o.anelastic_step(2.0)
        got = o.get_state()
        scale = max(np.abs(got[3]).max(), 1e-30) / case["dx"]
        assert np.abs(o.divergence()).max() <= 1e-11 * max(scale, 1e-6)
        assert np.array_equal(got[0], r0)
        wc.append(float(got[3][5, 1, 7] + got[3][5, 1, 8]) / 2)
    assert abs(float((got[4] * dz).sum()) - m0) <= 1e-12 * abs(m0)
    assert all(b > a > 0 for a, b in zip(wc, wc[1:]))           # upward and accelerating
    assert 0.05 < wc[-1] / r0[5, 0, 0] < 5.0                    # ~ B t reduced by the pressure: m/s after 16 s


def test_anelastic_mode_needs_a_flat_periodic_grid():
    case = wl.make_case(4, nx=8, ny=8, nz=96)
    o = erfo.Oracle(case)
    o.set_state(*case["state"])
    with pytest.raises(RuntimeError):
        o.anelastic_step(0.5)
    case = uniform_case(6, 6, 6, 100.0, 100.0, 50.0)
    case["periodic_x"] = 0
    o = erfo.Oracle(case)
    with pytest.raises(RuntimeError):
        o.anelastic_step(0.5)
