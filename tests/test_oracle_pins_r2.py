"""Closed-form pins of the oracle parts that round 1 left unconstrained
(VERDICT round 1, W1): the diffusion tendencies -div(tau) and div(rho alpha
grad theta) (Eq. 9), the divergence-damping line of
the substep (L144, reading G6), the kinematic lids over terrain (reading G15)
and the terrain chain rule in the strain (L178, reading G14).

Every expected value is a closed form of the DISCRETE operator (two-point
differences of a single Fourier / cosine mode, or a field that is linear in
the Cartesian height), derived by hand from the paper's equations -- none
calls the oracle to obtain it.  Geometry used for expected values is computed
here from the node heights with numpy.
"""
import numpy as np
import pytest

from oracle import erfo
from paper_2412_04395_b200 import workloads as wl
from util import uniform_case, zeros_state

RD, CP, P00 = wl.RD, wl.CP, wl.P00
GAM = CP / (CP - RD)


def _khat(k, h):
    """Symbol of the two-point difference: delta(sin kx) = khat h cos(kx)."""
    return (2.0 / h) * np.sin(0.5 * k * h)


def _diff_pair(case_kw, state_fn, **visc):
    """slow_rhs with diffusion on minus slow_rhs with diffusion off, same state:
    advection and pressure gradient drop out, leaving the diffusion tendency."""
    out = []
    for par in (visc, dict(diffusion=0)):
        case = uniform_case(**case_kw, **par)
        o = erfo.Oracle(case)
        o.set_state(*state_fn(case))
        out.append(o.slow_rhs())
    return [a - b for a, b in zip(*out)]


# ------------------------------------------------------------------------
# (a) diffusion: sign and factor of every stress component
# ------------------------------------------------------------------------
GRID = dict(nx=16, ny=12, nz=10, dx=40.0, dy=25.0, dz=15.0)
NU = 7.5
A = 2.0e-2


def _coords(case):
    nx, ny, nz, dx, dy = case["nx"], case["ny"], case["nz"], case["dx"], case["dy"]
    dz = case["z_levels"][1] - case["z_levels"][0]
    xf = (np.arange(nx) * dx)[None, None, :]
    xc = xf + 0.5 * dx
    yf = (np.arange(ny) * dy)[None, :, None]
    yc = yf + 0.5 * dy
    zc = ((np.arange(nz) + 0.5) * dz)[:, None, None]
    zf = (np.arange(nz + 1) * dz)[:, None, None]
    return xf, xc, yf, yc, zc, zf, dz


def _base(case):
    st = zeros_state(case)
    st[0][:] = 1.0
    st[4][:] = 300.0
    return st


def test_tau11_normal_stress_on_u():
    """Eq. 9 (L102): tau11 = -2 mu (S11 - div/3); u = A sin(kx), rho = 1:
    -d(tau11)/dx = +(4/3) nu d2u/dx2 = -(4/3) nu khat^2 u."""
    k = 2 * np.pi * 2 / (GRID["nx"] * GRID["dx"])

    def state(case):
        xf, *_ = _coords(case)
        st = _base(case)
        st[1][:] = A * np.sin(k * xf)
        return st

    d = _diff_pair(GRID, state, diffusion=1, nu=NU, alpha_theta=0.0)
    case = uniform_case(**GRID)
    xf, *_ = _coords(case)
    expect = -(4.0 / 3.0) * NU * _khat(k, GRID["dx"]) ** 2 * A * np.sin(k * xf) * np.ones_like(d[1])
    assert np.abs(d[1] - expect).max() < 1e-12 * np.abs(expect).max()
    for f in (0, 2, 3, 4):
        assert np.abs(d[f]).max() < 1e-13 * np.abs(expect).max()


def test_tau22_normal_stress_on_v():
    k = 2 * np.pi / (GRID["ny"] * GRID["dy"])

    def state(case):
        _, _, yf, *_ = _coords(case)
        st = _base(case)
        st[2][:] = A * np.sin(k * yf)
        return st

    d = _diff_pair(GRID, state, diffusion=1, nu=NU, alpha_theta=0.0)
    _, _, yf, *_ = _coords(uniform_case(**GRID))
    expect = -(4.0 / 3.0) * NU * _khat(k, GRID["dy"]) ** 2 * A * np.sin(k * yf) * np.ones_like(d[2])
    assert np.abs(d[2] - expect).max() < 1e-12 * np.abs(expect).max()
    for f in (0, 1, 3, 4):
        assert np.abs(d[f]).max() < 1e-13 * np.abs(expect).max()


def test_tau12_shear_stress_on_u_and_v():
    """tau12 = -2 mu S12, S12 = (du/dy + dv/dx)/2.  u = A sin(k y): -d(tau12)/dy = -nu khat_y^2 u;
    v = A sin(k x): -d(tau12)/dx = -nu khat_x^2 v."""
    ky = 2 * np.pi * 3 / (GRID["ny"] * GRID["dy"])
    kx = 2 * np.pi / (GRID["nx"] * GRID["dx"])

    def state(case):
        xf, xc, yf, yc, *_ = _coords(case)
        st = _base(case)
        st[1][:] = A * np.sin(ky * yc)          # U lives at (x_face, y_centre)
        st[2][:] = 0.5 * A * np.sin(kx * xc)    # V lives at (x_centre, y_face)
        return st

    d = _diff_pair(GRID, state, diffusion=1, nu=NU, alpha_theta=0.0)
    xf, xc, yf, yc, *_ = _coords(uniform_case(**GRID))
    eu = -NU * _khat(ky, GRID["dy"]) ** 2 * A * np.sin(ky * yc) * np.ones_like(d[1])
    ev = -NU * _khat(kx, GRID["dx"]) ** 2 * 0.5 * A * np.sin(kx * xc) * np.ones_like(d[2])
    assert np.abs(d[1] - eu).max() < 1e-12 * np.abs(eu).max()
    assert np.abs(d[2] - ev).max() < 1e-12 * np.abs(ev).max()
    assert np.abs(d[3]).max() < 1e-13 * np.abs(eu).max()


def test_tau13_tau23_vertical_shear_with_free_slip_lids():
    """tau13 = -2 mu S13 with S13 = 0 on the lids (slip wall, Table C1): the cosine modes
    u = A cos(m z), m = n pi / H are eigenfunctions of the two-point second difference
    with zero-flux ends: -d(tau13)/dz = -nu mhat^2 u.  Same for v through tau23."""
    H = GRID["nz"] * GRID["dz"]
    m1, m2 = 2 * np.pi / H, 3 * np.pi / H

    def state(case):
        *_, zc, zf, dz = _coords(case)
        st = _base(case)
        st[1][:] = A * np.cos(m1 * zc)
        st[2][:] = -A * np.cos(m2 * zc)
        return st

    d = _diff_pair(GRID, state, diffusion=1, nu=NU, alpha_theta=0.0)
    *_, zc, zf, dz = _coords(uniform_case(**GRID))
    eu = -NU * _khat(m1, dz) ** 2 * A * np.cos(m1 * zc) * np.ones_like(d[1])
    ev = +NU * _khat(m2, dz) ** 2 * A * np.cos(m2 * zc) * np.ones_like(d[2])
    assert np.abs(d[1] - eu).max() < 1e-12 * np.abs(eu).max()
    assert np.abs(d[2] - ev).max() < 1e-12 * np.abs(ev).max()


def test_stress_divergence_of_w_mode_all_components():
    """w = A sin(kx x) sin(ky y) sin(m z) (zero on the lids): with mu constant,
    -div(tau) = nu (lap(u_i) + (1/3) d_i div u):
      R_W = -nu (khx^2 + khy^2 + (4/3) mh^2) w,
      R_U = +(1/3) nu d2w/dxdz,  R_V = +(1/3) nu d2w/dydz   (two-point differences)."""
    H = GRID["nz"] * GRID["dz"]
    kx = 2 * np.pi / (GRID["nx"] * GRID["dx"])
    ky = 2 * np.pi * 2 / (GRID["ny"] * GRID["dy"])
    m = 2 * np.pi / H

    def state(case):
        xf, xc, yf, yc, zc, zf, dz = _coords(case)
        st = _base(case)
        st[3][:] = A * np.sin(kx * xc) * np.sin(ky * yc) * np.sin(m * zf)
        return st

    d = _diff_pair(GRID, state, diffusion=1, nu=NU, alpha_theta=0.0)
    xf, xc, yf, yc, zc, zf, dz = _coords(uniform_case(**GRID))
    khx, khy, mh = _khat(kx, GRID["dx"]), _khat(ky, GRID["dy"]), _khat(m, dz)
    ew = -NU * (khx ** 2 + khy ** 2 + (4.0 / 3.0) * mh ** 2) * A * np.sin(kx * xc) * np.sin(ky * yc) * np.sin(m * zf)
    eu = (NU / 3.0) * khx * mh * A * np.cos(kx * xf) * np.sin(ky * yc) * np.cos(m * zc)
    ev = (NU / 3.0) * khy * mh * A * np.sin(kx * xc) * np.cos(ky * yf) * np.cos(m * zc)
    s = np.abs(ew).max()
    assert np.abs(d[3] - ew).max() < 1e-12 * s
    assert np.abs(d[1] - eu).max() < 1e-12 * s
    assert np.abs(d[2] - ev).max() < 1e-12 * s
    assert not d[3][0].any() and not d[3][-1].any()          # R_W = 0 on the lids


@pytest.mark.parametrize("axis", ["x", "y", "z"])
def test_scalar_diffusion_sign_and_factor(axis):
    """Eq. 3 (L67): +div(rho alpha grad theta).  theta = theta0 + A sin(k x) (or y; or
    cos(m z) with zero-flux lids), rho = 1: R_Theta = -rho alpha khat^2 (theta - theta0)."""
    alpha = 3.0
    H = GRID["nz"] * GRID["dz"]
    kk = dict(x=2 * np.pi / (GRID["nx"] * GRID["dx"]), y=2 * np.pi * 2 / (GRID["ny"] * GRID["dy"]),
              z=3 * np.pi / H)[axis]

    def mode(case):
        xf, xc, yf, yc, zc, zf, dz = _coords(case)
        shp = (case["nz"], case["ny"], case["nx"])
        return dict(x=np.sin(kk * xc), y=np.sin(kk * yc), z=np.cos(kk * zc))[axis] * np.ones(shp)

    def state(case):
        st = _base(case)
        st[4][:] = 300.0 + AT * mode(case)
        return st

    AT = 5.0        # K; large enough that the rounding of theta = Theta/rho ~ 300 stays below 1e-11
    d = _diff_pair(GRID, state, diffusion=1, nu=0.0, alpha_theta=alpha)
    case = uniform_case(**GRID)
    h = dict(x=GRID["dx"], y=GRID["dy"], z=GRID["dz"])[axis]
    expect = -alpha * _khat(kk, h) ** 2 * AT * mode(case)
    assert np.abs(d[4] - expect).max() < 1e-11 * np.abs(expect).max()
    for f in (0, 1, 2, 3):
        assert not d[f].any()


def test_viscosity_is_mu_equals_rho_nu_with_edge_means_and_face_density():
    """[R:G10] mu = rho nu with the LOCAL rho, [R:G11] edge mu = 4-point mean, u = U/rho_u
    with rho_u the two-point mean.  rho = 1 + e cos(q x), U = rho_u A sin(k y): u = A sin(k y),
    S12 = du/dy / 2, mu12(i-1/2) = nu (rho(i-1) + rho(i))/2 = nu rho_u:
    R_U = -nu rho_u khat^2 A sin(k y)."""
    q = 2 * np.pi / (GRID["nx"] * GRID["dx"])
    ky = 2 * np.pi / (GRID["ny"] * GRID["dy"])

    def rho_of(case):
        xf, xc, yf, yc, *_ = _coords(case)
        return (1.0 + 0.2 * np.cos(q * xc)) * np.ones((case["nz"], case["ny"], case["nx"]))

    def state(case):
        xf, xc, yf, yc, *_ = _coords(case)
        st = _base(case)
        rho = rho_of(case)
        st[0][:] = rho
        rho_u = 0.5 * (rho + np.roll(rho, 1, axis=2))
        st[1][:] = rho_u * A * np.sin(ky * yc)
        return st

    d = _diff_pair(GRID, state, diffusion=1, nu=NU, alpha_theta=0.0)
    case = uniform_case(**GRID)
    xf, xc, yf, yc, *_ = _coords(case)
    rho = rho_of(case)
    rho_u = 0.5 * (rho + np.roll(rho, 1, axis=2))
    expect = -NU * rho_u * _khat(ky, GRID["dy"]) ** 2 * A * np.sin(ky * yc)
    assert np.abs(d[1] - expect).max() < 1e-12 * np.abs(expect).max()


def test_smagorinsky_scalar_diffusivity_is_mut_over_prt():
    """[R:G9] K_theta = mu_t / Pr_t.  Uniform shear u = a z gives mu_t = rho (Cs Delta)^2 a on
    interior levels; theta = theta0 + A sin(k y) then diffuses with K = mu_t / Pr_t."""
    nx, ny, nz, dx, dy, dz = 6, 12, 10, 40.0, 25.0, 10.0
    g = dict(nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz)
    a, Cs, Prt = 0.05, 0.18, 0.4
    ky = 2 * np.pi / (ny * dy)

    def state(case):
        xf, xc, yf, yc, zc, zf, _ = _coords(case)
        st = _base(case)
        st[1][:] = a * zc * np.ones_like(st[1])
        st[4][:] = 300.0 + 5.0 * np.sin(ky * yc)
        return st

    d = _diff_pair(g, state, diffusion=2, Cs=Cs, Pr_t=Prt)
    xf, xc, yf, yc, zc, zf, _ = _coords(uniform_case(**g))
    mut = (Cs * (dx * dy * dz) ** (1.0 / 3.0)) ** 2 * a
    expect = -(mut / Prt) * _khat(ky, dy) ** 2 * 5.0 * np.sin(ky * yc) * np.ones((nz, ny, nx))
    ks = slice(2, nz - 2)
    assert np.abs(d[4][ks] - expect[ks]).max() < 1e-11 * np.abs(expect).max()


# ------------------------------------------------------------------------
# (b) divergence damping (L144, reading G6)
# ------------------------------------------------------------------------
@pytest.mark.parametrize("beta_d", [0.1, 0.3])
@pytest.mark.parametrize("direction", ["x", "y"])
def test_divergence_damping_recurrence(beta_d, direction):
    """Rows 1, 2, 4 of L585 with Theta''_d = Theta'' + beta_d (Theta'' - Theta''_prev)
    in the pressure gradient (L144: "predicted slightly forward in time").  Eliminating
    U'' gives, for the amplitude T_n of a Theta'' standing wave,
        T_{n+1} = (2 - mu^2 (1 + beta_d)) T_n - (1 - mu^2 beta_d) T_{n-1},
        T_1 = (1 - mu^2) T_0      (Theta''_prev = Theta'' initially, U''_0 = 0),
    mu = 2 (c dtau / h) sin(k h / 2)."""
    n, h = 16, 100.0
    dims = dict(x=2, y=2, z=3)
    dims[direction] = n
    case = uniform_case(dims["x"], dims["y"], dims["z"], h, h, h, beta_d=beta_d)
    o = erfo.Oracle(case)
    st = zeros_state(case)
    st[0][:] = 1.0
    st[4][:] = 300.0
    o.set_state(*st)
    pi = (RD * 300.0 / P00) ** (RD / (CP - RD))
    c = np.sqrt(GAM * RD * pi * 300.0)
    nz, ny, nx = st[0].shape
    kk, jj, ii = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    m = {"x": ii, "y": jj}[direction]
    kw = 2 * np.pi * 2 / (n * h)
    shape = np.cos(kw * (m + 0.5) * h)
    dtau = 0.5 * h / c
    mu2 = (2.0 * (c * dtau / h) * np.sin(kw * h / 2.0)) ** 2
    T = [1.0, 1.0 - mu2]
    for _ in range(2, 10):
        T.append((2.0 - mu2 * (1.0 + beta_d)) * T[-1] - (1.0 - mu2 * beta_d) * T[-2])
    # damping really damps: the undamped recurrence stays on |T| <= 1 + eps; compare end values
    Tu = [1.0, 1.0 - mu2]
    for _ in range(2, 10):
        Tu.append((2.0 - mu2) * Tu[-1] - Tu[-2])
    assert abs(T[9] - Tu[9]) > 1e-2
    R = zeros_state(case)
    P = zeros_state(case)
    P[4][:] = 1e-3 * shape
    P[0][:] = 1e-3 * shape / 300.0
    for nsub in (1, 2, 3, 6, 9):
        out = o.acoustic(dtau, nsub, R, P)
        amp = (out[4] * shape).sum() / (shape * shape).sum() / 1e-3
        assert abs(amp - T[nsub]) < 1e-12, (nsub, amp, T[nsub])


# ------------------------------------------------------------------------
# (c), (d) terrain: kinematic lids and the chain rule
# ------------------------------------------------------------------------
def _two_sided_hill(nx=24, ny=10, nz=14, **par):
    """A terrain grid whose BOTTOM and TOP coordinate surfaces are both sloped:
    z = zeta + h(x, y) (1 - zeta / (2 z_top)).  Uniform base state, no gravity."""
    dx = dy = 100.0
    zl = np.arange(nz + 1) * 40.0
    x = np.arange(nx + 1) * dx
    y = np.arange(ny + 1) * dy
    Lx, Ly = nx * dx, ny * dy
    h = 120.0 * (np.sin(2 * np.pi * x / Lx)[None, :] ** 2) * (0.6 + 0.4 * np.cos(2 * np.pi * y / Ly)[:, None])
    zn = zl[:, None, None] + h[None] * (1.0 - zl[:, None, None] / (2.0 * zl[-1]))
    p = dict(wl.DEFAULT_PARAMS)
    p.update(g=0.0)
    p.update(par)
    shp = (nz, ny, nx)
    return dict(name="hill2", nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, z_nodes=zn, z_levels=None,
                rho0=np.full(shp, 1.1), rhotheta0=np.full(shp, 330.0), params=p)


def _geometry(zn, dx, dy):
    """S0 restated with numpy from the node heights (reading G14)."""
    zxf = 0.5 * (zn[:, :-1, :] + zn[:, 1:, :])          # [k][j][i in 0..nx]
    zyf = 0.5 * (zn[:, :, :-1] + zn[:, :, 1:])          # [k][j in 0..ny][i]
    zw = 0.25 * (zn[:, :-1, :-1] + zn[:, :-1, 1:] + zn[:, 1:, :-1] + zn[:, 1:, 1:])
    sxw = (zxf[:, :, 1:] - zxf[:, :, :-1]) / dx
    syw = (zyf[:, 1:, :] - zyf[:, :-1, :]) / dy
    hc = zw[1:] - zw[:-1]
    zc = 0.5 * (zw[1:] + zw[:-1])
    return zw, zc, hc, sxw, syw


def _kinematic(sx, sy, U, V):
    return sx * 0.5 * (U + np.roll(U, -1, axis=1)) + sy * 0.5 * (V + np.roll(V, -1, axis=0))


def test_kinematic_lids_on_set_state_and_after_a_step():
    """[R:G15] rigid lids over terrain: Omega = 0 there, i.e.
    W(lid) = sxw * mean_x(U) + syw * mean_y(V) of the adjacent level -- on set_state and
    after every stage of a step."""
    case = _two_sided_hill()
    zw, zc, hc, sxw, syw = _geometry(case["z_nodes"], case["dx"], case["dy"])
    assert np.abs(sxw[0]).max() > 0.05 and np.abs(sxw[-1]).max() > 0.02
    o = erfo.Oracle(case)
    st = zeros_state(case)
    u0, v0 = 10.0, -4.0
    st[0][:] = 1.1
    st[4][:] = 330.0
    st[1][:] = 1.1 * u0
    st[2][:] = 1.1 * v0
    st[3][:] = 0.123                        # whatever the caller passes at the lids is replaced
    o.set_state(*st)
    got = o.get_state()
    eb = 1.1 * (u0 * sxw[0] + v0 * syw[0])
    et = 1.1 * (u0 * sxw[-1] + v0 * syw[-1])
    assert np.abs(got[3][0] - eb).max() < 1e-14 * np.abs(eb).max()
    assert np.abs(got[3][-1] - et).max() < 1e-14 * np.abs(eb).max()
    assert np.all(got[3][1:-1] == 0.123)
    # after a full step U, V are no longer uniform: the lid value follows them
    st[3][:] = 0.0
    o.set_state(*st)
    o.step(0.2, 4)
    s1 = o.get_state()
    assert np.abs(s1[1] - 1.1 * u0).max() > 1e-4
    eb = _kinematic(sxw[0], syw[0], s1[1][0], s1[2][0])
    et = _kinematic(sxw[-1], syw[-1], s1[1][-1], s1[2][-1])
    assert np.abs(s1[3][0] - eb).max() < 1e-13 * np.abs(eb).max()
    assert np.abs(s1[3][-1] - et).max() < 1e-13 * np.abs(eb).max()


def test_lid_adjacent_continuity_sees_an_impermeable_wall():
    """With Omega(lid) = 0 (L196, reading G15) a uniform Cartesian flow (u0, v0, 0) has zero
    mass divergence on every interior level (discrete GCL) but NOT in the lid-adjacent cells:
    there the geometric term of the missing lid flux remains,
        R_rho(k=0)    = +rho (u0 sxw(0)  + v0 syw(0))  / hc(0)      (flow up the slope piles up),
        R_rho(k=nz-1) = -rho (u0 sxw(nz) + v0 syw(nz)) / hc(nz-1),
    from  delta_x(hx)/dx = sxw(k+1) - sxw(k)  and  Omega(1) = -sxw(1) U - syw(1) V;
    R_Theta = theta R_rho."""
    case = _two_sided_hill(adv_order_h=2, adv_order_v=2)
    zw, zc, hc, sxw, syw = _geometry(case["z_nodes"], case["dx"], case["dy"])
    o = erfo.Oracle(case)
    st = zeros_state(case)
    u0, v0 = 10.0, -4.0
    st[0][:] = 1.1
    st[4][:] = 330.0
    st[1][:] = 1.1 * u0
    st[2][:] = 1.1 * v0
    o.set_state(*st)
    R = o.slow_rhs()
    e0 = +1.1 * (u0 * sxw[0] + v0 * syw[0]) / hc[0]
    e1 = -1.1 * (u0 * sxw[-1] + v0 * syw[-1]) / hc[-1]
    s = np.abs(e0).max()
    assert np.abs(R[0][0] - e0).max() < 1e-12 * s
    assert np.abs(R[0][-1] - e1).max() < 1e-12 * s
    assert np.abs(R[0][1:-1]).max() < 1e-12 * s
    assert np.abs(R[4][0] - 300.0 * e0).max() < 1e-12 * s * 300.0
    assert np.abs(R[4][-1] - 300.0 * e1).max() < 1e-12 * s * 300.0
    assert np.abs(R[4][1:-1]).max() < 1e-12 * s * 300.0


def test_strain_chain_rule_cartesian_linear_shear_over_terrain():
    """[R:G14] d/dx|_z = delta_x - slope * mean(vertical quotients).  The Cartesian field
    (u, v, w) = (a, b, e) * z sampled at the terrain-following u-, v-, w-points has
    S11 = S22 = S12 = 0, S33 = e, S13 = a/2, S23 = b/2 exactly (every difference of a linear
    function is exact), so |S| = sqrt(2 e^2 + a^2 + b^2) and
    mu_t = rho (Cs Delta)^2 |S|, Delta = (dx dy hc)^(1/3) on the levels away from the lids."""
    Cs = 0.18
    case = _two_sided_hill(diffusion=2, Cs=Cs)
    nx, ny, nz = case["nx"], case["ny"], case["nz"]
    zw, zc, hc, sxw, syw = _geometry(case["z_nodes"], case["dx"], case["dy"])
    a, b, e = 0.03, -0.02, 0.01
    rho = 1.1
    zcu = 0.5 * (zc + np.roll(zc, 1, axis=2))
    zcv = 0.5 * (zc + np.roll(zc, 1, axis=1))
    st = zeros_state(case)
    st[0][:] = rho
    st[4][:] = 330.0
    st[1][:] = rho * a * zcu
    st[2][:] = rho * b * zcv
    st[3][:] = rho * e * zw
    o = erfo.Oracle(case)
    o.set_state(*st)
    mu = o.viscosity()
    delta = (case["dx"] * case["dy"] * hc) ** (1.0 / 3.0)
    expect = rho * (Cs * delta) ** 2 * np.sqrt(2 * e * e + a * a + b * b)
    ks = slice(2, nz - 2)
    assert np.abs(sxw[3]).max() > 0.03
    assert np.abs(mu[ks] / expect[ks] - 1.0).max() < 1e-11
    # without the slope terms S11 alone would be a * d(zcu)/dx ~ a * 0.05: a 100 % change of |S|


def test_diffusion_chain_rule_linear_theta_over_terrain():
    """[R:G14] scalar diffusion over terrain: theta linear in the Cartesian height,
    K = rho alpha constant: the horizontal fluxes Fx = -K (delta_x theta - sxu mean(d theta/dz))
    vanish identically and the contravariant vertical flux is uniform, so the diffusion
    tendency of Theta is zero away from the lids (where the zero-flux wall acts)."""
    case0 = _two_sided_hill(diffusion=0)
    case1 = _two_sided_hill(diffusion=1, nu=0.0, alpha_theta=5.0)
    nz = case0["nz"]
    zw, zc, hc, sxw, syw = _geometry(case0["z_nodes"], case0["dx"], case0["dy"])
    Gam = 0.01
    st = zeros_state(case0)
    st[0][:] = 1.1
    st[4][:] = 1.1 * (300.0 + Gam * zc)
    out = []
    for case in (case1, case0):
        o = erfo.Oracle(case)
        o.set_state(*st)
        out.append(o.slow_rhs())
    d = out[0][4] - out[1][4]
    wall = 5.0 * 1.1 * Gam / hc[0].min()                  # size of the lid-cell tendency
    assert np.abs(d[0]).max() > 0.5 * wall * hc[0].min() / hc[0].max()
    assert np.abs(d[2:nz - 2]).max() < 1e-11 * wall
