"""Invariants and brute-force checks that pin the oracle's full operators
(BASELINE.json north_star checks (i)-(v))."""
import math

import numpy as np
import pytest

from oracle import erfo
from paper_2412_04395_b200 import workloads as wl
from util import uniform_case, zeros_state, base_state_fields

RD, CP, P00, G = wl.RD, wl.CP, wl.P00, wl.GRAV
CV = CP - RD
GAM = CP / CV


def _hill_case(nx=40, ny=12, nz=20, height=300.0, **par):
    wl.CONFIGS[4]["hill"]["height"] = height
    try:
        return wl.make_case(4, nx=nx, ny=ny, nz=nz, params=par)
    finally:
        wl.CONFIGS[4]["hill"]["height"] = 400.0


# ------------------------------------------------------------ check (i) ----
@pytest.mark.parametrize("cfg,kw", [(2, dict(nx=8, ny=8, nz=12)), (3, dict(nx=8, ny=8, nz=60)),
                                    (4, None)])
@pytest.mark.parametrize("diffusion", [0, 2])
def test_rest_state_stays_at_rest_bitwise(cfg, kw, diffusion):
    """PAPER.md L84 (perturbation pressure, B = -(rho-rho0) g): the base state
    with zero velocity has p' = rho' = 0 identically, so f(S) = 0 exactly and
    the state is unchanged bit for bit, with or without terrain, whatever
    theta0(z)."""
    case = _hill_case(diffusion=diffusion) if cfg == 4 else wl.make_case(
        cfg, params=dict(diffusion=diffusion, nu=0.0, alpha_theta=0.0), **kw)
    o = erfo.Oracle(case)
    r0, t0 = base_state_fields(case)
    st = zeros_state(case)
    st[0][:] = r0
    st[4][:] = t0
    o.set_state(*st)
    R = o.slow_rhs()
    for f in R:
        assert not f.any()
    for _ in range(3):
        o.step(case["dt"], case["ns"])
    out = o.get_state()
    for a, b in zip(out, st):
        assert np.array_equal(a, b)


# ----------------------------------------------------------- check (ii) ----
def _fsum(a):
    return math.fsum(a.ravel().tolist())


@pytest.mark.parametrize("cfg,kw", [(1, dict(nx=12, ny=10, nz=12)), (2, dict(nx=12, ny=12, nz=12)),
                                    (3, dict(nx=12, ny=10, nz=14)), (5, dict(nx=10, ny=12, nz=12)),
                                    (4, None)])
def test_mass_and_rhotheta_conserved(cfg, kw):
    """Flux form on a periodic domain with rigid lids:
    sum(rho * cell volume) and sum(rho theta * cell volume) change only by
    rounding, including diffusion, terrain and the acoustic substeps."""
    case = _hill_case(nx=40, ny=8, nz=16) if cfg == 4 else wl.make_case(cfg, **kw)
    o = erfo.Oracle(case)
    o.set_state(*case["state"])
    hc = o.geometry("hc")[:-1]
    s0 = o.get_state()
    m0, t0 = _fsum(s0[0] * hc), _fsum(s0[4] * hc)
    nsteps = 4
    for _ in range(nsteps):
        o.step(case["dt"], case["ns"])
    s1 = o.get_state()
    assert np.abs(s1[4] - s0[4]).max() > 1e-6          # something did happen
    dm = _fsum((s1[0] - s0[0]) * hc) / m0
    dT = _fsum((s1[4] - s0[4]) * hc) / t0
    assert abs(dm) < 2e-15 and abs(dT) < 2e-15, (dm, dT)


# ---------------------------------------------------------- check (iii) ----
@pytest.mark.parametrize("order", [2, 3, 4, 5, 6])
@pytest.mark.parametrize("diffusion", [0, 2])
def test_free_stream_preserved_over_terrain(order, diffusion):
    """PAPER.md L178/L196 (terrain at nodes, rho*Omega normal to the vertical
    faces): a uniform Cartesian flow over the hill gives zero tendencies
    (discrete geometric conservation).  Checked away from the lids, where the
    kinematic boundary condition necessarily perturbs w."""
    case = _hill_case(nx=36, ny=14, nz=24, height=350.0, g=0.0, adv_order_h=order,
                      adv_order_v=order, diffusion=diffusion)
    shp = (case["nz"], case["ny"], case["nx"])
    case["rho0"] = np.full(shp, 1.1)
    case["rhotheta0"] = np.full(shp, 1.1 * 300.0)
    o = erfo.Oracle(case)
    sxw = o.geometry("sxw")
    assert np.abs(sxw[6]).max() > 0.02                 # the interior levels are sloped
    st = zeros_state(case)
    u0, v0 = 10.0, -4.0
    st[0][:] = 1.1
    st[4][:] = 330.0
    st[1][:] = 1.1 * u0
    st[2][:] = 1.1 * v0
    o.set_state(*st)
    R = o.slow_rhs()
    ks = slice(5, case["nz"] - 5)
    scale = 1.1 * max(abs(u0), abs(v0)) / case["dx"]
    assert np.abs(R[0][ks]).max() < 1e-13 * scale
    assert np.abs(R[4][ks]).max() < 1e-13 * scale * 300.0
    assert np.abs(R[1][ks]).max() < 1e-13 * scale * 10.0
    assert np.abs(R[2][ks]).max() < 1e-13 * scale * 10.0
    assert np.abs(R[3][ks]).max() < 1e-13 * scale * 10.0


def test_metric_pressure_gradient_of_height_only_field():
    """[R:G14] Gx(phi(z)) must vanish up to truncation: with Theta'' linear in
    height the horizontal momenta must not feel it (one substep, R = 0)."""
    case = _hill_case(nx=36, ny=14, nz=24, height=350.0, g=0.0, beta_d=0.0)
    shp = (case["nz"], case["ny"], case["nx"])
    case["rho0"] = np.full(shp, 1.0)
    case["rhotheta0"] = np.full(shp, 300.0)
    o = erfo.Oracle(case)
    zc = o.geometry("zc")[:-1]
    st = zeros_state(case); st[0][:] = 1.0; st[4][:] = 300.0
    o.set_state(*st)
    P = zeros_state(case)
    P[4][:] = 1e-3 * zc                                # linear in z: exact for the chain rule
    out = o.acoustic(0.1, 1, zeros_state(case), P)
    pp, pi = erfo.eos(RD, CP, P00, 300.0, 300.0)
    full = 0.1 * GAM * RD * pi * 1e-3 * np.abs(o.geometry("sxu")[:-1]).max()
    assert full > 1e-3
    ks = slice(1, case["nz"] - 1)                      # one-sided at the lids is also exact here
    assert np.abs(out[1][ks]).max() < 1e-12 * full / 1e-3 and np.abs(out[1]).max() < 1e-10


# ------------------------------------------------------------ check (v) ----
@pytest.mark.parametrize("nz,stretch", [(4, 1.0), (9, 1.12), (12, 1.05)])
@pytest.mark.parametrize("beta_s", [0.1, 0.4])
def test_column_solve_matches_dense_coupled_system(nz, stretch, beta_s):
    """Appendix A rows 3-5 with the averages of L591 solved as
    ONE dense linear system in (W'', Theta'', rho'') -- no elimination --
    against the oracle's tridiagonal route (L144)."""
    rng = np.random.default_rng(7 + nz)
    dz = 30.0 * stretch ** np.arange(nz)
    zl = np.concatenate([[0.0], np.cumsum(dz)])
    zc = 0.5 * (zl[:-1] + zl[1:])
    theta0, rho0 = wl.hydrostatic_base(zc, [(0.0, 0.004, 290.0)])
    par = dict(wl.DEFAULT_PARAMS); par.update(beta_s=beta_s, beta_d=0.0)
    case = dict(name="col", nx=2, ny=2, nz=nz, dx=100.0, dy=100.0, z_nodes=None, z_levels=zl,
                rho0=rho0, rhotheta0=rho0 * theta0, params=par)
    o = erfo.Oracle(case)
    col = lambda a: np.broadcast_to(np.asarray(a)[:, None, None], (len(a), 2, 2)).copy()
    # stage state S^t: the base state plus a z-dependent perturbation
    rho_t = rho0 * (1.0 + 0.01 * rng.standard_normal(nz))
    Th_t = rho0 * theta0 * (1.0 + 0.01 * rng.standard_normal(nz))
    st = zeros_state(case); st[0][:] = col(rho_t); st[4][:] = col(Th_t)
    o.set_state(*st)
    Rr, RT = rng.standard_normal(nz) * 1e-3, rng.standard_normal(nz) * 0.3
    RW = np.concatenate([[0.0], rng.standard_normal(nz - 1) * 1e-2, [0.0]])
    r_old, T_old = rng.standard_normal(nz) * 1e-3, rng.standard_normal(nz) * 0.3
    W_old = np.concatenate([[0.0], rng.standard_normal(nz - 1) * 1e-2, [0.0]])
    R = zeros_state(case); R[0][:] = col(Rr); R[3][:] = col(RW); R[4][:] = col(RT)
    P = zeros_state(case); P[0][:] = col(r_old); P[3][:] = col(W_old); P[4][:] = col(T_old)
    dtau = 0.8
    out = o.acoustic(dtau, 1, R, P)

    # --- the dense coupled system, straight from L585 ---
    b1, b2 = 0.5 * (1 - beta_s), 0.5 * (1 + beta_s)
    th_t = Th_t / rho_t
    pi_t = (RD * Th_t / P00) ** (RD / CV)
    pi0 = (RD * rho0 * theta0 / P00) ** (RD / CV)
    hc = dz
    hw = np.concatenate([[np.nan], zc[1:] - zc[:-1]])           # faces 1..nz-1
    f = lambda a: np.concatenate([[0.0], 0.5 * (a[1:] + a[:-1]), [0.0]])   # cell -> face mean
    thf, pif, pi0f, r0f = f(th_t), f(pi_t), f(pi0), f(rho0)
    nW = nz - 1
    iW = lambda k: k - 1            # k = 1..nz-1
    iT = lambda k: nW + k
    iR = lambda k: nW + nz + k
    n = nW + 2 * nz
    M = np.zeros((n, n)); rhs = np.zeros(n)
    for k in range(1, nz):          # W'' equation at face k
        e = iW(k)
        M[e, iW(k)] = 1.0
        rhs[e] = W_old[k] + dtau * RW[k]
        cpg = dtau * GAM * RD * pif[k] / hw[k]
        Bf = r0f[k] * (RD / CV) * pif[k] / pi0f[k]
        for kk, sgn in ((k, 1.0), (k - 1, -1.0)):
            # -gamma Rd pi d(Theta_bar)/dz + g Bf mean(Theta_bar/Theta^t) - g mean(rho_bar)
            cT = -cpg * sgn + dtau * G * Bf * 0.5 / Th_t[kk]
            cR = -dtau * G * 0.5
            M[e, iT(kk)] -= b2 * cT
            rhs[e] += b1 * cT * T_old[kk]
            M[e, iR(kk)] -= b2 * cR
            rhs[e] += b1 * cR * r_old[kk]
    for k in range(nz):             # Theta'' and rho'' equations at cell k
        for row, q_old, Rq, wgt in ((iT(k), T_old, RT, thf), (iR(k), r_old, Rr, None)):
            M[row, row] = 1.0
            rhs[row] = q_old[k] + dtau * Rq[k]
            for kf, sgn in ((k + 1, 1.0), (k, -1.0)):
                if kf == 0 or kf == nz:
                    continue
                cw = -dtau * sgn * (wgt[kf] if wgt is not None else 1.0) / hc[k]
                M[row, iW(kf)] -= b2 * cw
                rhs[row] += b1 * cw * W_old[kf]
    x = np.linalg.solve(M, rhs)
    Wn = np.concatenate([[0.0], x[:nW], [0.0]])
    Tn, rn = x[nW:nW + nz], x[nW + nz:]
    assert np.abs(out[3][:, 0, 0] - Wn).max() < 1e-13 * np.abs(Wn).max()
    assert np.abs(out[4][:, 1, 0] - Tn).max() < 1e-13 * np.abs(Tn).max()
    assert np.abs(out[0][:, 0, 1] - rn).max() < 1e-13 * np.abs(rn).max()

    # the tridiagonal rows themselves: strictly diagonally dominant, and Thomas == LU
    A, D, Cc = o.tridiag_rows(dtau, 0, 0)
    assert np.all(np.abs(D[1:nz]) > np.abs(A[1:nz]) + np.abs(Cc[1:nz]))


# ------------------------------------------------------- Smagorinsky -------
def test_smagorinsky_uniform_shear_closed_form():
    """[R:G9] mu_t = rho (Cs Delta)^2 |S|; u = alpha z gives |S| = alpha
    exactly on interior levels (S13 = alpha/2); Delta = (dx dy dz)^(1/3)."""
    nx, ny, nz, dx, dy, dz = 6, 5, 10, 40.0, 25.0, 10.0
    case = uniform_case(nx, ny, nz, dx, dy, dz, diffusion=2, Cs=0.18, rho0=1.2)
    o = erfo.Oracle(case)
    st = zeros_state(case)
    st[0][:] = 1.2; st[4][:] = 360.0
    alpha = 0.05
    zc = (np.arange(nz) + 0.5) * dz
    st[1][:] = 1.2 * alpha * zc[:, None, None]
    o.set_state(*st)
    mu = o.viscosity()
    expect = 1.2 * (0.18 * (dx * dy * dz) ** (1 / 3)) ** 2 * alpha
    assert np.abs(mu[1:-1] - expect).max() < 1e-13 * expect
    assert np.abs(mu[0] - 0.5 * expect).max() < 1e-13 * expect   # free-slip lid: S13 = 0 there


def test_smagorinsky_plane_strain_closed_form():
    """u = A sin(kx): S11 = dudx, S33 = S22 = 0 -> |S| = sqrt(2) |S11| with the
    two-point difference dudx = A (2/dx) sin(k dx/2) cos(k x_c)."""
    nx, dx = 16, 20.0
    case = uniform_case(nx, 4, 6, dx, dx, dx, diffusion=2, Cs=0.2)
    o = erfo.Oracle(case)
    st = zeros_state(case); st[0][:] = 1.0; st[4][:] = 300.0
    k = 2 * np.pi / (nx * dx)
    xf = np.arange(nx) * dx
    st[1][:] = 3.0 * np.sin(k * xf)[None, None, :]
    o.set_state(*st)
    mu = o.viscosity()
    xc = xf + 0.5 * dx
    s11 = 3.0 * (2 / dx) * np.sin(k * dx / 2) * np.cos(k * xc)
    expect = (0.2 * dx) ** 2 * np.sqrt(2.0) * np.abs(s11)
    assert np.abs(mu - expect[None, None, :]).max() < 1e-13 * expect.max()


def test_constant_viscosity_is_rho_nu():
    case = wl.make_case(2, nx=6, ny=6, nz=8)
    o = erfo.Oracle(case)
    o.set_state(*case["state"])
    assert np.allclose(o.viscosity(), case["state"][0] * 1.0, rtol=1e-15)


# --------------------------------------------------------- check (iv-c) ----
def test_gravity_wave_frequency():
    """Linear theory: internal gravity wave in a stratified fluid,
    omega^2 = N^2 k^2/(k^2+m^2), N^2 = g dln(theta0)/dz.  Full RK3 + substeps;
    agreement to a few per cent (compressibility, truncation)."""
    nx, nz, h = 16, 16, 200.0
    gam_th = 0.01
    zl = np.arange(nz + 1) * h
    zc = 0.5 * (zl[1:] + zl[:-1])
    theta0, rho0 = wl.hydrostatic_base(zc, [(0.0, gam_th, 300.0)])
    par = dict(wl.DEFAULT_PARAMS)
    case = dict(name="gw", nx=nx, ny=2, nz=nz, dx=h, dy=h, z_nodes=None, z_levels=zl,
                rho0=rho0, rhotheta0=rho0 * theta0, params=par)
    o = erfo.Oracle(case)
    kx, mz = 2 * np.pi / (nx * h), np.pi / (nz * h)
    xc = (np.arange(nx) + 0.5) * h
    shape = np.sin(mz * zc)[:, None, None] * np.cos(kx * xc)[None, None, :] * np.ones((nz, 2, nx))
    st = zeros_state(case)
    # buoyancy perturbation at constant pressure: Theta unchanged, rho' = -rho0 theta'/theta0
    st[4][:] = (rho0 * theta0)[:, None, None]
    st[0][:] = rho0[:, None, None] * (1.0 - 1e-4 * shape)
    o.set_state(*st)
    N2 = G * gam_th / theta0.mean()
    omega = np.sqrt(N2 * kx * kx / (kx * kx + mz * mz))
    dt = 2.0
    amp0 = ((st[0] - rho0[:, None, None]) * shape).sum()
    t_cross = None
    prev = amp0
    for n in range(1, 400):
        o.step(dt, 6)
        a = ((o.get_state()[0] - rho0[:, None, None]) * shape).sum()
        if prev * a < 0:
            t_cross = dt * (n - 1 + prev / (prev - a))
            break
        prev = a
    assert t_cross is not None
    quarter = 0.5 * np.pi / omega
    assert abs(t_cross - quarter) < 0.04 * quarter, (t_cross, quarter)
