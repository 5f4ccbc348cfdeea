"""Pins for the CPU oracle against what the paper and the mathematics fix
(SURVEY.md 8(c) "What pins the oracle"): EOS closed form (Eq. 7), RK3
amplification polynomial (Eq. 11-13), substep schedule (L170), rest state,
conservation, free-stream preservation over terrain, discrete acoustic
dispersion (Appendix A), Smagorinsky closed forms.  None of these retypes the
oracle's own formulae: each compares with a closed form or an invariant."""
import numpy as np
import pytest

from oracle import erfo
from paper_2412_04395_b200 import workloads as wl
from util import uniform_case, zeros_state, base_state_fields

RD, CP, P00 = wl.RD, wl.CP, wl.P00
GAM = CP / (CP - RD)


# ---------------------------------------------------------------- Eq. 7 ----
@pytest.mark.parametrize("Theta0", [300.0 * 1.16, 265.0 * 1.3, 320.0 * 0.4])
@pytest.mark.parametrize("rel", [0.0, 1e-9, -3e-6, 1e-3, -0.02, 0.1])
def test_eos_matches_eq7_in_long_double(Theta0, rel):
    """p = P00 (Rd rho theta / P00)^gamma; p' = p - p0.  The
    oracle's expm1/log1p form must equal the printed formula evaluated in
    extended precision, to a relative error of a few ulp OF p' (not of p)."""
    L = np.longdouble
    Theta = Theta0 * (1.0 + rel)
    pp, pi = erfo.eos(RD, CP, P00, Theta, Theta0)
    gam = L(CP) / (L(CP) - L(RD))
    p = L(P00) * (L(RD) * L(Theta) / L(P00)) ** gam
    p0 = L(P00) * (L(RD) * L(Theta0) / L(P00)) ** gam
    exact = p - p0
    # long double has 64 mantissa bits: the subtraction itself is good to ~1e-19*p
    tol = 8e-16 * abs(float(exact)) + 2e-19 * float(p) * 4
    assert abs(L(pp) - exact) <= tol, (pp, float(exact))
    pi_exact = (p / L(P00)) ** (L(RD) / L(CP))          # L84: pi = (p/P00)^(Rd/cp)
    assert abs(L(pi) - pi_exact) <= 4e-16 * float(pi_exact)


def test_eos_reference_values():
    """Textbook anchors: Theta = P00/Rd gives p = P00 and pi = 1 exactly;
    gamma = cp/cv = 1.4 for (287, 1004.5)."""
    assert abs(GAM - 1.4) < 1e-12
    pp, pi = erfo.eos(RD, CP, P00, P00 / RD, P00 / RD)
    assert pp == 0.0 and abs(pi - 1.0) < 2e-16


# ----------------------------------------------------------------- L170 ----
@pytest.mark.parametrize("ns", [2, 6, 8, 10])
def test_substep_schedule(ns):
    """one substep in stage 1; even number ns per dt; RK3 stage
    lengths dt/3, dt/2, dt (L140)."""
    dt = 0.6
    n1, tau1, dts1 = erfo.schedule(1, dt, ns)
    n2, tau2, dts2 = erfo.schedule(2, dt, ns)
    n3, tau3, dts3 = erfo.schedule(3, dt, ns)
    assert (n1, n2, n3) == (1, ns // 2, ns)
    assert np.isclose(n1 * tau1, dt / 3) and np.isclose(n2 * tau2, dt / 2) and np.isclose(n3 * tau3, dt)
    assert (dts1, dts2, dts3) == (dt / 3, dt / 2, dt)


def test_odd_substep_count_rejected():
    case = uniform_case(4, 4, 4, 100., 100., 100.)
    o = erfo.Oracle(case)
    st = zeros_state(case); st[0][:] = 1.0; st[4][:] = 300.0
    o.set_state(*st)
    with pytest.raises(RuntimeError):
        o.step(0.1, 5)


# ------------------------------------------------------------ Eq. 11-13 ----
def _acoustic_standing_wave(direction, n=16, h=100.0, eps_rel=1e-7):
    dims = dict(x=2, y=2, z=2); dims[direction] = n
    case = uniform_case(dims["x"], dims["y"], dims["z"], h, h, h, substep_mode=0,
                        adv_order_h=2, adv_order_v=2)
    st = zeros_state(case)
    rho0, th0 = 1.0, 300.0
    st[0][:] = rho0
    nz, ny, nx = st[0].shape
    kk, jj, ii = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    m = {"x": ii, "y": jj, "z": kk}[direction]
    # x,y: periodic mode; z: cosine mode compatible with the rigid lids
    kw = (2 * np.pi / (n * h)) if direction != "z" else (np.pi / (n * h))
    shape = np.cos(kw * (m + 0.5) * h)
    eps = eps_rel * rho0 * th0
    st[4][:] = rho0 * th0 + eps * shape
    # isentropic density perturbation so that theta stays uniform: rho'/rho = Theta'/Theta
    st[0][:] = rho0 * (1.0 + eps_rel * shape)
    return case, st, shape, eps, kw, h, rho0 * th0


@pytest.mark.parametrize("direction", ["x", "y", "z"])
def test_rk3_amplification_polynomial(direction):
    """Eq. 11-13 (L126-L132) applied to a linear system dS/dt = L S multiply an
    eigenmode by 1 + z + z^2/2 + z^3/6.  Small-amplitude sound wave on a
    uniform state at rest without substepping (L140): L has eigenvalues
    +-i w with w = c (2/h) sin(k h/2) (2nd-order C-grid differences), so the
    Theta' standing wave is multiplied by Re P(i w dt) = 1 - (w dt)^2/2."""
    case, st, shape, eps, kw, h, Th0 = _acoustic_standing_wave(direction)
    o = erfo.Oracle(case)
    o.set_state(*st)
    pp, pi = erfo.eos(RD, CP, P00, Th0, Th0)
    c = np.sqrt(GAM * RD * pi * 300.0)          # c^2 = gamma Rd T
    w = c * (2.0 / h) * np.sin(kw * h / 2.0)
    dt = 0.4 * h / c / 2.0
    o.step(dt, 2)
    s1 = o.get_state()
    amp = ((s1[4] - Th0) * shape).sum() / (shape * shape).sum() / eps
    y = w * dt
    assert abs(amp - (1.0 - y * y / 2.0)) < 2e-6, (amp, 1 - y * y / 2)
    # the momentum picks up Im P = y - y^3/6 (pins the 1/3 and 1/2 separately from above)
    comp = {"x": 1, "y": 2, "z": 3}[direction]
    mom = s1[comp]
    sh = mom.shape
    kk, jj, ii = np.meshgrid(np.arange(sh[0]), np.arange(sh[1]), np.arange(sh[2]), indexing="ij")
    mm = {"x": ii, "y": jj, "z": kk}[direction]
    sshape = np.sin(kw * mm * h)
    mamp = (mom * sshape).sum() / (sshape * sshape).sum()
    # dU/dt = -c^2/theta dTheta'/dx: |U| = (c/theta) * eps * Im P
    expect = (c / 300.0) * eps * (y - y ** 3 / 6.0)
    assert abs(abs(mamp) - expect) < 2e-6 * expect + 1e-9 * eps, (mamp, expect)


# -------------------------------------------------------- Appendix A -------
@pytest.mark.parametrize("direction", ["x", "y"])
def test_horizontal_acoustic_substep_dispersion(direction):
    """App. A rows 1,2,4 (L585) with beta_d = 0: forward-backward scheme.  A
    Theta'' standing wave obeys T_{n+1} = (2 - mu^2) T_n - T_{n-1},
    mu = 2 (c dtau/h) sin(k h/2), T_1 = (1 - mu^2) T_0: neutral (|lambda| = 1)."""
    n, h = 16, 100.0
    dims = dict(x=2, y=2, z=3); dims[direction] = n
    case = uniform_case(dims["x"], dims["y"], dims["z"], h, h, h, beta_d=0.0)
    o = erfo.Oracle(case)
    st = zeros_state(case); st[0][:] = 1.0; st[4][:] = 300.0
    o.set_state(*st)
    pp, pi = erfo.eos(RD, CP, P00, 300.0, 300.0)
    c = np.sqrt(GAM * RD * pi * 300.0)
    nz, ny, nx = st[0].shape
    kk, jj, ii = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    m = {"x": ii, "y": jj}[direction]
    kw = 2 * np.pi * 2 / (n * h)
    shape = np.cos(kw * (m + 0.5) * h)
    dtau = 0.5 * h / c
    mu = 2.0 * (c * dtau / h) * np.sin(kw * h / 2.0)
    R = zeros_state(case)
    P = zeros_state(case)
    P[4][:] = 1e-3 * shape
    P[0][:] = 1e-3 * shape / 300.0
    T = [1.0, 1.0 - mu * mu]
    for s in range(2, 9):
        T.append((2.0 - mu * mu) * T[-1] - T[-2])
    for nsub in (1, 2, 5, 8):
        out = o.acoustic(dtau, nsub, R, P)
        amp = (out[4] * shape).sum() / (shape * shape).sum() / 1e-3
        assert abs(amp - T[nsub]) < 1e-12, (nsub, amp, T[nsub])
        assert np.abs(out[4] - amp * 1e-3 * shape).max() < 1e-14   # stays a pure mode


@pytest.mark.parametrize("beta_s", [0.1, 0.0, 0.3])
def test_vertical_acoustic_substep_dispersion(beta_s):
    """App. A rows 3-5 (L585) with the averaging of L591 and g = 0: with
    psi = Theta''/theta + i W''/c the substep is psi <- psi (1 + i a b1)/(1 - i a b2),
    a = c dtau (2/dz) sin(m dz/2), b1 = (1-beta_s)/2, b2 = (1+beta_s)/2 (L589);
    |lambda|^2 = (1 + a^2 b1^2)/(1 + a^2 b2^2) <= 1."""
    nz, h = 24, 50.0
    case = uniform_case(2, 2, nz, 100.0, 100.0, h, beta_d=0.0, beta_s=beta_s)
    o = erfo.Oracle(case)
    st = zeros_state(case); st[0][:] = 1.0; st[4][:] = 300.0
    o.set_state(*st)
    pp, pi = erfo.eos(RD, CP, P00, 300.0, 300.0)
    c = np.sqrt(GAM * RD * pi * 300.0)
    mz = 3 * np.pi / (nz * h)
    zc = (np.arange(nz) + 0.5) * h
    shape = np.cos(mz * zc)[:, None, None] * np.ones((nz, 2, 2))
    dtau = 1.7 * h / c                     # vertically implicit: stable beyond CFL 1
    a = c * dtau * (2.0 / h) * np.sin(mz * h / 2.0)
    b1, b2 = 0.5 * (1 - beta_s), 0.5 * (1 + beta_s)
    lam = (1 + 1j * a * b1) / (1 - 1j * a * b2)
    R = zeros_state(case)
    P = zeros_state(case)
    P[4][:] = 1e-3 * shape
    for nsub in (1, 2, 3, 7):
        out = o.acoustic(dtau, nsub, R, P)
        amp = (out[4] * shape).sum() / (shape * shape).sum() / 1e-3
        assert abs(amp - (lam ** nsub).real) < 1e-12, (nsub, amp, (lam ** nsub).real)
        # W'' = -(c/theta) Im(psi) sin(m z_face) up to the sign convention of the mode
        zf = np.arange(nz + 1) * h
        wshape = np.sin(mz * zf)[:, None, None] * np.ones((nz + 1, 2, 2))
        wamp = (out[3] * wshape).sum() / (wshape * wshape).sum() / 1e-3
        assert abs(abs(wamp) - abs((lam ** nsub).imag) * c / 300.0) < 1e-12
