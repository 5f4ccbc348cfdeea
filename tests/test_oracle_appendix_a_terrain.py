"""Appendix A over terrain: the rho'' and Theta'' equations of one acoustic substep (PAPER.md L585 rows 4-5 with the
off-centred average of L589-L591), checked as residuals on the oracle's own inputs and outputs.

The test rebuilds everything the two equations contain with numpy from the node heights (L178) and the arrays that go
in and come out of `acoustic(dtau, 1, R, S'')`:
    Omega'' = W'' - sxw avg4(U'') - syw avg4(V'')   (zero on both lids)             -- the flux through a zeta-surface
    rho''new   = rho''old   + dtau [ R_rho   - D_h(U''new, V''new)          - d_zeta(b2 Omega''new + b1 Omega''old) / hc ]
    Theta''new = Theta''old + dtau [ R_Theta - D_h(theta U''new, theta V''new) - d_zeta(theta_f (b2 Omega''new + b1 Omega''old)) / hc ]
    D_h(F, G) = [ d_x(hx F) / dx + d_y(hy G) / dy ] / hc,   b1 = (1 - beta_s)/2, b2 = (1 + beta_s)/2
The definition of Omega is the one the slow continuity equation uses, and that one is fixed by free-stream preservation
over terrain (a uniform Cartesian wind has zero divergence only with the four-point means and these face heights:
tests/test_oracle_pins.py).  So the residuals pin, in the substep, the SIZE and the averaging of the explicit slope part
omega of W'' (reading G16), the face heights hx / hy in the horizontal divergence, the beta weights on old and new
Omega'' and the lids -- none of which a flat column can see."""
import numpy as np
import pytest

from test_oracle_symmetry import _problem, _state

TOL = 1e-12  # of the largest term of the equation


def _geometry(zn, dx, dy):
    zxf = 0.5 * (zn[:, :-1, :] + zn[:, 1:, :])            # centres of x-faces: [nz+1][ny][nx+1]
    zyf = 0.5 * (zn[:, :, :-1] + zn[:, :, 1:])            # centres of y-faces: [nz+1][ny+1][nx]
    zw = 0.25 * (zn[:, :-1, :-1] + zn[:, :-1, 1:] + zn[:, 1:, :-1] + zn[:, 1:, 1:])
    hx = (zxf[1:] - zxf[:-1])[:, :, :-1]                  # thickness of the low-x face of cell i
    hy = (zyf[1:] - zyf[:-1])[:, :-1, :]
    hc = zw[1:] - zw[:-1]
    sxw = (zxf[:, :, 1:] - zxf[:, :, :-1]) / dx           # slope of the w-face, [nz+1][ny][nx]
    syw = (zyf[:, 1:, :] - zyf[:, :-1, :]) / dy
    return hx, hy, hc, sxw, syw


def _xp(a):
    return np.roll(a, -1, axis=2)


def _yp(a):
    return np.roll(a, -1, axis=1)


def _omega(U, V, W, sxw, syw):
    Om = np.zeros_like(W)
    ubar = 0.25 * (U[:-1] + _xp(U)[:-1] + U[1:] + _xp(U)[1:])
    vbar = 0.25 * (V[:-1] + _yp(V)[:-1] + V[1:] + _yp(V)[1:])
    Om[1:-1] = W[1:-1] - sxw[1:-1] * ubar - syw[1:-1] * vbar
    return Om


@pytest.mark.parametrize("order,beta_s", [(5, 0.1), (3, 0.3), (2, 0.0)])
def test_continuity_and_theta_equations_of_a_substep_over_terrain(oracle_lib, order, beta_s):
    erfo = oracle_lib
    case, st = _problem(True, order, seed=90 + order)
    case["params"]["beta_s"] = beta_s
    dx, dy = case["dx"], case["dy"]
    hx, hy, hc, sxw, syw = _geometry(case["z_nodes"], dx, dy)
    assert np.abs(sxw).max() > 0.05 and np.abs(syw).max() > 0.05
    o = erfo.Oracle(case)
    o.set_state(*st)
    S = o.get_state()
    theta = S[4] / S[0]
    R = o.slow_rhs()
    P0 = [0.01 * a for a in _state(case, seed=91)]
    P0[3][0] = P0[3][-1] = 0.0
    dtau = case["dt"] / case["ns"]
    P1 = o.acoustic(dtau, 1, R, P0)
    o.close()
    b1, b2 = 0.5 * (1.0 - beta_s), 0.5 * (1.0 + beta_s)
    Om = b2 * _omega(P1[1], P1[2], P1[3], sxw, syw) + b1 * _omega(P0[1], P0[2], P0[3], sxw, syw)
    assert np.abs(P1[3][1:-1] - Om[1:-1]).max() > 1e-3 * np.abs(P1[3]).max()  # the slope part is not negligible here
    Un, Vn = P1[1], P1[2]
    FU, FV = hx * Un, hy * Vn
    thx = 0.5 * (np.roll(theta, 1, axis=2) + theta)
    thy = 0.5 * (np.roll(theta, 1, axis=1) + theta)
    thf = np.zeros_like(Om)
    thf[1:-1] = 0.5 * (theta[:-1] + theta[1:])
    terms_r = [(_xp(FU) - FU) / dx / hc, (_yp(FV) - FV) / dy / hc, (Om[1:] - Om[:-1]) / hc]
    terms_T = [(_xp(FU * thx) - FU * thx) / dx / hc, (_yp(FV * thy) - FV * thy) / dy / hc,
               (thf[1:] * Om[1:] - thf[:-1] * Om[:-1]) / hc]
    res_r = P1[0] - P0[0] - dtau * (R[0] - sum(terms_r))
    res_T = P1[4] - P0[4] - dtau * (R[4] - sum(terms_T))
    scale_r = dtau * max(np.abs(t).max() for t in terms_r)
    scale_T = dtau * max(np.abs(t).max() for t in terms_T)
    assert np.abs(res_r).max() <= TOL * scale_r, np.abs(res_r).max() / scale_r
    assert np.abs(res_T).max() <= TOL * scale_T, np.abs(res_T).max() / scale_T
