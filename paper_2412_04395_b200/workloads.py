"""Seeded synthetic workloads (inputs only -- none of the method's arithmetic).

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU
oracle's tests: it produces plain numpy data (grid, base state, initial state,
parameters) for the five configurations of BASELINE.json and for arbitrary
small variants of them.  The recipe is the one stated in DESIGN.md
("Input recipe") after SURVEY.md 8(d):

* constants Rd=287, cp=1004.5, g=9.81, P00 = surface pressure = 1e5 Pa
  (PAPER.md L82);
* base state = closed-form continuous hydrostatic profile for a piecewise-linear
  theta0(z), evaluated at the cell-centre heights (the base state is data for
  the library; PAPER.md L227 describes ERF's own Newton-Raphson variant);
* initial rho = rho0, Theta = rho0 (theta0 + theta'), U = rho_u (u0 + u'),
  V = rho_v (v0 + v'), W = 0 (the library imposes the lids);
* noise from numpy.random.default_rng(seed) (PCG64), drawn level by level in
  [k][j][i] order, theta' first, then u', then v'.

No public dataset is involved; shapes follow the paper's LES / terrain set-ups
(Table C1).
"""
from __future__ import annotations

import copy

import numpy as np

RD, CP, GRAV, P00 = 287.0, 1004.5, 9.81, 1.0e5

DEFAULT_PARAMS = dict(Rd=RD, cp=CP, g=GRAV, p00=P00, adv_order_h=2, adv_order_v=2, diffusion=0,
                      nu=0.0, alpha_theta=0.0, Cs=0.18, Pr_t=1.0, beta_s=0.1, beta_d=0.1,
                      substep_mode=1, scalar_adv=0)


def hydrostatic_base(z, layers):
    """theta0, rho0 at heights ``z`` (any shape) for a piecewise-linear theta0.

    ``layers`` = [(z_bottom, lapse_rate), ...] ascending, first z_bottom = 0, with
    theta0(0) = layers_theta_surface given as the third element of the first tuple:
    [(0.0, gamma0, theta_surface), (z1, gamma1), ...].
    """
    z = np.asarray(z, dtype=np.float64)
    theta = np.empty_like(z)
    pi = np.empty_like(z)
    zb, gam, th_b = layers[0]
    pi_b = 1.0  # surface pressure = P00
    bounds = [l[0] for l in layers[1:]] + [np.inf]
    for n, top in enumerate(bounds):
        gam = layers[n][1]
        sel = (z >= zb) & (z < top) if n > 0 else (z < top)
        dz = z[sel] - zb
        th = th_b + gam * dz
        theta[sel] = th
        if gam == 0.0:
            pi[sel] = pi_b - GRAV * dz / (CP * th_b)
        else:
            pi[sel] = pi_b - GRAV / (CP * gam) * np.log(th / th_b)
        if np.isfinite(top):
            dzt = top - zb
            th_t = th_b + gam * dzt
            pi_b = (pi_b - GRAV * dzt / (CP * th_b)) if gam == 0.0 else (
                pi_b - GRAV / (CP * gam) * np.log(th_t / th_b))
            th_b, zb = th_t, top
    rho = P00 * pi ** ((CP - RD) / RD) / (RD * theta)
    return theta, rho


def _levels_uniform(nz, dz):
    return np.arange(nz + 1, dtype=np.float64) * dz


def _levels_stretched(nz, dz0, ratio, dzmax):
    dz = np.minimum(dz0 * ratio ** np.arange(nz, dtype=np.float64), dzmax)
    return np.concatenate([[0.0], np.cumsum(dz)])


def gaussian_hill_nodes(nx, ny, dx, dy, z_levels, height, halfwidth, xc=None, yc=None,
                        i0=0, j0=0):
    """Node heights [(nz+1)][(ny+1)][(nx+1)] over h = height*exp(-r^2/a^2) with
    basic-terrain-following decay z = zeta + h (1 - zeta/z_top)."""
    x = (np.arange(nx + 1) + i0) * dx
    y = (np.arange(ny + 1) + j0) * dy
    h = height * np.exp(-(((x[None, :] - xc) ** 2 + (y[:, None] - yc) ** 2) / halfwidth ** 2))
    zt = z_levels[-1]
    return z_levels[:, None, None] + h[None, :, :] * (1.0 - z_levels[:, None, None] / zt)


def cell_centre_heights(z_nodes):
    zw = 0.25 * (z_nodes[:, :-1, :-1] + z_nodes[:, :-1, 1:] + z_nodes[:, 1:, :-1] + z_nodes[:, 1:, 1:])
    return 0.5 * (zw[:-1] + zw[1:])


# name -> recipe; sizes may be overridden in make_case (crops / small variants)
CONFIGS = {
    1: dict(nx=32, ny=32, nz=32, dx=100.0, dy=100.0, dz=100.0, seed=1001,
            layers=[(0.0, 0.0, 300.0)], u0=10.0, v0=0.0,
            noise=dict(kind="uniform", theta=0.5, uv=0.1, below=np.inf),
            params=dict(adv_order_h=2, adv_order_v=2, diffusion=0),
            dt=0.5, ns=6, steps=1),
    2: dict(nx=128, ny=128, nz=64, dx=50.0, dy=50.0, dz=20.0, seed=1002,
            layers=[(0.0, 0.003, 300.0)], u0=8.0, v0=2.0,
            noise=dict(kind="normal", theta=0.2, uv=0.0, below=400.0),
            params=dict(adv_order_h=5, adv_order_v=5, diffusion=1, nu=1.0, alpha_theta=1.0),
            dt=0.25, ns=6, steps=20),
    3: dict(nx=256, ny=256, nz=128, dx=10.0, dy=10.0, dz=10.0, seed=1003,
            layers=[(0.0, 0.0, 300.0), (500.0, 0.008)], u0=10.0, v0=0.0,
            noise=dict(kind="uniform", theta=0.1, uv=0.0, below=200.0),
            params=dict(adv_order_h=3, adv_order_v=3, diffusion=2, Cs=0.18),
            dt=0.1, ns=6, steps=100),
    4: dict(nx=512, ny=512, nz=96, dx=100.0, dy=100.0, seed=1004,
            stretch=dict(dz0=20.0, ratio=1.03, dzmax=200.0),
            hill=dict(height=400.0, halfwidth=1000.0),
            layers=[(0.0, 0.003, 300.0)], u0=10.0, v0=0.0,
            noise=None,
            params=dict(adv_order_h=5, adv_order_v=5, diffusion=2, Cs=0.18),
            dt=0.5, ns=8, steps=50),
    5: dict(nx=1024, ny=1024, nz=128, dx=5.0, dy=5.0, dz=5.0, seed=1005,
            layers=[(0.0, 0.01, 265.0)], u0=8.0, v0=0.0,
            noise=dict(kind="uniform", theta=0.25, uv=0.0, below=50.0),
            params=dict(adv_order_h=5, adv_order_v=5, diffusion=2, Cs=0.18),
            dt=0.05, ns=6, steps=20),
}


def make_case(config, nx=None, ny=None, nz=None, seed=None, params=None, hill_center=None,
              with_state=True):
    """Build one workload.  ``config`` in 1..5; nx/ny/nz override the size (same
    spacing, time step, parameters and noise recipe), ``params`` overrides
    entries of the parameter struct.  Returns a dict of plain numpy data."""
    r = copy.deepcopy(CONFIGS[config])
    nx = nx or r["nx"]
    ny = ny or r["ny"]
    nz = nz or r["nz"]
    seed = r["seed"] if seed is None else seed
    par = dict(DEFAULT_PARAMS)
    par.update(r["params"])
    if params:
        par.update(params)
    case = dict(name=f"cfg{config}_{nx}x{ny}x{nz}", config=config, nx=nx, ny=ny, nz=nz,
                dx=r["dx"], dy=r["dy"], dt=r["dt"], ns=r["ns"], steps=r["steps"], params=par,
                z_nodes=None, z_levels=None)
    if "stretch" in r:
        zl = _levels_stretched(nz, **r["stretch"])
    else:
        zl = _levels_uniform(nz, r["dz"])
    if "hill" in r:
        xc, yc = hill_center if hill_center else (0.5 * nx * r["dx"], 0.5 * ny * r["dy"])
        zn = gaussian_hill_nodes(nx, ny, r["dx"], r["dy"], zl, r["hill"]["height"],
                                 r["hill"]["halfwidth"], xc, yc)
        # periodic closure: the hill is ~0 at the boundary; make it exact
        zn[:, :, -1] = zn[:, :, 0]
        zn[:, -1, :] = zn[:, 0, :]
        case["z_nodes"] = zn
        zc = cell_centre_heights(zn)                      # [nz][ny][nx]
    else:
        case["z_levels"] = zl
        zc = 0.5 * (zl[:-1] + zl[1:])                     # [nz]
    theta0, rho0 = hydrostatic_base(zc, r["layers"])
    case["rho0"] = rho0
    case["rhotheta0"] = rho0 * theta0
    if not with_state:
        return case
    shape = (nz, ny, nx)
    rng = np.random.default_rng(seed)
    zc3 = zc if zc.ndim == 3 else np.broadcast_to(zc[:, None, None], shape)
    th_p = np.zeros(shape)
    u_p = np.zeros(shape)
    v_p = np.zeros(shape)
    nz_spec = r["noise"]
    if nz_spec is not None:
        # levels that can carry noise (flat grids: a prefix of the levels)
        kmax = nz if not np.isfinite(nz_spec["below"]) else int(
            np.searchsorted(zc3.min(axis=(1, 2)), nz_spec["below"]))
        mask = zc3[:kmax] < nz_spec["below"]

        def draw(amp):
            if amp == 0.0:
                return np.zeros((kmax, ny, nx))
            if nz_spec["kind"] == "uniform":
                return rng.uniform(-amp, amp, size=(kmax, ny, nx))
            return rng.normal(0.0, amp, size=(kmax, ny, nx))

        th_p[:kmax] = draw(nz_spec["theta"]) * mask
        u_p[:kmax] = draw(nz_spec["uv"]) * mask
        v_p[:kmax] = draw(nz_spec["uv"]) * mask
    rho0_3 = rho0 if rho0.ndim == 3 else np.broadcast_to(rho0[:, None, None], shape)
    th0_3 = theta0 if theta0.ndim == 3 else np.broadcast_to(theta0[:, None, None], shape)
    rho = np.array(rho0_3, dtype=np.float64)
    rho_u = 0.5 * (rho + np.roll(rho, 1, axis=2))
    rho_v = 0.5 * (rho + np.roll(rho, 1, axis=1))
    case["state"] = [rho, rho_u * (r["u0"] + u_p), rho_v * (r["v0"] + v_p),
                     np.zeros((nz + 1, ny, nx)), rho * (th0_3 + th_p)]
    return case


def window(case, i0, j0, wx, wy, state=None):
    """Cut a wx-by-wy column window (periodic wrap of indices) out of ``case``:
    same spacing / parameters, base state and node heights restricted to the
    window.  Used to check full-size GPU results against the oracle on sampled
    outputs: after one step the window's central region is independent of the
    (wrong) periodic closure at the window's own edges."""
    nx, ny = case["nx"], case["ny"]
    ii = (i0 + np.arange(wx)) % nx
    jj = (j0 + np.arange(wy)) % ny
    sub = {k: v for k, v in case.items() if k not in ("state", "z_nodes", "rho0", "rhotheta0")}
    sub.update(nx=wx, ny=wy, name=f"{case['name']}_win{i0}_{j0}_{wx}x{wy}")
    if case.get("z_nodes") is not None:
        ii1 = (i0 + np.arange(wx + 1)) % nx
        jj1 = (j0 + np.arange(wy + 1)) % ny
        sub["z_nodes"] = np.ascontiguousarray(case["z_nodes"][:, jj1][:, :, ii1])
    else:
        sub["z_nodes"] = None
    for key in ("rho0", "rhotheta0"):
        a = case[key]
        sub[key] = a if a.ndim == 1 else np.ascontiguousarray(a[:, jj][:, :, ii])
    st = state if state is not None else case.get("state")
    if st is not None:
        sub["state"] = [np.ascontiguousarray(a[:, jj][:, :, ii]) for a in st]
    return sub
