"""erf_poisson_modes_noalloc, the one entry point of liberf_b200.so that never allocates device memory.

Why it exists: some users of the library run where a cudaMalloc is not theirs to make -- inside an application whose
own allocator has taken the whole GPU, under a memory budget their own buffers fill, or in a loop that cannot take the
device-wide synchronisation an allocation costs.  They pass their own input and output arrays; the solver's work space
(one double per mode and level) is a fixed 8 MiB array built into the library, which is why the problem size is capped
(ERF_NOALLOC_MAX_VALUES), why every call on a GPU shares that array, and why this file checks two calls IN A ROW: the
second call starts with the first call's leftovers in the work space and must not care.

The check is against the path that already exists: erf_project on a context (cudaMalloc'ed work arrays) leaves
p' = psi after one projection from p' = 0.  The new entry point is only the middle of that projection -- the tridiagonal
solve per horizontal Fourier mode -- so the test does the plumbing around it with numpy (divergence of the momenta, fft2
per level before, ifft2 after) and compares psi with the tolerance the anelastic parity test uses for p'.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests."""
import ctypes as C

import numpy as np
import pytest

from paper_2412_04395_b200 import workloads as wl

TOL_PSI = 1e-10  # relative to max |psi|: the bound tests/test_gpu_parity.py puts on p' after erf_project


@pytest.fixture(scope="module")
def B():
    from paper_2412_04395_b200 import binding, build
    build.build()
    binding.load()
    return binding


def _problem(cfg, seed, stretch, **kw):
    """A flat periodic case with momenta far from divergence-free (the recipe of test_anelastic_mode_matches_oracle)."""
    case = wl.make_case(cfg, **kw)
    nz, ny, nx = case["nz"], case["ny"], case["nx"]
    if stretch != 1.0:
        dz = np.diff(case["z_levels"])[0] * stretch ** np.arange(nz)
        case["z_levels"] = np.concatenate([[0.0], np.cumsum(dz)])
    rng = np.random.default_rng(seed)
    rho0 = np.broadcast_to(case["rho0"][:, None, None], (nz, ny, nx)).copy()
    st = [rho0, case["state"][1] + 0.5 * rng.standard_normal((nz, ny, nx)),
          case["state"][2] + 0.5 * rng.standard_normal((nz, ny, nx)), 0.3 * rng.standard_normal((nz + 1, ny, nx)),
          case["state"][4].copy()]
    st[3][0] = st[3][-1] = 0.0
    return case, st, 4.0 * case["dt"]


def _psi_existing_path(torch, B, case, st, dt):
    d = B.Dycore(case)
    d.set_state(*[torch.as_tensor(np.ascontiguousarray(a)).cuda() for a in st])
    d.project(dt)
    psi = d.pprime().cpu().numpy()
    d.close()
    return psi


def _psi_no_alloc(torch, B, case, st, dt):
    """Geometry, divergence and the transforms on the host; the solve through the entry point under test."""
    zl = np.asarray(case["z_levels"], dtype=np.float64)
    dz = np.diff(zl)
    zc = 0.5 * (zl[:-1] + zl[1:])
    dzw = np.zeros(case["nz"] + 1)
    dzw[1:-1] = zc[1:] - zc[:-1]
    U, V, W = st[1], st[2], st[3]
    div = ((np.roll(U, -1, axis=2) - U) / case["dx"] + (np.roll(V, -1, axis=1) - V) / case["dy"]
           + (W[1:] - W[:-1]) / dz[:, None, None])
    hat = np.fft.fft2(div, axes=(1, 2))
    re = torch.as_tensor(np.ascontiguousarray(hat.real)).cuda()
    im = torch.as_tensor(np.ascontiguousarray(hat.imag)).cuda()
    B.erf_poisson_modes_noalloc(case["nx"], case["ny"], case["nz"], case["dx"], case["dy"], dt,
                                torch.as_tensor(dz).cuda(), torch.as_tensor(dzw).cuda(), re, im)
    torch.cuda.synchronize()
    sol = re.cpu().numpy() + 1j * im.cpu().numpy()
    back = np.fft.ifft2(sol, axes=(1, 2))
    assert np.abs(back.imag).max() <= 1e-12 * np.abs(back.real).max()  # a real psi: the modes come in conjugate pairs
    return back.real, (re.cpu().numpy(), im.cpu().numpy())


@pytest.mark.gpu
def test_no_alloc_solve_matches_erf_project_on_two_calls_in_a_row(B):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    # two different problems back to back (different sizes, one stretched, one at the size limit's scale in x-y), then
    # the first again: each call finds the previous call's c' in the shared work space
    probs = [_problem(3, 901, 1.05, nx=48, ny=20, nz=33), _problem(2, 902, 1.0, nx=64, ny=32, nz=17)]
    refs = [_psi_existing_path(torch, B, *p) for p in probs]
    raw = []
    for p, ref in list(zip(probs, refs)) + [(probs[0], refs[0])]:
        psi, hat = _psi_no_alloc(torch, B, *p)
        raw.append(hat)
        assert np.abs(ref).max() > 0.0
        err = np.abs(psi - ref).max() / np.abs(ref).max()
        assert err <= TOL_PSI, err
    # same inputs, different leftovers in the work space: bit-identical output
    assert np.array_equal(raw[0][0], raw[2][0]) and np.array_equal(raw[0][1], raw[2][1])


@pytest.mark.gpu
def test_no_alloc_solve_at_the_size_limit(B):
    """nx*ny*nz == ERF_NOALLOC_MAX_VALUES exactly (128 x 128 x 64) runs and still matches the existing path."""
    import torch
    p = _problem(2, 903, 1.0, nx=128, ny=128, nz=64)
    assert p[0]["nx"] * p[0]["ny"] * p[0]["nz"] == B.ERF_NOALLOC_MAX_VALUES
    ref = _psi_existing_path(torch, B, *p)
    psi, _ = _psi_no_alloc(torch, B, *p)
    assert np.abs(psi - ref).max() <= TOL_PSI * np.abs(ref).max()


def test_no_alloc_entry_point_refuses_bad_sizes_before_touching_cuda(B):
    """No GPU needed: a null array or a non-positive size is ERF_EINVAL, one value more than the built-in work space
    holds is ERF_ETOOLARGE -- both decided before the first CUDA call, so the dummy addresses are never used."""
    lib = B.load()
    f = lib.erf_poisson_modes_noalloc
    dummy = C.c_void_p(256)
    ok = (dummy, dummy, dummy, dummy, None)
    assert f(8, 8, 8, 1.0, 1.0, 1.0, None, dummy, dummy, dummy, None) == B.ERF_EINVAL
    assert f(8, 8, 8, 1.0, 1.0, 1.0, dummy, dummy, dummy, None, None) == B.ERF_EINVAL
    assert f(0, 8, 8, 1.0, 1.0, 1.0, *ok) == B.ERF_EINVAL
    assert f(8, 8, 8, 1.0, 1.0, 0.0, *ok) == B.ERF_EINVAL
    assert f(8, 8, 8, -1.0, 1.0, 1.0, *ok) == B.ERF_EINVAL
    assert f(128, 128, 65, 1.0, 1.0, 1.0, *ok) == B.ERF_ETOOLARGE
    assert f(B.ERF_NOALLOC_MAX_VALUES + 1, 1, 1, 1.0, 1.0, 1.0, *ok) == B.ERF_ETOOLARGE
    assert f(2 ** 31 - 1, 2 ** 31 - 1, 2 ** 31 - 1, 1.0, 1.0, 1.0, *ok) == B.ERF_ETOOLARGE  # no wrap-around
    assert b"ERF_NOALLOC_MAX_VALUES" in lib.erf_strerror(B.ERF_ETOOLARGE)
