"""The C-ABI boundary without a GPU: liberf_b200.so builds, loads, exports every symbol
include/erf_b200.h declares, validates arguments before touching CUDA, and the Python
binding refuses to run without a device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2412_04395_b200 import binding as B
from paper_2412_04395_b200 import workloads as wl
from util import field_errors

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2412_04395_b200 import build
    build.build()
    return B.load()


def _declared():
    names = set()
    for fn in os.listdir(os.path.join(ROOT, "include")):
        if not fn.endswith(".h"):
            continue
        src = open(os.path.join(ROOT, "include", fn)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(erf_[a-z0-9_]+)\s*\(", src))
    return names


def test_every_declared_symbol_is_exported(lib):
    decl = _declared()
    assert {"erf_create", "erf_set_state", "erf_rk3_step", "erf_get_state", "erf_destroy"} <= decl
    for name in decl:
        assert hasattr(lib, name), name
    assert decl == set(B.EXPORTS)


def test_struct_layouts_match_header():
    # field order and C types as in include/erf_b200.h (natural alignment on both sides)
    assert [f[0] for f in B.erf_grid._fields_] == ["nx", "ny", "nz", "dx", "dy", "periodic_x", "periodic_y"]
    assert C.sizeof(B.erf_grid) == 40
    assert C.sizeof(B.erf_metrics) == 40
    assert C.sizeof(B.erf_params) == 144  # 4 doubles, 3 ints padded to 16, 6 doubles, 2 ints, 2 doubles, int (padded), 2 doubles
    hdr = open(os.path.join(ROOT, "include", "erf_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    body = hdr[hdr.index("typedef struct {", hdr.index("erf_metrics;")):hdr.index("} erf_params;")]
    order = re.findall(r"\b(Rd|cp|g|p00|adv_order_h|adv_order_v|diffusion|nu|alpha_theta|Cs|Pr_t|beta_s|beta_d|substep_mode|scalar_adv|ray_depth|ray_coef|ray_fields|ray_uref|ray_vref)\b[,;]", body)
    assert order == [f[0] for f in B.erf_params._fields_]


def test_strerror(lib):
    for code in (0, -1, -2, -3, -4, -99):
        s = lib.erf_strerror(code)
        assert isinstance(s, bytes) and len(s) > 0
    assert lib.erf_strerror(0) == b"ok"


def _args(case, periodic=(1, 1)):
    g = B.erf_grid(case["nx"], case["ny"], case["nz"], case["dx"], case["dy"], *periodic)
    zl = np.ascontiguousarray(case["z_levels"])
    r0 = np.ascontiguousarray(case["rho0"])
    t0 = np.ascontiguousarray(case["rhotheta0"])
    m = B.erf_metrics(None, zl.ctypes.data, r0.ctypes.data, t0.ctypes.data, 1)
    return g, m, B.make_params(case["params"]), (zl, r0, t0)


def test_create_validates_before_cuda(lib):
    case = wl.make_case(1, nx=4, ny=4, nz=4, with_state=False)
    g, m, p, keep = _args(case)
    h = C.c_void_p()
    assert lib.erf_create(None, C.byref(m), C.byref(p), None, C.byref(h)) == B.ERF_EINVAL
    assert lib.erf_create(C.byref(g), C.byref(m), C.byref(p), None, None) == B.ERF_EINVAL
    bad = dict(case["params"]); bad["ray_fields"] = 16
    assert lib.erf_create(C.byref(g), C.byref(m), C.byref(B.make_params(bad)), None, C.byref(h)) == B.ERF_EINVAL
    bad = dict(case["params"]); bad["adv_order_h"] = 7
    assert lib.erf_create(C.byref(g), C.byref(m), C.byref(B.make_params(bad)), None, C.byref(h)) == B.ERF_EINVAL
    g3 = B.erf_grid(0, 4, 4, 1.0, 1.0, 1, 1)
    assert lib.erf_create(C.byref(g3), C.byref(m), C.byref(p), None, C.byref(h)) == B.ERF_EINVAL
    m2 = B.erf_metrics(None, None, m.rho0, m.rhotheta0, 1)
    assert lib.erf_create(C.byref(g), C.byref(m2), C.byref(p), None, C.byref(h)) == B.ERF_EINVAL
    assert not h.value


def test_null_context_calls(lib):
    assert lib.erf_rk3_step(None, 1.0, 6, None) == B.ERF_EINVAL
    assert lib.erf_set_state(None, None, None, None, None, None, None) == B.ERF_EINVAL
    assert lib.erf_get_state(None, None, None, None, None, None, None) == B.ERF_EINVAL
    assert lib.erf_set_path(None, 0) == B.ERF_EINVAL
    assert lib.erf_launch_count(None) == 0
    lib.erf_destroy(None)  # no-op


def test_no_cpu_fallback(lib):
    """Without a CUDA device the product path must fail loudly."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    case = wl.make_case(1, nx=4, ny=4, nz=4, with_state=False)
    g, m, p, keep = _args(case)
    h = C.c_void_p()
    assert lib.erf_create(C.byref(g), C.byref(m), C.byref(p), None, C.byref(h)) == B.ERF_ECUDA
    with pytest.raises(RuntimeError):
        B.Dycore(case)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2412_04395_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), fn
                for word in ("erfo", "erf_oracle", "liberf_oracle"):
                    assert word not in src, (fn, word)


def test_field_error_norm():
    a = [np.ones((2, 2, 2)) * s for s in (1.0, 10.0, 1.0, 0.1, 300.0)]
    b = [x.copy() for x in a]
    b[3] = b[3] + 1e-3
    e = field_errors(b, a)
    assert e[0] == 0 and e[4] == 0
    assert abs(e[3] - 1e-4) < 1e-12  # W error is measured against the shared momentum scale (10)
