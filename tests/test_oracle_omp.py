"""The optional OpenMP build of the oracle (same source, -fopenmp; used only for the long GPU parity runs) must
give the serial build's results bit for bit: no loop of the step carries a reduction."""
import numpy as np
import pytest

from oracle import erfo
from paper_2412_04395_b200 import workloads as wl


def _run(case, steps):
    o = erfo.Oracle(case)
    o.set_state(*case["state"])
    for _ in range(steps):
        o.step(case["dt"], case["ns"])
    out = o.get_state()
    o.close()
    return out


@pytest.mark.parametrize("cfg,kw,steps", [(1, dict(), 1), (2, dict(nx=48, ny=40, nz=64), 3),
                                          (3, dict(nx=24, ny=36, nz=40), 2), (4, dict(nx=28, ny=20, nz=96), 2)])
def test_openmp_build_is_bitwise_the_serial_build(cfg, kw, steps):
    case = wl.make_case(cfg, **kw)
    try:
        erfo.use_openmp(False)
        a = _run(case, steps)
        erfo.use_openmp(True)
        b = _run(case, steps)
    finally:
        erfo.use_openmp(False)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
