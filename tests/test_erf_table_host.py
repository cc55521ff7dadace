"""The raster's own fp64 erf (csrc/erf_table.cuh: 48 intervals of width 1/8, degree-12 Taylor polynomials from erf's ODE)
evaluated on the HOST through wcsim_debug_erf -- the same code the kernels run -- against scipy's erf and the printed
values of Abramowitz & Stegun Table 7.1 (tests/golden/erf_table.txt).  No device is touched."""
import shutil

import numpy as np
import pytest
from conftest import golden

pytestmark = pytest.mark.skipif(shutil.which("nvcc") is None, reason="nvcc not on PATH")


def test_table_erf_matches_library_erf_everywhere():
    from scipy.special import erf
    from paper_2203_02479_b200 import binding as B
    rng = np.random.default_rng(3)
    z = np.concatenate([rng.uniform(-6.5, 6.5, 400_000), rng.normal(0, 1.5, 200_000),
                        np.arange(-48, 49) * 0.125,                      # interval boundaries
                        np.nextafter(np.arange(1, 49) * 0.125, -np.inf),  # just below them
                        [0.0, -0.0, 1e-300, -1e-300, 5.99999, 6.0, 7.0, 30.0, -30.0, 1e300, -1e300]])
    got = B.wcsim_debug_erf(z)
    ref = erf(z)
    assert np.max(np.abs(got - ref)) <= 2.3e-16          # one ulp of 1
    tiny = np.abs(z) < 1e-200                            # bin weights are differences of erf values: the absolute error
    assert np.max(np.abs(got[tiny])) <= 3e-17            # is what matters, so erf(0) need not be exactly 0
    assert np.all(np.abs(got) <= 1.0)
    nz = z != 0.0
    assert np.array_equal(got[nz], -B.wcsim_debug_erf(-z[nz]))   # odd


def test_table_erf_has_no_jump_at_interval_boundaries():
    from paper_2203_02479_b200 import binding as B
    for k in range(1, 48):
        x = k * 0.125
        pts = np.array([np.nextafter(x, -np.inf), x, np.nextafter(x, np.inf)])
        v = B.wcsim_debug_erf(pts)
        assert abs(v[1] - v[0]) <= 2.3e-16 and abs(v[2] - v[1]) <= 2.3e-16  # at most one ulp of 1 where the polynomial changes


def test_table_erf_reproduces_printed_values():
    from paper_2203_02479_b200 import binding as B
    rows = golden("erf_table.txt")
    x = np.array([float(r[0]) for r in rows])
    want = np.array([float(r[1]) for r in rows])
    assert np.max(np.abs(B.wcsim_debug_erf(x) - want)) <= 6e-11  # ten printed decimals
