"""The fp32 normal-quantile polynomial of the raster's guarded fast path (csrc/rng.cuh, c_z32[]) is the output of
csrc/z32_fit.py: this test re-runs the fit and compares it with the initialiser in the header, so the script beside the
kernels cannot drift from the constants the kernels use.  (The kernel's exactness does not rest on the fit: the guard band
is measured over all 2^32 words on the GPU, tests/test_gpu_fastpath.py.)"""
import importlib.util
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2203_02479_b200", "csrc")


def test_fit_reproduces_the_coefficients_in_rng_cuh():
    spec = importlib.util.spec_from_file_location("z32_fit", os.path.join(CSRC, "z32_fit.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mono, err = mod.fit()
    fitted = mono.astype(np.float32)[::-1]  # highest power first, as in the header
    src = open(os.path.join(CSRC, "rng.cuh")).read()
    m = re.search(r"c_z32\[9\]\s*=\s*\{([^}]*)\}", src)
    assert m, "c_z32[9] initialiser not found in rng.cuh"
    header = np.array([np.float32(t.strip().rstrip("f")) for t in m.group(1).split(",")], dtype=np.float32)
    assert header.shape == (9,) and err < 2e-7
    # the same fp32 numbers; a least-squares solver of another LAPACK build may move the smallest coefficients by an ulp
    # or two, which the tolerance allows (the polynomial's value changes by < 1e-9 then)
    assert np.allclose(fitted, header, rtol=1e-5, atol=0.0), (fitted, header)
    d = np.linspace(-2.5, 2.5, 1001)
    assert np.max(np.abs(np.polyval(fitted.astype(np.float64), d) - np.polyval(header.astype(np.float64), d))) < 1e-8
