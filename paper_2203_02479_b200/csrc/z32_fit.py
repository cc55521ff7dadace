"""Coefficients of the fp32 estimate of the normal quantile used by the raster's guarded fast path (csrc/rng.cuh,
z32_from_word): Phi^-1(u) = x g(wl) with x = 2u - 1, wl = -ln(1 - x^2), g a polynomial in (wl - 2.5) on 0 <= wl <= 5.

    python paper_2203_02479_b200/csrc/z32_fit.py        # prints the C initialiser of c_z32[]

The fit is a Lawson-reweighted least-squares approximation of the relative error against scipy's ndtri.  Nothing here is
trusted by the kernel: the guard band of the fast path uses the error of the fp32 routine measured exhaustively against
the device's own fp64 AS 241 routine over all 2^32 words (wcsim_debug_z32_scan, tests/test_gpu_fastpath.py).
"""
import numpy as np
from numpy.polynomial import chebyshev as C, polynomial as P
from scipy.special import erfinv

W0, DEG = 5.0, 8


def fit():
    n = 4000
    wl = 0.5 * W0 * (1 - np.cos(np.pi * (np.arange(n) + 0.5) / n))
    x = np.sqrt(-np.expm1(-wl))
    g = np.sqrt(2.0) * erfinv(x) / x
    tt = 2 * wl / W0 - 1
    wts = np.ones(n)
    best = None
    for _ in range(200):
        c = C.chebfit(tt, g, DEG, w=np.sqrt(wts) / g)
        err = np.abs(C.chebval(tt, c) - g) / g
        if best is None or err.max() < best[1]:
            best = (c, err.max())
        wts = wts * (err / err.max() + 1e-3)
        wts /= wts.sum()
    c, e = best
    # Chebyshev in tt = (wl - W0/2) / (W0/2)  ->  monomial in d = wl - W0/2
    mono = C.cheb2poly(c) / (0.5 * W0) ** np.arange(DEG + 1)
    return mono, e


if __name__ == "__main__":
    mono, e = fit()
    wl = np.linspace(1e-9, W0, 400001)
    x = np.sqrt(-np.expm1(-wl))
    g = np.sqrt(2.0) * erfinv(x) / x
    m32 = mono.astype(np.float32).astype(np.float64)
    err = np.abs(P.polyval(wl - 0.5 * W0, m32) - g) / g
    print("// degree %d on wl in [0, %g]: max relative error %.2e (fp32-rounded coefficients, exact arithmetic)" % (DEG, W0, err.max()))
    print("static __constant__ float c_z32[%d] = {%s};  // highest power first" % (
        DEG + 1, ", ".join("%.9ef" % v for v in m32[::-1])))
