"""ctypes front end of oracle/wcsim_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_2203_02479_b200.
Every function here only marshals numpy arrays into the C routine of the same
name; the arithmetic (and its citations of PAPER.md) lives in wcsim_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wcsim_oracle.c")
_LIB = os.path.join(_HERE, "libwcoracle.so")
_CFLAGS = ["-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC"]
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile wcsim_oracle.c with gcc (building the checker is not using it)."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + ".tmp%d" % os.getpid()
            subprocess.check_call(["gcc", *_CFLAGS, "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        f64p, f32p = C.POINTER(C.c_double), C.POINTER(C.c_float)
        i32p, i64p, u64p, u32p = C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_uint64), C.POINTER(C.c_uint32)
        L.wco_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.wco_philox4x32_10.restype = None
        L.wco_fluct_word.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64]
        L.wco_fluct_word.restype = C.c_uint32
        L.wco_noise_word.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32]
        L.wco_noise_word.restype = C.c_uint32
        L.wco_norm_ppf.argtypes = [C.c_double]
        L.wco_norm_ppf.restype = C.c_double
        L.wco_binomial.argtypes = [C.c_double, C.c_double, C.c_uint32]
        L.wco_binomial.restype = C.c_double
        L.wco_normal_draw.argtypes = [C.c_double, C.c_double, C.c_uint32]
        L.wco_normal_draw.restype = C.c_double
        L.wco_axis_extent.argtypes = [C.c_double, C.c_double, C.c_double, i64p, i64p]
        L.wco_axis_extent.restype = None
        L.wco_axis_weight.argtypes = [C.c_int64, C.c_double, C.c_double]
        L.wco_axis_weight.restype = C.c_double
        L.wco_patch_axes.argtypes = [C.c_float] * 4 + [C.c_double, i64p, i64p, i64p, i64p, f64p, C.c_int, f64p, C.c_int]
        L.wco_patch_axes.restype = C.c_int
        L.wco_raster_scatter.argtypes = [C.c_int, C.c_int, f32p, f32p, f32p, f32p, f32p, C.c_int64, u64p, C.c_uint64,
                                         C.c_uint64, C.c_int, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, f64p,
                                         i32p, i64p, C.c_int]
        L.wco_raster_scatter.restype = C.c_int
        L.wco_convolve_direct.argtypes = [C.c_int, C.c_int, f64p, f64p, C.c_int, C.c_int, f64p]
        L.wco_convolve_direct.restype = C.c_int
        L.wco_convolve_impact.argtypes = [C.c_int, C.c_int, C.c_int, f64p, f64p, C.c_int, C.c_int, f64p]
        L.wco_convolve_impact.restype = C.c_int
        L.wco_convolve_points.argtypes = [C.c_int, C.c_int, f64p, f64p, C.c_int, C.c_int, C.c_int64, i32p, i32p, f64p]
        L.wco_convolve_points.restype = C.c_int
        L.wco_convolve_fft.argtypes = [C.c_int, C.c_int, f64p, f64p, C.c_int, C.c_int, C.c_int, C.c_int, f64p]
        L.wco_convolve_fft.restype = C.c_int
        L.wco_noise_amp.argtypes = [C.c_int, f64p]
        L.wco_noise_amp.restype = None
        L.wco_noise_spectrum.argtypes = [C.c_int, C.c_uint64, C.c_uint32, f64p, f64p, f64p]
        L.wco_noise_spectrum.restype = None
        L.wco_noise_points.argtypes = [C.c_int, C.c_uint64, f64p, C.c_int64, i32p, i32p, f64p]
        L.wco_noise_points.restype = C.c_int
        L.wco_noise_add.argtypes = [C.c_int, C.c_int, C.c_int, C.c_uint64, f64p, f64p]
        L.wco_noise_add.restype = C.c_int
        L.wco_fft.argtypes = [f64p, f64p, C.c_int, C.c_int]
        L.wco_fft.restype = C.c_int
        L.wco_num_threads.argtypes = []
        L.wco_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().wco_num_threads())


def set_num_threads(n: int) -> None:
    """Threads of the loops over independent rows (timing only)."""
    L = lib()
    L.wco_set_num_threads.argtypes = [C.c_int]
    L.wco_set_num_threads.restype = None
    L.wco_set_num_threads(int(n))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().wco_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def fluct_word(seed, depo_id, g) -> int:
    return int(lib().wco_fluct_word(seed, depo_id, g))


def noise_word(seed, wire, k) -> int:
    return int(lib().wco_noise_word(seed, wire, k))


def norm_ppf(u: float) -> float:
    return float(lib().wco_norm_ppf(float(u)))


def binomial(N: float, p: float, w: int) -> float:
    return float(lib().wco_binomial(float(N), float(p), int(w) & 0xFFFFFFFF))


def normal_draw(N: float, p: float, w: int) -> float:
    """The normal-approximation draw of the paper's Kokkos port (reading A21)."""
    return float(lib().wco_normal_draw(float(N), float(p), int(w) & 0xFFFFFFFF))


def axis_extent(centre, sigma, nsigma=3.0):
    i0, i1 = C.c_int64(), C.c_int64()
    lib().wco_axis_extent(float(centre), float(sigma), float(nsigma), C.byref(i0), C.byref(i1))
    return i0.value, i1.value


def axis_weight(i, centre, sigma) -> float:
    return float(lib().wco_axis_weight(int(i), float(centre), float(sigma)))


def patch_axes(t0, x0, sigma_t, sigma_x, nsigma=3.0, max_bins=4096):
    """Extents and per-axis weights of one depo: (it0, ix0, wt[], wx[])."""
    it0, it1, ix0, ix1 = C.c_int64(), C.c_int64(), C.c_int64(), C.c_int64()
    wt = np.zeros(max_bins)
    wx = np.zeros(max_bins)
    rc = lib().wco_patch_axes(np.float32(t0), np.float32(x0), np.float32(sigma_t), np.float32(sigma_x), float(nsigma),
                              C.byref(it0), C.byref(it1), C.byref(ix0), C.byref(ix1),
                              _p(wt, C.c_double), max_bins, _p(wx, C.c_double), max_bins)
    if rc != 0:
        raise ValueError("wco_patch_axes rc=%d" % rc)
    return it0.value, ix0.value, wt[: it1.value - it0.value].copy(), wx[: ix1.value - ix0.value].copy()


def drift(x, y, z, t, q, *, v_drift, D_L, D_T, tick, t_origin=0.0, lifetime=0.0, x_plane=0.0, cos_theta=1.0,
          sin_theta=0.0, pitch_origin=0.0, pitch=1.0):
    """Reading A22: electron groups (cm, us, electrons) -> depos of one plane (ticks, pitches)."""
    x, y, z, t, q = (_f32(a) for a in (x, y, z, t, q))
    n = x.shape[0]
    out = {k: np.empty(n, dtype=np.float32) for k in ("t0", "x0", "sigma_t", "sigma_x", "q")}
    f32p = C.POINTER(C.c_float)
    L = lib()
    L.wco_drift.argtypes = [f32p] * 5 + [C.c_int64] + [C.c_double] * 11 + [f32p] * 5
    L.wco_drift.restype = C.c_int
    rc = L.wco_drift(*[_p(a, C.c_float) for a in (x, y, z, t, q)], n, float(v_drift), float(D_L), float(D_T), float(tick),
                     float(t_origin), float(lifetime), float(x_plane), float(cos_theta), float(sin_theta),
                     float(pitch_origin), float(pitch), *[_p(out[k], C.c_float) for k in ("t0", "x0", "sigma_t", "sigma_x", "q")])
    if rc != 0:
        raise ValueError("wco_drift rc=%d" % rc)
    return out


def digitize(M, gain, baseline, bits=12):
    """Reading A23: ideal ADC codes of an fp32 grid, int16."""
    M = np.ascontiguousarray(M, dtype=np.float32)
    adc = np.empty(M.shape, dtype=np.int16)
    L = lib()
    L.wco_digitize.argtypes = [C.POINTER(C.c_float), C.c_int64, C.c_float, C.c_float, C.c_int, C.POINTER(C.c_int16)]
    L.wco_digitize.restype = C.c_int
    rc = L.wco_digitize(_p(M, C.c_float), M.size, float(gain), float(baseline), int(bits), _p(adc, C.c_int16))
    if rc != 0:
        raise ValueError("wco_digitize rc=%d" % rc)
    return adc


def _fluct_mode(fluctuate) -> int:
    """False/0: off, True/1: binomial (A6), 2 or "normal": normal approximation (A21)."""
    if fluctuate == "normal":
        return 2
    if fluctuate == "binomial":
        return 1
    m = int(fluctuate)
    if m not in (0, 1, 2):
        raise ValueError("fluctuate must be 0, 1 or 2")
    return m


def raster_scatter(n_wires, n_ticks, depos, *, seed=0, fluctuate=False, nsigma=3.0, ids=None, id_base=0,
                   window=None, want_totals=False, S=None, normalize=False):
    """depos = dict(t0,x0,sigma_t,sigma_x,q) of float arrays.  Returns (S_window fp64, totals|None, stats)."""
    t0, x0, st, sx, q = (_f32(depos[k]) for k in ("t0", "x0", "sigma_t", "sigma_x", "q"))
    n = t0.shape[0]
    w0, w1, k0, k1 = window if window is not None else (0, n_wires, 0, n_ticks)
    if S is None:
        S = np.zeros((w1 - w0, k1 - k0), dtype=np.float64)
    assert S.shape == (w1 - w0, k1 - k0) and S.dtype == np.float64 and S.flags.c_contiguous
    totals = np.zeros(n, dtype=np.int32) if want_totals else None
    stats = np.zeros(2, dtype=np.int64)
    idp = None
    if ids is not None:
        ids = np.ascontiguousarray(ids, dtype=np.uint64)
        assert ids.shape[0] == n
        idp = _p(ids, C.c_uint64)
    rc = lib().wco_raster_scatter(n_wires, n_ticks, _p(t0, C.c_float), _p(x0, C.c_float), _p(st, C.c_float),
                                  _p(sx, C.c_float), _p(q, C.c_float), n, idp, id_base, seed, _fluct_mode(fluctuate),
                                  float(nsigma), w0, w1, k0, k1, _p(S, C.c_double),
                                  _p(totals, C.c_int32) if want_totals else None, _p(stats, C.c_int64),
                                  int(bool(normalize)))
    if rc != 0:
        raise ValueError("wco_raster_scatter rc=%d" % rc)
    return S, totals, {"skipped": int(stats[0]), "drawn": int(stats[1])}


def convolve_direct(S, R):
    S, R = _f64(S), _f64(R)
    M = np.zeros_like(S)
    rc = lib().wco_convolve_direct(S.shape[0], S.shape[1], _p(S, C.c_double), _p(R, C.c_double), R.shape[0], R.shape[1],
                                   _p(M, C.c_double))
    if rc != 0:
        raise ValueError("wco_convolve_direct rc=%d" % rc)
    return M


def convolve_impact(Sf, R, K):
    """Reading A25: Sf [n_wires*K][n_ticks] (fine row x*K + k = impact position k of wire x), R [K][n_rw][n_rt];
    returns M [n_wires][n_ticks]."""
    Sf, R = _f64(Sf), _f64(R)
    K = int(K)
    if R.ndim != 3 or R.shape[0] != K or Sf.shape[0] % K:
        raise ValueError("R must be [K][n_rw][n_rt] and Sf must have a multiple of K rows")
    n_wires = Sf.shape[0] // K
    M = np.zeros((n_wires, Sf.shape[1]))
    rc = lib().wco_convolve_impact(n_wires, Sf.shape[1], K, _p(Sf, C.c_double), _p(R, C.c_double), R.shape[1],
                                   R.shape[2], _p(M, C.c_double))
    if rc != 0:
        raise ValueError("wco_convolve_impact rc=%d" % rc)
    return M


def convolve_points(S, R, px, pt):
    S, R = _f64(S), _f64(R)
    px = np.ascontiguousarray(px, dtype=np.int32)
    pt = np.ascontiguousarray(pt, dtype=np.int32)
    out = np.zeros(px.shape[0])
    rc = lib().wco_convolve_points(S.shape[0], S.shape[1], _p(S, C.c_double), _p(R, C.c_double), R.shape[0], R.shape[1],
                                   px.shape[0], _p(px, C.c_int32), _p(pt, C.c_int32), _p(out, C.c_double))
    if rc != 0:
        raise ValueError("wco_convolve_points rc=%d" % rc)
    return out


def convolve_fft(S, R, pad_w, pad_t):
    S, R = _f64(S), _f64(R)
    M = np.zeros_like(S)
    rc = lib().wco_convolve_fft(S.shape[0], S.shape[1], _p(S, C.c_double), _p(R, C.c_double), R.shape[0], R.shape[1],
                                int(pad_w), int(pad_t), _p(M, C.c_double))
    if rc != 0:
        raise ValueError("wco_convolve_fft rc=%d" % rc)
    return M


def noise_amp(P):
    amp = np.zeros(P // 2 + 1)
    lib().wco_noise_amp(int(P), _p(amp, C.c_double))
    return amp


def noise_spectrum(P, seed, wire, amp=None):
    amp = noise_amp(P) if amp is None else _f64(amp)
    zre, zim = np.zeros(P // 2 + 1), np.zeros(P // 2 + 1)
    lib().wco_noise_spectrum(int(P), seed, wire, _p(amp, C.c_double), _p(zre, C.c_double), _p(zim, C.c_double))
    return zre + 1j * zim


def noise_points(P, seed, wires, ticks, amp=None):
    wires = np.ascontiguousarray(wires, dtype=np.int32)
    ticks = np.ascontiguousarray(ticks, dtype=np.int32)
    out = np.zeros(wires.shape[0])
    a = None if amp is None else _f64(amp)
    rc = lib().wco_noise_points(int(P), seed, None if a is None else _p(a, C.c_double), wires.shape[0],
                                _p(wires, C.c_int32), _p(ticks, C.c_int32), _p(out, C.c_double))
    if rc != 0:
        raise ValueError("wco_noise_points rc=%d" % rc)
    return out


def noise_add(M, P, seed, amp=None):
    """M[wire][tick] (fp64, modified in place and returned) += N."""
    assert M.dtype == np.float64 and M.flags.c_contiguous
    a = None if amp is None else _f64(amp)
    rc = lib().wco_noise_add(int(P), M.shape[0], M.shape[1], seed, None if a is None else _p(a, C.c_double),
                             _p(M, C.c_double))
    if rc != 0:
        raise ValueError("wco_noise_add rc=%d" % rc)
    return M


def fft(z, sign=-1):
    z = np.asarray(z, dtype=np.complex128)
    re, im = np.ascontiguousarray(z.real), np.ascontiguousarray(z.imag)
    rc = lib().wco_fft(_p(re, C.c_double), _p(im, C.c_double), z.shape[0], sign)
    if rc != 0:
        raise ValueError("wco_fft rc=%d" % rc)
    return re + 1j * im
