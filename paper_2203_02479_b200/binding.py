"""Thin ctypes binding of libwcsim.so (include/wcsim.h): argument marshalling only.

Every function has the name and the argument order of the C call it wraps; device arrays are torch CUDA tensors
(torch supplies device memory and the stream, nothing else) and are passed down as raw pointers.  There is no CPU
fallback: if the library cannot be loaded the import of this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
import weakref

import numpy as np

from . import build as _build

WCSIM_OK, WCSIM_EINVAL, WCSIM_ENOMEM, WCSIM_ECUDA, WCSIM_ESTATE, WCSIM_ETOOBIG = 0, -1, -2, -3, -4, -5
WCSIM_NOALLOC_MAX_BINS = 524288  # include/wcsim.h
WCSIM_SCATTER_ATOMIC, WCSIM_SCATTER_TILED, WCSIM_SCATTER_FIXED = 0, 1, 2
WCSIM_WIRES_AUTO, WCSIM_WIRES_FFT, WCSIM_WIRES_DIRECT = 0, 1, 2

# every symbol include/wcsim.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "wcsim_plan_create", "wcsim_raster_scatter", "wcsim_convolve", "wcsim_add_noise", "wcsim_arm_noise",
    "wcsim_plan_destroy", "wcsim_clear", "wcsim_clear_output", "wcsim_sync", "wcsim_set_scatter_mode", "wcsim_set_wire_mode",
    "wcsim_charge_ptr", "wcsim_output_ptr", "wcsim_get_dims", "wcsim_get_stats", "wcsim_reset_stats",
    "wcsim_simulate_host", "wcsim_set_profiling", "wcsim_get_stage_times", "wcsim_get_launch_count",
    "wcsim_debug_philox", "wcsim_debug_binomial", "wcsim_debug_response_spectrum", "wcsim_debug_erf", "wcsim_simulate_host_async", "wcsim_debug_normal_draw", "wcsim_drift", "wcsim_digitize", "wcsim_set_normalize",
    "wcsim_debug_fast_normal", "wcsim_debug_z32_scan",
    "wcsim_plan_create_planes", "wcsim_raster_scatter_planes", "wcsim_get_plane_rows", "wcsim_simulate_host_adc_async",
    "wcsim_plan_create_impact", "wcsim_get_charge_dims",
    "wcsim_raster_scatter_noalloc",
    "wcsim_graph_update", "wcsim_get_wire_mode",
    "wcsim_raster_scatter_planes_seeded", "wcsim_arm_noise_planes", "wcsim_add_noise_planes",
    "wcsim_graph_begin", "wcsim_graph_end", "wcsim_graph_launch", "wcsim_graph_destroy",
    "wcsim_strerror", "wcsim_last_cuda_error", "wcsim_version",
]


class wcsim_pad(C.Structure):
    _fields_ = [("wires", C.c_int), ("ticks", C.c_int)]


class wcsim_depos(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("t0", "x0", "sigma_t", "sigma_x", "q")]


class wcsim_drift_params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("v_drift", "D_L", "D_T", "tick", "t_origin", "lifetime")]


class wcsim_plane_geom(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("x_plane", "cos_theta", "sin_theta", "pitch_origin", "pitch")]


class wcsim_stats(C.Structure):
    _fields_ = [("depos_skipped", C.c_ulonglong), ("bins_drawn", C.c_ulonglong)]


class WcsimError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        msg = lib().wcsim_strerror(status).decode()
        if status == WCSIM_ECUDA:
            msg += " [cudaError_t %d]" % lib().wcsim_last_cuda_error()
        super().__init__("%s: %s (%d)" % (where, msg, status))


_lib = None


def lib():
    """The loaded libwcsim.so (built in-tree with nvcc on first use).  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, ll, ull, i = C.c_void_p, C.c_longlong, C.c_ulonglong, C.c_int
        L.wcsim_plan_create.argtypes = [C.POINTER(vp), i, i, vp, i, i, wcsim_pad, C.c_float, i, vp]
        L.wcsim_raster_scatter.argtypes = [vp, C.POINTER(wcsim_depos), ll, ull, ull, i, vp]
        L.wcsim_convolve.argtypes = [vp]
        L.wcsim_add_noise.argtypes = [vp, vp, ull]
        L.wcsim_arm_noise.argtypes = [vp, vp, ull]
        L.wcsim_plan_destroy.argtypes = [vp]
        L.wcsim_clear.argtypes = [vp]
        L.wcsim_clear_output.argtypes = [vp]
        L.wcsim_sync.argtypes = [vp]
        L.wcsim_set_scatter_mode.argtypes = [vp, i]
        L.wcsim_set_wire_mode.argtypes = [vp, i]
        L.wcsim_set_normalize.argtypes = [vp, i]
        L.wcsim_get_wire_mode.argtypes = [vp, C.POINTER(i)]
        L.wcsim_charge_ptr.argtypes = [vp, C.POINTER(vp)]
        L.wcsim_output_ptr.argtypes = [vp, C.POINTER(vp)]
        L.wcsim_get_dims.argtypes = [vp] + [C.POINTER(i)] * 4
        L.wcsim_get_stats.argtypes = [vp, C.POINTER(wcsim_stats)]
        L.wcsim_reset_stats.argtypes = [vp]
        L.wcsim_simulate_host.argtypes = [vp, vp, vp, vp, vp, vp, ll, ull, i, i, ull, vp]
        L.wcsim_simulate_host_async.argtypes = [vp, vp, vp, vp, vp, vp, ll, ull, i, i, ull, vp]
        L.wcsim_set_profiling.argtypes = [vp, i]
        L.wcsim_get_stage_times.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(ull), i]
        L.wcsim_get_launch_count.argtypes = [vp, C.POINTER(ull)]
        L.wcsim_debug_philox.argtypes = [vp, vp, vp, ll, vp]
        L.wcsim_debug_binomial.argtypes = [vp, vp, vp, vp, ll, vp]
        L.wcsim_debug_normal_draw.argtypes = [vp, vp, vp, vp, ll, vp]
        L.wcsim_debug_fast_normal.argtypes = [vp, vp, vp, vp, vp, ll, vp]
        L.wcsim_debug_z32_scan.argtypes = [ull, ull, vp, vp]
        L.wcsim_debug_response_spectrum.argtypes = [vp, vp]
        L.wcsim_debug_erf.argtypes = [vp, vp, ll]
        L.wcsim_digitize.argtypes = [vp, C.c_float, C.c_float, i, vp]
        L.wcsim_drift.argtypes = [vp, vp, vp, vp, vp, ll, C.POINTER(wcsim_drift_params), C.POINTER(wcsim_plane_geom), i,
                                  C.POINTER(wcsim_depos), vp]
        L.wcsim_plan_create_planes.argtypes = [C.POINTER(vp), i, C.POINTER(i), i, C.POINTER(vp), i, i, i, C.c_float, i, vp]
        L.wcsim_raster_scatter_planes.argtypes = [vp, C.POINTER(wcsim_depos), C.POINTER(ll), ull, i]
        L.wcsim_raster_scatter_planes_seeded.argtypes = [vp, C.POINTER(wcsim_depos), C.POINTER(ll), C.POINTER(ull), i]
        L.wcsim_arm_noise_planes.argtypes = [vp, vp, C.POINTER(ull)]
        L.wcsim_add_noise_planes.argtypes = [vp, vp, C.POINTER(ull)]
        L.wcsim_get_plane_rows.argtypes = [vp, i, C.POINTER(i), C.POINTER(i)]
        L.wcsim_simulate_host_adc_async.argtypes = [vp, vp, vp, vp, vp, vp, ll, ull, i, i, ull, C.c_float, C.c_float, i, vp]
        L.wcsim_plan_create_impact.argtypes = [C.POINTER(vp), i, i, i, C.POINTER(vp), i, i, i, C.c_float, i, vp]
        L.wcsim_get_charge_dims.argtypes = [vp, C.POINTER(i), C.POINTER(i), C.POINTER(i)]
        L.wcsim_raster_scatter_noalloc.argtypes = [i, i, C.POINTER(wcsim_depos), ll, ull, ull, i, C.c_float, vp, vp]
        L.wcsim_graph_begin.argtypes = [vp]
        L.wcsim_graph_end.argtypes = [vp, C.POINTER(vp)]
        L.wcsim_graph_launch.argtypes = [vp]
        L.wcsim_graph_update.argtypes = [vp, vp]
        L.wcsim_graph_destroy.argtypes = [vp]
        L.wcsim_strerror.argtypes = [i]
        L.wcsim_strerror.restype = C.c_char_p
        L.wcsim_last_cuda_error.argtypes = []
        L.wcsim_version.argtypes = []
        L.wcsim_version.restype = C.c_char_p
        for name in SYMBOLS:
            fn = getattr(L, name)
            if fn.restype is not C.c_char_p:
                fn.restype = C.c_int
        _lib = L
    return _lib


def _check(status, where):
    if status != WCSIM_OK:
        raise WcsimError(status, where)


def _dev_ptr(t, dtype=None):
    """Raw device pointer of a contiguous torch CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError("expected dtype %s, got %s" % (dtype, t.dtype))
    return C.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


class _Borrowed:
    """A device buffer owned by a plan, exposed through __cuda_array_interface__ so torch can view it without a copy."""

    def __init__(self, ptr, shape, owner):
        self._owner = owner
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": "<f4", "data": (int(ptr), False),
                                         "version": 2, "strides": None}


# ---- the C calls, one to one ------------------------------------------------------------------------------------
def wcsim_plan_create(n_wires, n_ticks, response, pad=(0, 0), nsigma=3.0, scatter_mode=WCSIM_SCATTER_ATOMIC,
                      stream=None):
    """response: host numpy array [n_rwires][n_rticks] float32.  Returns the opaque plan handle."""
    r = np.ascontiguousarray(response, dtype=np.float32)
    if r.ndim != 2:
        raise ValueError("response must be 2-D [n_rwires][n_rticks]")
    h = C.c_void_p()
    st = lib().wcsim_plan_create(C.byref(h), int(n_wires), int(n_ticks), r.ctypes.data_as(C.c_void_p), r.shape[0],
                                 r.shape[1], wcsim_pad(int(pad[0]), int(pad[1])), float(nsigma), int(scatter_mode),
                                 _stream_ptr(stream))
    _check(st, "wcsim_plan_create")
    return h


WCSIM_FLUCT_OFF, WCSIM_FLUCT_BINOMIAL, WCSIM_FLUCT_NORMAL = 0, 1, 2


def _fluct(fluctuate) -> int:
    """False/0: off; True/1/"binomial": reading A6; 2/"normal": the Kokkos port's normal approximation (A21)."""
    if isinstance(fluctuate, str):
        return {"off": 0, "binomial": 1, "normal": 2}[fluctuate]
    return int(fluctuate)


def wcsim_raster_scatter(plan, depos, n=None, depo_id_base=0, seed=0, fluctuate=False, dev_depo_totals=None):
    """depos: dict (or object) of torch CUDA float32 tensors t0, x0, sigma_t, sigma_x, q."""
    import torch
    get = (lambda k: depos[k]) if isinstance(depos, dict) else (lambda k: getattr(depos, k))
    arrs = [get(k) for k in ("t0", "x0", "sigma_t", "sigma_x", "q")]
    if n is None:
        n = arrs[0].numel()
    for a in arrs:
        if a.numel() < n:
            raise ValueError("depo array shorter than n")
    d = wcsim_depos(*[_dev_ptr(a, torch.float32) for a in arrs])
    st = lib().wcsim_raster_scatter(plan, C.byref(d), int(n), int(depo_id_base), int(seed), _fluct(fluctuate),
                                    _dev_ptr(dev_depo_totals, torch.int32))
    _check(st, "wcsim_raster_scatter")


def wcsim_raster_scatter_noalloc(n_wires, n_ticks, depos, dev_S, n=None, depo_id_base=0, seed=0, fluctuate=False,
                                 nsigma=3.0, stream=None):
    """Raster + scatter-add into the caller's own grid, for code that may not allocate device memory (no plan, no
    cudaMalloc: the kernel's scratch is a fixed 4 MiB array built into libwcsim.so).  dev_S: torch CUDA float32 tensor of
    n_wires * n_ticks elements, accumulated into.  Grids above WCSIM_NOALLOC_MAX_BINS bins raise WcsimError
    (WCSIM_ETOOBIG).  The first call on a device synchronises `stream` once; calls that overlap on the GPU race on the
    shared scratch (include/wcsim.h has the full contract)."""
    import torch
    get = (lambda k: depos[k]) if isinstance(depos, dict) else (lambda k: getattr(depos, k))
    arrs = [get(k) for k in ("t0", "x0", "sigma_t", "sigma_x", "q")]
    if n is None:
        n = arrs[0].numel()
    for a in arrs:
        if a.numel() < n:
            raise ValueError("depo array shorter than n")
    if dev_S is not None and dev_S.numel() < int(n_wires) * int(n_ticks):
        raise ValueError("dev_S holds fewer than n_wires * n_ticks floats")
    d = wcsim_depos(*[_dev_ptr(a, torch.float32) for a in arrs])
    st = lib().wcsim_raster_scatter_noalloc(int(n_wires), int(n_ticks), C.byref(d), int(n), int(depo_id_base), int(seed),
                                            _fluct(fluctuate), float(nsigma), _dev_ptr(dev_S, torch.float32),
                                            _stream_ptr(stream))
    _check(st, "wcsim_raster_scatter_noalloc")


def wcsim_convolve(plan):
    _check(lib().wcsim_convolve(plan), "wcsim_convolve")


def _amp_ptr(amp):
    if amp is None:
        return None, None
    a = np.ascontiguousarray(amp, dtype=np.float32)
    return a, a.ctypes.data_as(C.c_void_p)


def wcsim_add_noise(plan, amp=None, seed=0):
    keep, p = _amp_ptr(amp)
    _check(lib().wcsim_add_noise(plan, p, int(seed)), "wcsim_add_noise")


def wcsim_arm_noise(plan, amp=None, seed=0):
    keep, p = _amp_ptr(amp)
    _check(lib().wcsim_arm_noise(plan, p, int(seed)), "wcsim_arm_noise")


def wcsim_plan_destroy(plan):
    _check(lib().wcsim_plan_destroy(plan), "wcsim_plan_destroy")


def wcsim_clear(plan):
    _check(lib().wcsim_clear(plan), "wcsim_clear")


def wcsim_clear_output(plan):
    _check(lib().wcsim_clear_output(plan), "wcsim_clear_output")


def wcsim_sync(plan):
    _check(lib().wcsim_sync(plan), "wcsim_sync")


def wcsim_set_scatter_mode(plan, scatter_mode):
    _check(lib().wcsim_set_scatter_mode(plan, int(scatter_mode)), "wcsim_set_scatter_mode")


def wcsim_set_normalize(plan, on):
    _check(lib().wcsim_set_normalize(plan, int(bool(on))), "wcsim_set_normalize")


def wcsim_set_wire_mode(plan, wire_mode):
    _check(lib().wcsim_set_wire_mode(plan, int(wire_mode)), "wcsim_set_wire_mode")


def wcsim_get_wire_mode(plan):
    """The wire-axis route wcsim_convolve takes on this plan now (WCSIM_WIRES_DIRECT or WCSIM_WIRES_FFT)."""
    m = C.c_int()
    _check(lib().wcsim_get_wire_mode(plan, C.byref(m)), "wcsim_get_wire_mode")
    return m.value


def wcsim_get_dims(plan):
    v = [C.c_int() for _ in range(4)]
    _check(lib().wcsim_get_dims(plan, *[C.byref(x) for x in v]), "wcsim_get_dims")
    return tuple(x.value for x in v)


def _borrow(plan, fn, name, rows=None):
    import torch
    p = C.c_void_p()
    _check(fn(plan, C.byref(p)), name)
    n_wires, n_ticks, _, _ = wcsim_get_dims(plan)
    return torch.as_tensor(_Borrowed(p.value, (rows or n_wires, n_ticks), plan), device="cuda")


def wcsim_get_charge_dims(plan):
    """(rows, ticks, impact positions per wire) of the charge grid S."""
    v = [C.c_int() for _ in range(3)]
    _check(lib().wcsim_get_charge_dims(plan, *[C.byref(x) for x in v]), "wcsim_get_charge_dims")
    return tuple(x.value for x in v)


def wcsim_charge_ptr(plan):
    """S as a torch view [rows][n_ticks] of the plan's buffer (borrowed: valid until wcsim_plan_destroy)."""
    return _borrow(plan, lib().wcsim_charge_ptr, "wcsim_charge_ptr", rows=wcsim_get_charge_dims(plan)[0])


def wcsim_output_ptr(plan):
    """M as a torch view [n_wires][n_ticks] of the plan's buffer (borrowed)."""
    return _borrow(plan, lib().wcsim_output_ptr, "wcsim_output_ptr")


def wcsim_get_stats(plan):
    s = wcsim_stats()
    _check(lib().wcsim_get_stats(plan, C.byref(s)), "wcsim_get_stats")
    return {"depos_skipped": int(s.depos_skipped), "bins_drawn": int(s.bins_drawn)}


def wcsim_reset_stats(plan):
    _check(lib().wcsim_reset_stats(plan), "wcsim_reset_stats")


def _host_ptr(a, itemsize=4):
    """(pointer, element count) of a contiguous HOST array of `itemsize`-byte elements (numpy, or a torch CPU tensor)."""
    if hasattr(a, "data_ptr"):
        if a.is_cuda or not a.is_contiguous() or a.element_size() != itemsize:
            raise ValueError("expected a contiguous host tensor of %d-byte elements" % itemsize)
        return C.c_void_p(a.data_ptr()), a.numel()
    if a.dtype.itemsize != itemsize or not a.flags.c_contiguous:
        raise ValueError("expected a C-contiguous host array of %d-byte elements" % itemsize)
    return a.ctypes.data_as(C.c_void_p), a.size


def _host_depo_ptrs(host_depos, n):
    ptrs = [_host_ptr(host_depos[k]) for k in ("t0", "x0", "sigma_t", "sigma_x", "q")]
    for k in ("t0", "x0", "sigma_t", "sigma_x", "q"):
        if not str(host_depos[k].dtype).endswith("float32"):
            raise ValueError("host depo array %s must be float32" % k)
    if n is None:
        n = ptrs[0][1]
    if any(cnt < n for _, cnt in ptrs):
        raise ValueError("host depo array shorter than n")
    return [p for p, _ in ptrs], int(n)


def wcsim_simulate_host(plan, host_depos, host_M, n=None, seed=0, fluctuate=False, noise=False, noise_seed=0,
                        _fn="wcsim_simulate_host"):
    """host_depos: dict of HOST float32 arrays (numpy, or torch CPU tensors -- pinned makes the copies asynchronous);
    host_M: HOST float32 [n_wires][n_ticks], written."""
    ptrs, n = _host_depo_ptrs(host_depos, n)
    pm, cnt = _host_ptr(host_M)
    n_wires, n_ticks, _, _ = wcsim_get_dims(plan)
    if cnt != n_wires * n_ticks:
        raise ValueError("host_M must hold n_wires * n_ticks = %d floats, got %d" % (n_wires * n_ticks, cnt))
    st = getattr(lib(), _fn)(plan, *ptrs, n, int(seed), _fluct(fluctuate), int(bool(noise)), int(noise_seed), pm)
    _check(st, _fn)


def wcsim_simulate_host_async(plan, host_depos, host_M, **kw):
    """As wcsim_simulate_host without the final synchronisation: host_M is valid after wcsim_sync(plan)."""
    wcsim_simulate_host(plan, host_depos, host_M, _fn="wcsim_simulate_host_async", **kw)


def wcsim_simulate_host_adc_async(plan, host_depos, host_adc, gain, baseline, bits=12, n=None, seed=0, fluctuate=False,
                                  noise=False, noise_seed=0):
    """host_adc: HOST int16 [n_wires][n_ticks], written; valid after wcsim_sync(plan)."""
    ptrs, n = _host_depo_ptrs(host_depos, n)
    pa, cnt = _host_ptr(host_adc, 2)
    n_wires, n_ticks, _, _ = wcsim_get_dims(plan)
    if cnt != n_wires * n_ticks:
        raise ValueError("host_adc must hold n_wires * n_ticks = %d int16, got %d" % (n_wires * n_ticks, cnt))
    st = lib().wcsim_simulate_host_adc_async(plan, *ptrs, n, int(seed), _fluct(fluctuate), int(bool(noise)),
                                             int(noise_seed), float(gain), float(baseline), int(bits), pa)
    _check(st, "wcsim_simulate_host_adc_async")


def wcsim_plan_create_planes(n_wires, n_ticks, responses, pad_ticks=0, nsigma=3.0, scatter_mode=WCSIM_SCATTER_ATOMIC,
                             stream=None):
    """n_wires: one int per plane; responses: one host array [n_rwires][n_rticks] per plane (same shape)."""
    rs = [np.ascontiguousarray(r, dtype=np.float32) for r in responses]
    if len(rs) != len(n_wires) or not rs or any(r.ndim != 2 or r.shape != rs[0].shape for r in rs):
        raise ValueError("one 2-D response of the same shape per plane")
    nw = (C.c_int * len(rs))(*[int(w) for w in n_wires])
    rp = (C.c_void_p * len(rs))(*[r.ctypes.data_as(C.c_void_p) for r in rs])
    h = C.c_void_p()
    st = lib().wcsim_plan_create_planes(C.byref(h), len(rs), nw, int(n_ticks), rp, rs[0].shape[0], rs[0].shape[1],
                                        int(pad_ticks), float(nsigma), int(scatter_mode), _stream_ptr(stream))
    _check(st, "wcsim_plan_create_planes")
    return h


def wcsim_plan_create_impact(n_wires, n_ticks, responses, pad_ticks=0, nsigma=3.0, scatter_mode=WCSIM_SCATTER_ATOMIC,
                             stream=None):
    """responses: host array [n_impact][n_rwires][n_rticks] (reading A25)."""
    r = np.ascontiguousarray(responses, dtype=np.float32)
    if r.ndim != 3:
        raise ValueError("responses must be 3-D [n_impact][n_rwires][n_rticks]")
    rp = (C.c_void_p * r.shape[0])(*[r[k].ctypes.data_as(C.c_void_p) for k in range(r.shape[0])])
    h = C.c_void_p()
    st = lib().wcsim_plan_create_impact(C.byref(h), int(n_wires), int(n_ticks), r.shape[0], rp, r.shape[1], r.shape[2],
                                        int(pad_ticks), float(nsigma), int(scatter_mode), _stream_ptr(stream))
    _check(st, "wcsim_plan_create_impact")
    return h


def wcsim_raster_scatter_planes(plan, depos, n=None, seed=0, fluctuate=False):
    """depos: one dict of torch CUDA float32 tensors t0, x0, sigma_t, sigma_x, q per plane."""
    import torch
    keys = ("t0", "x0", "sigma_t", "sigma_x", "q")
    if n is None:
        n = [d["t0"].numel() for d in depos]
    for d, cnt in zip(depos, n):
        if any(d[k].numel() < cnt for k in keys):
            raise ValueError("depo array shorter than n")
    ds = (wcsim_depos * len(depos))(*[wcsim_depos(*[_dev_ptr(d[k], torch.float32) for k in keys]) for d in depos])
    ns = (C.c_longlong * len(depos))(*[int(c) for c in n])
    _check(lib().wcsim_raster_scatter_planes(plan, ds, ns, int(seed), _fluct(fluctuate)), "wcsim_raster_scatter_planes")


def wcsim_raster_scatter_planes_seeded(plan, depos, seeds, n=None, fluctuate=False):
    """The same with one fluctuation seed per plane (reading A26): seeds[p] keys plane p's Philox draws."""
    import torch
    keys = ("t0", "x0", "sigma_t", "sigma_x", "q")
    if len(seeds) != len(depos) or len(depos) != _n_planes(plan):
        raise ValueError("one depo dict and one seed per plane of the plan")
    if n is None:
        n = [d["t0"].numel() for d in depos]
    for d, cnt in zip(depos, n):
        if any(d[k].numel() < cnt for k in keys):
            raise ValueError("depo array shorter than n")
    ds = (wcsim_depos * len(depos))(*[wcsim_depos(*[_dev_ptr(d[k], torch.float32) for k in keys]) for d in depos])
    ns = (C.c_longlong * len(depos))(*[int(c) for c in n])
    sd = (C.c_ulonglong * len(seeds))(*[int(x) for x in seeds])
    _check(lib().wcsim_raster_scatter_planes_seeded(plan, ds, ns, sd, _fluct(fluctuate)), "wcsim_raster_scatter_planes_seeded")


def _n_planes(plan) -> int:
    a, b, n = C.c_int(), C.c_int(), 0
    while lib().wcsim_get_plane_rows(plan, n, C.byref(a), C.byref(b)) == WCSIM_OK:
        n += 1
    return n


def _plane_seeds(plan, seeds):
    if len(seeds) != _n_planes(plan):
        raise ValueError("one seed per plane of the plan")
    return (C.c_ulonglong * len(seeds))(*[int(x) for x in seeds])


def wcsim_arm_noise_planes(plan, amp=None, seeds=()):
    """wcsim_arm_noise with one noise seed per plane of a multi-plane plan (reading A26)."""
    keep, p = _amp_ptr(amp)
    _check(lib().wcsim_arm_noise_planes(plan, p, _plane_seeds(plan, seeds)), "wcsim_arm_noise_planes")


def wcsim_add_noise_planes(plan, amp=None, seeds=()):
    keep, p = _amp_ptr(amp)
    _check(lib().wcsim_add_noise_planes(plan, p, _plane_seeds(plan, seeds)), "wcsim_add_noise_planes")


def wcsim_get_plane_rows(plan, plane):
    a, b = C.c_int(), C.c_int()
    _check(lib().wcsim_get_plane_rows(plan, int(plane), C.byref(a), C.byref(b)), "wcsim_get_plane_rows")
    return a.value, b.value


def wcsim_graph_begin(plan):
    _check(lib().wcsim_graph_begin(plan), "wcsim_graph_begin")


def wcsim_graph_end(plan):
    g = C.c_void_p()
    _check(lib().wcsim_graph_end(plan, C.byref(g)), "wcsim_graph_end")
    return g


def wcsim_graph_update(plan, graph):
    _check(lib().wcsim_graph_update(plan, graph), "wcsim_graph_update")


def wcsim_graph_launch(graph):
    _check(lib().wcsim_graph_launch(graph), "wcsim_graph_launch")


def wcsim_graph_destroy(graph):
    _check(lib().wcsim_graph_destroy(graph), "wcsim_graph_destroy")


STAGES = ("raster", "rows_forward", "cols", "rows_inverse", "noise", "convolve")
WCSIM_PROFILE_KERNELS, WCSIM_PROFILE_CALLS = 1, 2


def wcsim_set_profiling(plan, level):
    """0 / False off; True or WCSIM_PROFILE_KERNELS: a span per kernel; WCSIM_PROFILE_CALLS: one span per call."""
    _check(lib().wcsim_set_profiling(plan, int(level)), "wcsim_set_profiling")


def wcsim_get_stage_times(plan, reset=True):
    """{stage: (total ms, spans)} accumulated since the last reset (synchronises)."""
    ms = (C.c_double * len(STAGES))()
    calls = (C.c_ulonglong * len(STAGES))()
    _check(lib().wcsim_get_stage_times(plan, ms, calls, int(bool(reset))), "wcsim_get_stage_times")
    return {s: (float(ms[k]), int(calls[k])) for k, s in enumerate(STAGES)}


def wcsim_get_launch_count(plan):
    v = C.c_ulonglong()
    _check(lib().wcsim_get_launch_count(plan, C.byref(v)), "wcsim_get_launch_count")
    return int(v.value)


def wcsim_debug_philox(dev_ctr, dev_key, dev_out, n, stream=None):
    _check(lib().wcsim_debug_philox(_dev_ptr(dev_ctr), _dev_ptr(dev_key), _dev_ptr(dev_out), int(n),
                                    _stream_ptr(stream)), "wcsim_debug_philox")


def wcsim_debug_binomial(dev_N, dev_p, dev_w, dev_k, n, stream=None):
    _check(lib().wcsim_debug_binomial(_dev_ptr(dev_N), _dev_ptr(dev_p), _dev_ptr(dev_w), _dev_ptr(dev_k), int(n),
                                      _stream_ptr(stream)), "wcsim_debug_binomial")


def wcsim_digitize(plan, gain, baseline, bits, dev_adc):
    """dev_adc: DEVICE int16 tensor of n_wires*n_ticks elements, written (ideal ADC of reading A23)."""
    import torch
    n_wires, n_ticks, _, _ = wcsim_get_dims(plan)
    if dev_adc is None or dev_adc.numel() < n_wires * n_ticks:
        raise ValueError("dev_adc must hold n_wires * n_ticks int16")
    _check(lib().wcsim_digitize(plan, float(gain), float(baseline), int(bits), _dev_ptr(dev_adc, torch.int16)),
           "wcsim_digitize")


def wcsim_drift(groups, params, planes, out, n=None, stream=None):
    """groups: dict x, y, z, t, q of DEVICE float32 tensors; params: dict of wcsim_drift_params fields; planes: list of
    dicts of wcsim_plane_geom fields; out: list (one per plane) of dicts t0, x0, sigma_t, sigma_x, q of DEVICE float32
    tensors, written."""
    import torch
    ptrs = [_dev_ptr(groups[k], torch.float32) for k in ("x", "y", "z", "t", "q")]
    if n is None:
        n = groups["x"].numel()
    if any(groups[k].numel() < n for k in ("x", "y", "z", "t", "q")):
        raise ValueError("group array shorter than n")
    if len(out) != len(planes) or any(o[k].numel() < n for o in out for k in ("t0", "x0", "sigma_t", "sigma_x", "q")):
        raise ValueError("one set of output arrays of at least n floats per plane")
    prm = wcsim_drift_params(**{k: float(params.get(k, 0.0)) for k, _ in wcsim_drift_params._fields_})
    geo = (wcsim_plane_geom * len(planes))(*[wcsim_plane_geom(**{k: float(p[k]) for k, _ in wcsim_plane_geom._fields_})
                                            for p in planes])
    outs = (wcsim_depos * len(planes))(*[wcsim_depos(*[_dev_ptr(o[k], torch.float32) for k in ("t0", "x0", "sigma_t", "sigma_x", "q")])
                                         for o in out])
    _check(lib().wcsim_drift(*ptrs, int(n), C.byref(prm), geo, len(planes), outs, _stream_ptr(stream)), "wcsim_drift")


def wcsim_debug_fast_normal(dev_N, dev_p, dev_w, dev_k, dev_ok, n, stream=None):
    _check(lib().wcsim_debug_fast_normal(_dev_ptr(dev_N), _dev_ptr(dev_p), _dev_ptr(dev_w), _dev_ptr(dev_k),
                                         _dev_ptr(dev_ok), int(n), _stream_ptr(stream)), "wcsim_debug_fast_normal")


def wcsim_debug_z32_scan(first_word, n_words, dev_out4, stream=None):
    _check(lib().wcsim_debug_z32_scan(int(first_word), int(n_words), _dev_ptr(dev_out4), _stream_ptr(stream)),
           "wcsim_debug_z32_scan")


def wcsim_debug_normal_draw(dev_N, dev_p, dev_w, dev_k, n, stream=None):
    _check(lib().wcsim_debug_normal_draw(_dev_ptr(dev_N), _dev_ptr(dev_p), _dev_ptr(dev_w), _dev_ptr(dev_k), int(n),
                                         _stream_ptr(stream)), "wcsim_debug_normal_draw")


def wcsim_debug_erf(z):
    """The raster's table erf evaluated on the host (no device needed)."""
    import numpy as np
    z = np.ascontiguousarray(z, dtype=np.float64)
    out = np.empty_like(z)
    _check(lib().wcsim_debug_erf(z.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p), int(z.size)),
           "wcsim_debug_erf")
    return out


def wcsim_debug_response_spectrum(plan):
    _, _, pad_w, pad_t = wcsim_get_dims(plan)
    out = np.zeros((pad_w, pad_t // 2 + 1, 2), dtype=np.float32)
    _check(lib().wcsim_debug_response_spectrum(plan, out.ctypes.data_as(C.c_void_p)), "wcsim_debug_response_spectrum")
    return out[..., 0] + 1j * out[..., 1]


def wcsim_version():
    return lib().wcsim_version().decode()


class Plan:
    """Context-managed plan handle: `with Plan(...) as p: p.raster_scatter(...); p.convolve(); M = p.output()`."""

    def __init__(self, n_wires, n_ticks, response, pad=(0, 0), nsigma=3.0, scatter_mode=WCSIM_SCATTER_ATOMIC,
                 stream=None):
        self.handle = wcsim_plan_create(n_wires, n_ticks, response, pad, nsigma, scatter_mode, stream)
        self.n_wires, self.n_ticks, self.pad_w, self.pad_t = wcsim_get_dims(self.handle)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def destroy(self):
        if self.handle is not None:
            for r in getattr(self, "_graphs", []):  # the library refuses to free a plan its graphs still point at
                g = r()
                if g is not None:
                    g.destroy()
            h, self.handle = self.handle, None
            wcsim_plan_destroy(h)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def raster_scatter(self, depos, **kw):
        wcsim_raster_scatter(self.handle, depos, **kw)

    def convolve(self):
        wcsim_convolve(self.handle)

    def add_noise(self, amp=None, seed=0):
        wcsim_add_noise(self.handle, amp, seed)

    def arm_noise(self, amp=None, seed=0):
        wcsim_arm_noise(self.handle, amp, seed)

    def clear(self):
        wcsim_clear(self.handle)

    def clear_output(self):
        wcsim_clear_output(self.handle)

    def sync(self):
        wcsim_sync(self.handle)

    def set_scatter_mode(self, mode):
        wcsim_set_scatter_mode(self.handle, mode)

    def set_normalize(self, on):
        wcsim_set_normalize(self.handle, on)

    def wire_mode(self):
        return wcsim_get_wire_mode(self.handle)

    def set_wire_mode(self, mode):
        wcsim_set_wire_mode(self.handle, mode)

    def charge(self):
        return wcsim_charge_ptr(self.handle)

    def output(self):
        return wcsim_output_ptr(self.handle)

    def stats(self):
        return wcsim_get_stats(self.handle)

    def reset_stats(self):
        wcsim_reset_stats(self.handle)

    def set_profiling(self, enable):
        wcsim_set_profiling(self.handle, enable)

    def stage_times(self, reset=True):
        return wcsim_get_stage_times(self.handle, reset)

    def launch_count(self):
        return wcsim_get_launch_count(self.handle)

    def simulate_host(self, host_depos, host_M, **kw):
        wcsim_simulate_host(self.handle, host_depos, host_M, **kw)

    def digitize(self, gain, baseline, bits=12, out=None):
        import torch
        if out is None:
            out = torch.empty((self.n_wires, self.n_ticks), dtype=torch.int16, device="cuda")
        wcsim_digitize(self.handle, gain, baseline, bits, out)
        return out

    def simulate_host_async(self, host_depos, host_M, **kw):
        wcsim_simulate_host_async(self.handle, host_depos, host_M, **kw)

    def simulate_host_adc_async(self, host_depos, host_adc, gain, baseline, bits=12, **kw):
        wcsim_simulate_host_adc_async(self.handle, host_depos, host_adc, gain, baseline, bits, **kw)

    def response_spectrum(self):
        return wcsim_debug_response_spectrum(self.handle)

    def raster_scatter_planes(self, depos, seeds=None, **kw):
        if seeds is not None:
            return wcsim_raster_scatter_planes_seeded(self.handle, depos, seeds, **kw)
        wcsim_raster_scatter_planes(self.handle, depos, **kw)

    def arm_noise_planes(self, amp=None, seeds=()):
        wcsim_arm_noise_planes(self.handle, amp, seeds)

    def add_noise_planes(self, amp=None, seeds=()):
        wcsim_add_noise_planes(self.handle, amp, seeds)

    def plane_rows(self, plane):
        return wcsim_get_plane_rows(self.handle, plane)

    def graph_begin(self):
        wcsim_graph_begin(self.handle)

    def graph_end(self):
        g = Graph(wcsim_graph_end(self.handle), self)
        self._graphs = [r for r in getattr(self, "_graphs", []) if r() is not None] + [weakref.ref(g)]
        return g


class PlanesPlan(Plan):
    """A multi-plane plan (wcsim_plan_create_planes): the planes of one event through one launch sequence."""

    def __init__(self, n_wires, n_ticks, responses, pad_ticks=0, nsigma=3.0, scatter_mode=WCSIM_SCATTER_ATOMIC, stream=None):
        self.handle = wcsim_plan_create_planes(n_wires, n_ticks, responses, pad_ticks, nsigma, scatter_mode, stream)
        self.n_wires, self.n_ticks, self.pad_w, self.pad_t = wcsim_get_dims(self.handle)
        self.n_planes = len(n_wires)


class ImpactPlan(Plan):
    """A plan with sub-wire impact positions (wcsim_plan_create_impact, reading A25): depos in units of pitch / n_impact."""

    def __init__(self, n_wires, n_ticks, responses, pad_ticks=0, nsigma=3.0, scatter_mode=WCSIM_SCATTER_ATOMIC, stream=None):
        self.handle = wcsim_plan_create_impact(n_wires, n_ticks, responses, pad_ticks, nsigma, scatter_mode, stream)
        self.n_wires, self.n_ticks, self.pad_w, self.pad_t = wcsim_get_dims(self.handle)
        self.n_impact = wcsim_get_charge_dims(self.handle)[2]


class Graph:
    """A captured launch sequence of a plan (wcsim_graph_*); keeps the plan alive."""

    def __init__(self, handle, plan):
        self.handle, self.plan = handle, plan

    def launch(self):
        wcsim_graph_launch(self.handle)

    def update(self):
        """Ends a capture begun with plan.graph_begin() and rewrites this graph's parameters with the sequence just
        recorded (new seeds, depo counts, pointers): see wcsim_graph_update in include/wcsim.h."""
        wcsim_graph_update(self.plan.handle, self.handle)

    def destroy(self):
        if self.handle is not None:
            h, self.handle = self.handle, None
            wcsim_graph_destroy(h)

    def __del__(self):
        try:
            if self.plan.handle is not None:
                self.destroy()
        except Exception:
            pass
