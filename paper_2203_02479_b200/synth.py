"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds none of the method's arithmetic: it only draws the depositions
(centre, widths, charge) and tabulates the detector response that both the CUDA
path and the test oracle receive as plain arrays.  The paper's GEANT4 data set
 is not available; these events stand in for it with the shapes
BASELINE.json `configs` prescribe (recipe: DESIGN.md "Input recipe").
It imports neither the CUDA binding nor oracle/.
"""
from __future__ import annotations

import numpy as np

# BASELINE.json configs[1]: D_L = 4, D_T = 8.8 cm^2/s, v_drift = 0.16 cm/us, pitch 0.5 cm, tick 0.5 us
_DL, _DT, _VDRIFT, _PITCH, _TICK = 4.0, 8.8, 0.16, 0.5, 0.5


def response(n_rwires: int = 21, n_rticks: int = 200, unipolar: bool = False) -> np.ndarray:
    """R[dx + c][dt], tick fastest: exp(-x^2/4.5) (t/8)^4 exp(-t/8) (1 - t/40)  (configs[0]);
    the collection-plane variant drops the last factor (configs[3])."""
    c = (n_rwires - 1) // 2
    x = np.arange(-c, c + 1, dtype=np.float64)[:, None]
    t = np.arange(n_rticks, dtype=np.float64)[None, :]
    r = np.exp(-x * x / 4.5) * (t / 8.0) ** 4 * np.exp(-t / 8.0)
    if not unipolar:
        r = r * (1.0 - t / 40.0)
    return np.ascontiguousarray(r.astype(np.float32))


def response_impact(n_impact: int, n_rwires: int = 21, n_rticks: int = 200, unipolar: bool = False) -> np.ndarray:
    """R[k][dx + c][dt] for n_impact impact positions per wire (reading A25): the analytic form of configs[0] evaluated at
    the distance between the target wire and the source position, x = dx - delta_k, delta_k = (k + 1/2)/n_impact - 1/2
    (position k of a wire sits delta_k pitches from that wire's centre)."""
    c = (n_rwires - 1) // 2
    k = np.arange(n_impact, dtype=np.float64)[:, None, None]
    x = np.arange(-c, c + 1, dtype=np.float64)[None, :, None] - ((k + 0.5) / n_impact - 0.5)
    t = np.arange(n_rticks, dtype=np.float64)[None, None, :]
    r = np.exp(-x * x / 4.5) * (t / 8.0) ** 4 * np.exp(-t / 8.0)
    if not unipolar:
        r = r * (1.0 - t / 40.0)
    return np.ascontiguousarray(r.astype(np.float32))


def to_impact_units(depos: dict, n_impact: int) -> dict:
    """The same depos with x0 and sigma_x in units of pitch / n_impact (what a plan with impact positions takes)."""
    out = dict(depos)
    for key in ("x0", "sigma_x"):
        out[key] = np.ascontiguousarray((depos[key].astype(np.float64) * n_impact).astype(np.float32))
    return out


def _rng(gen_seed: int, plane: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=np.array([gen_seed, 0x47454E00 + plane], dtype=np.uint64)))


def _charge(rng, n):
    return np.exp(np.log(5000.0) + 0.5 * rng.standard_normal(n))


def _pack(t0, x0, st, sx, q):
    f = lambda a: np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))
    return {"t0": f(t0), "x0": f(x0), "sigma_t": f(st), "sigma_x": f(sx), "q": f(q)}


def depos_uniform_box(n, gen_seed=1, plane=0):
    """configs[0]: t0~U[50,450), x0~U[8,56), sigma_t~U[0.5,3], sigma_x~U[0.3,2], Q~LogNormal(5000, 0.5)."""
    rng = _rng(gen_seed, plane)
    t0 = rng.uniform(50.0, 450.0, n)
    x0 = rng.uniform(8.0, 56.0, n)
    st = rng.uniform(0.5, 3.0, n)
    sx = rng.uniform(0.3, 2.0, n)
    return _pack(t0, x0, st, sx, _charge(rng, n))


def depos_tracks(n, n_wires, n_ticks, line_frac, n_seg, td_max_ms, gen_seed=1, plane=0, sigma_scale=1.0,
                 shuffle=False):
    """configs[1]-[4]: `line_frac` of the depos at 0.3-tick spacing along `n_seg` straight segments
    (equal count each, stored consecutively), the rest uniform over the grid; drift time
    td~U[0,td_max) per depo gives sigma_t = sqrt(2 D_L td)/v_drift/tick, sigma_x = sqrt(2 D_T td)/pitch."""
    rng = _rng(gen_seed, plane)
    per = int(round(n * line_frac)) // n_seg
    n_line = per * n_seg
    n_uni = n - n_line
    ta = rng.uniform(0.0, max(n_ticks - 0.3 * per, 1.0), n_seg)
    xa = rng.uniform(0.0, n_wires, n_seg)
    xb = rng.uniform(0.0, n_wires, n_seg)
    k = np.arange(per, dtype=np.float64)[None, :]
    t_line = (ta[:, None] + 0.3 * k).reshape(-1)
    x_line = (xa[:, None] + (xb - xa)[:, None] * k / per).reshape(-1)
    t0 = np.concatenate([t_line, rng.uniform(0.0, n_ticks, n_uni)])
    x0 = np.concatenate([x_line, rng.uniform(0.0, n_wires, n_uni)])
    td = rng.uniform(0.0, td_max_ms * 1e-3, n)  # seconds
    st = np.sqrt(2.0 * _DL * td) / _VDRIFT / _TICK * sigma_scale   # cm / (cm/us) / (us/tick)
    sx = np.sqrt(2.0 * _DT * td) / _PITCH * sigma_scale
    q = _charge(rng, n)
    if shuffle:
        perm = rng.permutation(n)
        t0, x0, st, sx, q = t0[perm], x0[perm], st[perm], sx[perm], q[perm]
    return _pack(t0, x0, st, sx, q)


def _with_plane_seeds(cfg: dict) -> dict:
    """Every plane dict carries fluct_seed and noise_seed (the event's own where the plane names none)."""
    for pl in cfg["planes"]:
        pl.setdefault("fluct_seed", cfg["fluct_seed"])
        pl.setdefault("noise_seed", cfg["noise_seed"])
    return cfg


def config(i: int, *, n_depos: int | None = None, shuffle: bool = False, sigma_scale: float = 1.0) -> dict:
    """The workload of BASELINE.json configs[i] as a dict:
    planes: list of dict(n_wires, n_ticks, pad_w, pad_t, response, depos); fluctuate, noise, seeds, nsigma.
    `n_depos` overrides the per-plane depo count (bounded samples of the same distribution)."""
    base = {"nsigma": 3.0, "fluct_seed": 1, "noise_seed": 1, "gen_seed": 1, "noise": False}
    if i == 0:
        n = n_depos or 100
        planes = [dict(n_wires=64, n_ticks=512, pad_w=128, pad_t=1024, response=response(),
                       depos=depos_uniform_box(n))]
        return _with_plane_seeds({**base, "name": "configs[0] tiny 64x512, 100 depos", "fluctuate": False, "planes": planes})
    if i in (1, 2):
        n = n_depos or (100_000 if i == 1 else 1_000_000)
        frac, nseg, td = (0.9, 50, 2.25) if i == 1 else (0.8, 500, 4.5)
        nseg = max(1, min(nseg, n // 200))
        planes = [dict(n_wires=800, n_ticks=6000, pad_w=1024, pad_t=8192, response=response(),
                       depos=depos_tracks(n, 800, 6000, frac, nseg, td, shuffle=shuffle, sigma_scale=sigma_scale))]
        return _with_plane_seeds({**base, "name": "configs[%d] 800x6000, %d depos" % (i, n), "fluctuate": True, "planes": planes})
    if i == 3:
        n = n_depos or 200_000
        planes = []
        for p, nw in enumerate((800, 800, 960)):
            nseg = max(1, min(100, n // 200))
            # every plane has its own fluctuation and noise seed (reading A26: the planes of an anode are independent,
            # PAPER.md:30, so wire x of U, V and W must not carry the same noise waveform); plane 0 keeps the event's
            planes.append(dict(n_wires=nw, n_ticks=6000, pad_w=1024, pad_t=8192, response=response(unipolar=(p == 2)),
                               depos=depos_tracks(n, nw, 6000, 0.9, nseg, 2.25, plane=p, shuffle=shuffle),
                               fluct_seed=base["fluct_seed"] + 0x1000 * p, noise_seed=base["noise_seed"] + 0x1000 * p))
        return _with_plane_seeds({**base, "name": "configs[3] APA 3 planes x %d depos + noise" % n, "fluctuate": True,
                                  "noise": True, "planes": planes})
    if i == 4:
        n = n_depos or 10_000_000
        nseg = max(1, min(5000, n // 200))
        planes = [dict(n_wires=2560, n_ticks=9600, pad_w=4096, pad_t=16384, response=response(41, 400),
                       depos=depos_tracks(n, 2560, 9600, 0.7, nseg, 4.5, shuffle=shuffle))]
        return _with_plane_seeds({**base, "name": "configs[4] 2560x9600, %d depos" % n, "fluctuate": True, "planes": planes})
    raise ValueError("config index must be 0..4")
