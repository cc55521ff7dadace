"""Pins of the oracle's drift step (reading A22; groups are "diffused into a 2D distribution along the
drifting and wire pitch directions" before the three tasks the paper times)."""
import math

import numpy as np

import oracle as O

K = dict(v_drift=0.16, D_L=4.0, D_T=8.8, tick=0.5, pitch=0.5)  # BASELINE.json configs[1]


def one(x, y=0.0, z=0.0, t=0.0, q=1000.0, **kw):
    a = lambda v: np.array([v], dtype=np.float32)
    out = O.drift(a(x), a(y), a(z), a(t), a(q), **{**K, **kw})
    return {k: float(v[0]) for k, v in out.items()}


def test_widths_of_configs_1_at_its_longest_drift():
    """BASELINE.json configs[1]: td ~ U[0, 2.25 ms] 'giving sigma_t = sqrt(2 D_L td)/v_drift and sigma_x = sqrt(2 D_T td)/pitch';
    SURVEY 8(a) evaluates them at td = 2.25 ms: sigma_t <= 1.677 ticks, sigma_x <= 0.398 pitch."""
    x = 0.16 * 2250.0  # cm travelled in 2.25 ms at 0.16 cm/us
    r = one(x)
    assert abs(r["sigma_t"] - 1.677) < 5e-4
    assert abs(r["sigma_x"] - 0.398) < 5e-4
    assert abs(r["t0"] - 2250.0 / 0.5) < 1e-2  # 4500 ticks of drift


def test_closed_forms_and_projection():
    rng = np.random.default_rng(2)
    n = 2000
    x = rng.uniform(2, 360, n).astype(np.float32)
    y = rng.uniform(-300, 300, n).astype(np.float32)
    z = rng.uniform(0, 700, n).astype(np.float32)
    t = rng.uniform(0, 100, n).astype(np.float32)
    q = rng.lognormal(np.log(5000), 0.5, n).astype(np.float32)
    th = math.radians(35.7)
    out = O.drift(x, y, z, t, q, **K, t_origin=-10.0, lifetime=3000.0, x_plane=1.5, cos_theta=math.cos(th),
                  sin_theta=math.sin(th), pitch_origin=-250.0)
    td = (x.astype(np.float64) - 1.5) / 0.16
    assert np.allclose(out["t0"], (t + td + 10.0) / 0.5, rtol=1e-6)
    assert np.allclose(out["x0"], (y * math.cos(th) + z * math.sin(th) + 250.0) / 0.5, rtol=1e-6, atol=1e-4)
    # sigma^2 grows linearly with the drift time, in the ratio D_L : D_T once the units are undone
    st_cm = out["sigma_t"].astype(np.float64) * 0.5 * 0.16
    sx_cm = out["sigma_x"].astype(np.float64) * 0.5
    assert np.allclose(st_cm ** 2, 2 * 4.0e-6 * td, rtol=1e-5)
    assert np.allclose(sx_cm ** 2 / st_cm ** 2, 8.8 / 4.0, rtol=1e-5)
    assert np.allclose(out["q"], q * np.exp(-td / 3000.0), rtol=1e-6)
    # rotating the wire direction by 90 degrees swaps the roles of y and z
    o2 = O.drift(x, y, z, t, q, **K, cos_theta=0.0, sin_theta=1.0)
    assert np.allclose(o2["x0"], z / 0.5, rtol=1e-6)


def test_edge_cases():
    r = one(0.0)  # on the plane: no drift, no diffusion, no attenuation
    assert r["sigma_t"] == 0.0 and r["sigma_x"] == 0.0 and r["t0"] == 0.0 and r["q"] == 1000.0
    r = one(-1.0)  # behind the plane
    assert all(math.isnan(v) for v in r.values())
    r = one(16.0, lifetime=0.0)
    assert r["q"] == 1000.0
    r = one(16.0, lifetime=100.0)  # td = 100 us = one lifetime
    assert abs(r["q"] - 1000.0 / math.e) < 1e-3


def test_drifted_groups_raster_like_hand_made_depos():
    """drift -> raster equals raster of the same (t0, x0, sigma, Q) written by hand."""
    r = one(100.0, y=12.3, t=5.0, q=4000.0)
    d = {k: np.array([v], dtype=np.float32) for k, v in r.items()}
    S, _, _ = O.raster_scatter(64, 2048, d, fluctuate=False)
    assert abs(S.sum() - 4000.0) < 0.02 * 4000.0
    wire = np.argmax(S.sum(axis=1))
    assert wire == int(math.floor(r["x0"]))
