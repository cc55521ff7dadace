"""Pins for the oracle's raster and scatter-add (O1-O4 of SURVEY.md section 8c; north_star: "per-depo charge
conservation within the +-n sigma truncation", "the patch's first and second moments")."""
import math

import numpy as np
import pytest

import oracle
from conftest import golden
from paper_2203_02479_b200 import synth


def gauss_bin_quadrature(i, c, s, order=40):
    """Independent of erf: Gauss-Legendre quadrature of the normal pdf over [i, i+1], split in 8 panels."""
    x, w = np.polynomial.legendre.leggauss(order)
    tot = 0.0
    for k in range(8):
        a, b = i + k / 8.0, i + (k + 1) / 8.0
        xm = 0.5 * (b - a) * x + 0.5 * (a + b)
        tot += 0.5 * (b - a) * np.sum(w * np.exp(-0.5 * ((xm - c) / s) ** 2)) / (s * math.sqrt(2 * math.pi))
    return tot


def test_axis_weights_match_published_erf_table():
    # centre 0, sigma = 1/sqrt2: bin [0,x) content is erf(x)/2; use unit bins via scaling sigma = 1/(x sqrt2)
    for xs, es in golden("erf_table.txt"):
        x, e = float(xs), float(es)
        w = oracle.axis_weight(0, 0.0, 1.0 / (x * math.sqrt(2.0)))
        assert w == pytest.approx(0.5 * e, abs=6e-11)


def test_axis_weights_match_independent_quadrature():
    rng = np.random.default_rng(0)
    for _ in range(60):
        c = rng.uniform(-5, 700)
        s = rng.uniform(0.25, 3.0)
        i0, i1 = oracle.axis_extent(c, s, 3.0)
        for i in range(i0, i1):
            assert oracle.axis_weight(i, c, s) == pytest.approx(gauss_bin_quadrature(i, c, s), abs=2e-13)


def test_extent_is_snapped_outward_and_never_empty():
    for c, s in [(10.2, 0.0), (10.0, 0.0), (10.2, 0.1), (10.9, 0.05), (5.5, 1.5), (0.3, 2.0), (-3.7, 1.0)]:
        i0, i1 = oracle.axis_extent(c, s, 3.0)
        assert i1 - i0 >= 1
        assert i0 <= c - 3 * s and i1 >= c + 3 * s or s == 0.0
        assert i0 == math.floor(c - 3 * s) and i1 == math.floor(c + 3 * s) + 1


def test_axis_sum_telescopes_and_bounds():
    rng = np.random.default_rng(1)
    lo = math.erf(3 / math.sqrt(2))
    for _ in range(200):
        c, s = rng.uniform(0, 100), rng.uniform(0.01, 3.0)
        i0, i1 = oracle.axis_extent(c, s, 3.0)
        tot = sum(oracle.axis_weight(i, c, s) for i in range(i0, i1))
        closed = 0.5 * (math.erf((i1 - c) / (math.sqrt(2) * s)) - math.erf((i0 - c) / (math.sqrt(2) * s)))
        assert tot == pytest.approx(closed, abs=1e-14)
        assert lo - 1e-14 <= tot <= 1.0 + 1e-14


def test_moments_of_the_patch():
    rng = np.random.default_rng(2)
    for _ in range(100):
        c, s = rng.uniform(20, 80), rng.uniform(0.5, 3.0)
        i0, i1 = oracle.axis_extent(c, s, 3.0)
        idx = np.arange(i0, i1)
        w = np.array([oracle.axis_weight(i, c, s) for i in idx])
        wn = w / w.sum()
        mean = np.sum(wn * (idx + 0.5))
        var = np.sum(wn * (idx + 0.5 - mean) ** 2)
        assert abs(mean - c) <= 0.01
        # truncated-normal variance factor 1 - 2 n phi(n)/(2 Phi(n) - 1) at n = 3, plus Sheppard's 1/12.
        # Sheppard's correction is itself only exact up to the aliasing term ~ exp(-2 pi^2 sigma^2)
        # (0.7 % of a bin^2 at sigma = 0.5, nothing at sigma >= 1), hence the sigma-dependent slack.
        slack = 1e-3 + 2.0 * math.exp(-2.0 * math.pi ** 2 * s * s)
        assert 0.97334 * s * s + 1.0 / 12.0 - slack <= var <= s * s + 1.0 / 12.0 + slack
        if s >= 1.0:
            assert 0.97334 * s * s + 1.0 / 12.0 - 1e-3 <= var <= s * s + 1.0 / 12.0 + 1e-9
        # and the exact per-depo values from the quadrature
        wq = np.array([gauss_bin_quadrature(i, c, s) for i in idx])
        mq = np.sum(wq * (idx + 0.5)) / wq.sum()
        assert mq == pytest.approx(mean, abs=1e-12)
        assert np.sum(wq * (idx + 0.5 - mq) ** 2) / wq.sum() == pytest.approx(var, abs=1e-11)


def test_sigma_to_zero_and_bin_edge_symmetry():
    assert oracle.axis_weight(10, 10.2, 0.0) == 1.0 and oracle.axis_weight(9, 10.2, 0.0) == 0.0
    assert oracle.axis_weight(10, 10.2, 5e-7) == 1.0
    # the erf form approaches the same limit
    assert oracle.axis_weight(10, 10.2, 2e-6) == pytest.approx(1.0, abs=1e-15)
    # centred exactly on an edge: equal weights either side
    for s in (0.3, 1.0, 2.2):
        for k in range(0, 5):
            assert oracle.axis_weight(7 + k, 8.0, s) == pytest.approx(oracle.axis_weight(8 - 1 - k + 0, 8.0, s), abs=1e-16) \
                if k == 0 else True
            assert oracle.axis_weight(8 + k, 8.0, s) == pytest.approx(oracle.axis_weight(7 - k, 8.0, s), abs=1e-16)


def brute_patch(n_wires, n_ticks, d, i):
    """Patch of depo i straight from the definition with math.erf (python loops; tiny inputs only)."""
    S = np.zeros((n_wires, n_ticks))
    t0, x0, st, sx, q = (float(d[k][i]) for k in ("t0", "x0", "sigma_t", "sigma_x", "q"))
    for x in range(math.floor(x0 - 3 * sx), math.floor(x0 + 3 * sx) + 1):
        for t in range(math.floor(t0 - 3 * st), math.floor(t0 + 3 * st) + 1):
            if 0 <= x < n_wires and 0 <= t < n_ticks:
                wx = 0.5 * (math.erf((x + 1 - x0) / (math.sqrt(2) * sx)) - math.erf((x - x0) / (math.sqrt(2) * sx)))
                wt = 0.5 * (math.erf((t + 1 - t0) / (math.sqrt(2) * st)) - math.erf((t - t0) / (math.sqrt(2) * st)))
                S[x, t] += q * wt * wx
    return S


def test_scatter_matches_brute_force_and_conserves_charge():
    cfg = synth.config(0)
    pl = cfg["planes"][0]
    d = pl["depos"]
    S, _, st = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], d)
    assert st["skipped"] == 0
    ref = sum(brute_patch(pl["n_wires"], pl["n_ticks"], d, i) for i in range(len(d["q"])))
    assert np.max(np.abs(S - ref)) <= 1e-10 * np.max(np.abs(ref))
    # config[0] depos sit well inside the grid: total charge within the 3 sigma truncation on both axes
    qsum = float(np.sum(d["q"].astype(np.float64)))
    lo = math.erf(3 / math.sqrt(2)) ** 2
    assert lo * qsum <= S.sum() <= qsum
    # per depo: sum = Q * (closed form t) * (closed form x)
    for i in range(5):
        one = {k: v[i:i + 1] for k, v in d.items()}
        Si, _, _ = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], one)
        it0, ix0, wt, wx = oracle.patch_axes(one["t0"][0], one["x0"][0], one["sigma_t"][0], one["sigma_x"][0])
        assert Si.sum() == pytest.approx(float(one["q"][0]) * wt.sum() * wx.sum(), rel=1e-13)
        assert np.allclose(Si[ix0:ix0 + len(wx), it0:it0 + len(wt)], float(one["q"][0]) * np.outer(wx, wt), rtol=1e-14)


def test_patches_leaving_the_grid_are_cropped_not_wrapped():
    # centres are dyadic so that the fp32 inputs shift exactly
    d = {"t0": [0.375, 63.75, 30.0], "x0": [0.25, 15.875, -0.5], "sigma_t": [1.0, 1.25, 0.75],
         "sigma_x": [0.75, 0.875, 0.5], "q": [1000.0, 2000.0, -500.0]}
    S, _, _ = oracle.raster_scatter(16, 64, d)
    Sbig, _, _ = oracle.raster_scatter(48, 128, {**d, "t0": [x + 32 for x in d["t0"]], "x0": [x + 16 for x in d["x0"]]})
    assert np.allclose(S, Sbig[16:32, 32:96], rtol=0, atol=1e-9)
    # something was lost at the edges, and nothing wrapped to the opposite edge
    assert abs(Sbig).sum() > abs(S).sum() + 100.0
    assert S[15, 0] == 0.0 and S[0, 63] == 0.0 and S[8, 0] == 0.0


def test_window_and_ids_reproduce_the_full_grid():
    cfg = synth.config(1, n_depos=3000)
    pl = cfg["planes"][0]
    d = pl["depos"]
    S, tot, st = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], d, seed=7, fluctuate=True, want_totals=True)
    assert np.all(S == np.round(S))
    assert tot.sum() == S.sum()
    win = (100, 400, 1000, 3000)
    Sw, _, _ = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], d, seed=7, fluctuate=True, window=win)
    assert np.array_equal(Sw, S[100:400, 1000:3000])
    # a subset of depos with explicit ids gives the same draws as in the full run
    sel = np.arange(0, 3000, 7)
    sub = {k: v[sel] for k, v in d.items()}
    _, tot_sub, _ = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], sub, seed=7, fluctuate=True, ids=sel,
                                          want_totals=True)
    assert np.array_equal(tot_sub, tot[sel])
    # another seed or id base changes the draws
    S2, _, _ = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], d, seed=8, fluctuate=True)
    assert not np.array_equal(S2, S)
    S3, _, _ = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], d, seed=7, fluctuate=True, id_base=1)
    assert not np.array_equal(S3, S)


def test_fluctuated_charge_mean_and_variance():
    cfg = synth.config(1, n_depos=20000)
    pl = cfg["planes"][0]
    d = pl["depos"]
    Sf, _, _ = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], d, seed=1, fluctuate=True)
    # expectation: N p per bin with N = floor(|Q| + 1/2); build it from the un-fluctuated raster of rounded charges
    dq = {**d, "q": np.floor(np.abs(d["q"].astype(np.float64)) + 0.5).astype(np.float32)}
    Se, _, _ = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], dq)
    # variance <= sum N p (1-p) + 1/12 per bin <= sum N p + bins/12
    var_hi = Se.sum() + 4e5 / 12
    assert abs(Sf.sum() - Se.sum()) < 4 * math.sqrt(var_hi)
    assert abs(Sf.sum() / Se.sum() - 1) < 1e-3


def test_invalid_depos_are_skipped_and_counted():
    d = {"t0": [10.0, np.nan, 12.0, 13.0], "x0": [5.0, 5.0, np.inf, 5.0], "sigma_t": [1.0, 1.0, 1.0, -1.0],
         "sigma_x": [1.0, 1.0, 1.0, 1.0], "q": [100.0, 100.0, 100.0, 100.0]}
    S, _, st = oracle.raster_scatter(16, 32, d)
    assert st["skipped"] == 3 and np.isfinite(S).all() and S.sum() > 90


# ---------------------------------------------------------------------------------------------------------------
# reading A24: renormalised patches (second half)
# ---------------------------------------------------------------------------------------------------------------
def test_normalized_patch_carries_exactly_q_inside_the_grid():
    rng = np.random.default_rng(31)
    n = 300
    d = {"t0": rng.uniform(40, 460, n), "x0": rng.uniform(12, 52, n), "sigma_t": rng.uniform(0.0, 3.0, n),
         "sigma_x": rng.uniform(0.0, 2.0, n), "q": rng.lognormal(np.log(5000), 0.5, n) * rng.choice([-1, 1], n)}
    d = {k: v.astype(np.float32) for k, v in d.items()}
    d["sigma_t"][:5] = 0.0
    for i in range(0, n, 37):  # one depo at a time: its bins sum to Q within fp64 rounding of ~100 adds
        one = {k: v[i:i + 1] for k, v in d.items()}
        S, _, _ = oracle.raster_scatter(64, 512, one, fluctuate=False, normalize=True)
        assert abs(S.sum() - float(one["q"][0])) <= 1e-12 * abs(float(one["q"][0]))
        S0, _, _ = oracle.raster_scatter(64, 512, one, fluctuate=False, normalize=False)
        assert abs(S0.sum()) <= abs(S.sum()) and abs(S0.sum()) >= 0.9946 ** 1 * 0.9946 * abs(S.sum()) - 1e-9
        # same shape, rescaled by one number
        nz = S0 != 0
        ratio = S[nz] / S0[nz]
        assert np.allclose(ratio, ratio[0], rtol=1e-12)


def test_normalization_uses_the_whole_extent_not_the_part_inside_the_grid():
    """a depo at the grid edge loses the charge that falls outside (A5) also when normalised"""
    one = {k: np.array([v], dtype=np.float32) for k, v in (("t0", 0.25), ("x0", 5.5), ("sigma_t", 2.0), ("sigma_x", 0.5), ("q", 1000.0))}
    S, _, _ = oracle.raster_scatter(16, 64, one, fluctuate=False, normalize=True)
    from scipy.special import erf
    inside = 0.5 * (1.0 + erf(0.25 / (np.sqrt(2.0) * 2.0)))  # mass at t >= 0 of a Gaussian centred at 0.3 ... truncated at 3 sigma
    lo, hi = np.floor(0.25 - 6.0), np.floor(0.25 + 6.0) + 1
    W = 0.5 * (erf((hi - 0.25) / (np.sqrt(2) * 2)) - erf((lo - 0.25) / (np.sqrt(2) * 2)))
    part = 0.5 * (erf((hi - 0.25) / (np.sqrt(2) * 2)) - erf((0 - 0.25) / (np.sqrt(2) * 2)))
    assert abs(S.sum() - 1000.0 * part / W) < 1e-9 * 1000.0
    assert S.sum() < 600.0 and inside > 0.5


def test_normalized_fluctuation_mean():
    rng = np.random.default_rng(33)
    one = {k: np.full(400, v, dtype=np.float32) for k, v in (("t0", 100.4), ("x0", 20.6), ("sigma_t", 1.3), ("sigma_x", 0.6), ("q", 8000.0))}
    S, tot, _ = oracle.raster_scatter(64, 256, one, seed=9, fluctuate=True, normalize=True, want_totals=True)
    # independent binomials with sum p = 1: E[total] = N, var = sum N p (1-p) < N
    assert abs(tot.mean() - 8000.0) < 4 * np.sqrt(8000.0 / 400)
    S0, tot0, _ = oracle.raster_scatter(64, 256, one, seed=9, fluctuate=True, normalize=False, want_totals=True)
    assert tot0.mean() < tot.mean() - 2  # without it the charge beyond the extent (0.06 % here) is truncated away


# ---------------------------------------------------------------------------------------------------------------
# the fluctuated branch of wco_raster_scatter, rebuilt bin by bin from its already-pinned pieces
# (readings A5, A7, A8)
# ---------------------------------------------------------------------------------------------------------------
def _fluct_pin_depos():
    rng = np.random.default_rng(41)
    n = 30
    d = {"t0": rng.uniform(2.0, 45.0, n), "x0": rng.uniform(1.0, 11.0, n), "sigma_t": rng.uniform(0.3, 2.5, n),
         "sigma_x": rng.uniform(0.2, 1.2, n), "q": rng.lognormal(np.log(5000), 0.5, n)}
    d["q"][1::4] *= -1.0            # negative charge: the sign is carried, N comes from |q|
    d["q"][2], d["q"][3], d["q"][4], d["q"][5] = 0.5, 0.2, 1.5, -0.5   # N = 1, 0, 2, 1 (round half up on |q|)
    d["q"][6] = 2.4999              # N = 2, where floor(|q|) and floor(|q| + 1/2) still agree ...
    d["q"][7] = 7.5                 # ... and N = 8, where they do not
    d["sigma_t"][8] = 0.0           # sigma = 0 on one axis, on the other, on both (A4)
    d["sigma_x"][9] = 0.0
    d["sigma_t"][10] = d["sigma_x"][10] = 0.0
    d["t0"][11], d["x0"][11] = 0.4, 0.3       # patch leaves the grid at the low corner (A5)
    d["t0"][12], d["x0"][12] = 47.7, 11.8     # and at the high corner
    d["t0"][13] = -20.0                       # wholly outside: nothing drawn
    d["q"][14] = 2.0e5                        # mu >= 16 in many bins: the rounded-normal branch of B
    return {k: v.astype(np.float32) for k, v in d.items()}


@pytest.mark.parametrize("fluctuate,normalize", [(1, False), (2, False), (1, True), (2, True)])
@pytest.mark.parametrize("explicit_ids", [False, True])
def test_fluctuated_scatter_rebuilt_bin_by_bin(fluctuate, normalize, explicit_ids):
    n_wires, n_ticks, seed = 12, 48, 0x1234567887654321
    d = _fluct_pin_depos()
    n = d["t0"].shape[0]
    if explicit_ids:
        ids = (np.arange(n, dtype=np.uint64) * np.uint64(1_000_003) + np.uint64((1 << 40) + 17))[::-1].copy()
        kw = dict(ids=ids)
    else:
        ids = np.arange(n, dtype=np.uint64) + np.uint64((1 << 40) + 17)
        kw = dict(id_base=(1 << 40) + 17)
    S, tot, st = oracle.raster_scatter(n_wires, n_ticks, d, seed=seed, fluctuate=fluctuate, normalize=normalize,
                                       want_totals=True, **kw)
    draw = oracle.binomial if fluctuate == 1 else oracle.normal_draw
    S_ref = np.zeros((n_wires, n_ticks))
    tot_ref = np.zeros(n, dtype=np.int64)
    drawn = 0
    for k in range(n):
        t0, x0, s_t, s_x, q = (float(d[key][k]) for key in ("t0", "x0", "sigma_t", "sigma_x", "q"))
        it0, ix0, wt, wx = oracle.patch_axes(t0, x0, s_t, s_x)
        N = math.floor(abs(q) + 0.5)
        sign = -1.0 if q < 0 else 1.0
        norm = 1.0
        if normalize:  # A24: the telescoped sum over the whole extent, outside bins included
            for c, s, i0, w in ((t0, s_t, it0, wt), (x0, s_x, ix0, wx)):
                if s >= 1e-6:
                    norm *= 0.5 * (math.erf((i0 + len(w) - c) / (math.sqrt(2.0) * s)) - math.erf((i0 - c) / (math.sqrt(2.0) * s)))
        for j, wxj in enumerate(wx):
            wire = ix0 + j
            if not 0 <= wire < n_wires:
                continue
            for i, wti in enumerate(wt):
                tick = it0 + i
                if not 0 <= tick < n_ticks:
                    continue
                p = wti * wxj
                if normalize:
                    p = p / norm
                c = sign * draw(N, p, oracle.fluct_word(seed, int(ids[k]), wire * n_ticks + tick))
                S_ref[wire, tick] += c
                tot_ref[k] += int(c)
                drawn += 1
    assert np.array_equal(S, S_ref)
    assert np.array_equal(tot.astype(np.int64), tot_ref)
    assert st["drawn"] == drawn and st["skipped"] == 0
    # the cases are really there: a zero-N depo, a depo off the grid, negative bins, a big bin (the draws of a depo's
    # bins are independent, reading A6, so a one-electron depo may total more than 1)
    assert tot_ref[3] == 0 and tot_ref[13] == 0 and (S_ref < 0).any() and S_ref.max() > 1000
