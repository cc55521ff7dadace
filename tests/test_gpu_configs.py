"""GPU parity at BASELINE.json's FULL sizes (configs[1..4]), in the launch configuration bench.py times (plan
created with the config's padding, default wire mode, L2 in whatever state the previous call left it).

configs[1..3]: the oracle rasters every depo (seconds), so the fluctuated integer grid S is compared bin by bin over
the whole plane; M is compared over the whole plane with the oracle's FFT route and, on sampled outputs, with the
plain double sum of Eq. (1) -- the definition.
configs[4] (10 M depos, 2560 x 9600): the oracle re-evaluates S on sampled WINDOWS from the depos that can reach them
(wco_raster_scatter's window arguments; the same Philox words since the key is the absolute bin), and M on sampled
interior points of those windows by the double sum.  Properties that hold at any size cover the rest of the grid:
S integer valued, its total equal to the sum of the per-depo totals, within 3 sigma of sum N p.

Tolerances (BASELINE.json north_star): integer grids equal, flipped bins <= 1e-6 of drawn bins; M rel-L2 <= 1e-5 and
max-abs <= 1e-4 max|M|; noise alone by the same two bounds.  Every measured figure is recorded
(conftest.record) and written to gpurun_out/parity_measured.json."""
import math

import numpy as np
import pytest

from conftest import record

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

REL_L2, MAX_ABS, FLIP_BUDGET = 1e-5, 1e-4, 1e-6


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (run with -m gpu on the B200 box)")
    from paper_2203_02479_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def O():
    import oracle
    oracle.lib()
    return oracle


def to_dev(depos):
    return {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in depos.items()}


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def check_M(got, ref, what):
    got = np.asarray(got, dtype=np.float64)
    r, m, scale = rel_l2(got, ref), float(np.max(np.abs(got - ref))), float(np.max(np.abs(ref)))
    record(what, rel_l2=r, max_abs_over_scale=m / max(scale, 1e-300), outputs=int(got.size))
    assert r <= REL_L2, "%s: rel-L2 %.3e" % (what, r)
    assert m <= MAX_ABS * scale, "%s: max-abs %.3e vs scale %.3e" % (what, m, scale)


def points_close(got, ref, M_full, what):
    """sampled outputs: max-abs as for the whole plane; the rel-L2 budget scaled to the sample, i.e. the squared
    error allowed on n of M.size outputs is n / M.size of the whole plane's (REL_L2 |M|)^2"""
    got, ref = np.asarray(got, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    scale = float(np.max(np.abs(M_full)))
    assert float(np.max(np.abs(got - ref))) <= MAX_ABS * scale, what
    budget = REL_L2 * math.sqrt(got.size / M_full.size) * float(np.linalg.norm(M_full.astype(np.float64)))
    err = float(np.linalg.norm(got - ref))
    record(what, sampled_outputs=int(got.size), l2_err_over_budget=err / max(budget, 1e-300),
           max_abs_over_scale=float(np.max(np.abs(got - ref))) / max(scale, 1e-300))
    assert err <= budget, (what, err, budget)


def check_points(O, S_ref, R, M_gpu, rng, n_pts, what):
    """M at sampled outputs against the plain double sum over the oracle's S (the definition, Eq. 1)."""
    nw, nt = S_ref.shape
    px = rng.integers(0, nw, n_pts)
    pt = rng.integers(0, nt, n_pts)
    points_close(M_gpu[px, pt], O.convolve_points(S_ref, R, px, pt), M_gpu, what)


def expected_charge(depos, n_wires, n_ticks, nsigma=3.0):
    """sum over in-grid bins of N p per depo, from the telescoped erf sums (a property check, not the oracle)."""
    from scipy.special import erf
    t0, x0 = depos["t0"].astype(np.float64), depos["x0"].astype(np.float64)
    st, sx = depos["sigma_t"].astype(np.float64), depos["sigma_x"].astype(np.float64)
    N = np.floor(np.abs(depos["q"].astype(np.float64)) + 0.5) * np.sign(depos["q"])

    def axis(c, s, n):
        lo = np.clip(np.floor(c - nsigma * s), 0, n)
        hi = np.clip(np.floor(c + nsigma * s) + 1.0, 0, n)
        with np.errstate(divide="ignore", invalid="ignore"):
            w = 0.5 * (erf((hi - c) / (math.sqrt(2.0) * s)) - erf((lo - c) / (math.sqrt(2.0) * s)))
        inside = (np.floor(c) >= lo) & (np.floor(c) < hi)
        w = np.where(s < 1e-6, inside.astype(np.float64), w)
        return np.where(hi > lo, w, 0.0)

    p = axis(t0, st, n_ticks) * axis(x0, sx, n_wires)
    return float(np.sum(N * p)), float(np.sum(np.abs(N) * p))


def run_plane(B, pl, cfg, *, fluctuate, mode=0, want_totals=False, noise=False, convolve=True):
    plan = B.Plan(pl["n_wires"], pl["n_ticks"], pl["response"], pad=(pl["pad_w"], pl["pad_t"]), nsigma=cfg["nsigma"],
                  scatter_mode=mode)
    d = to_dev(pl["depos"])
    n = pl["depos"]["t0"].shape[0]
    totals = torch.zeros(n, dtype=torch.int32, device="cuda") if want_totals else None
    plan.clear()
    plan.raster_scatter(d, seed=pl["fluct_seed"], fluctuate=fluctuate, dev_depo_totals=totals)
    if noise:
        plan.arm_noise(None, seed=pl["noise_seed"])
    if convolve:
        plan.convolve()
    plan.sync()
    S = plan.charge().cpu().numpy()
    M = plan.output().cpu().numpy() if convolve else None
    st = plan.stats()
    plan.destroy()
    return S, M, (totals.cpu().numpy() if want_totals else None), st


# ---------------------------------------------------------------------------------------------------------------
# configs[1] and configs[2]: whole plane
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("idx", [1, 2])
def test_config_1_2_full(B, O, idx):
    from paper_2203_02479_b200 import synth
    cfg = synth.config(idx)
    pl = cfg["planes"][0]
    nw, nt, R = pl["n_wires"], pl["n_ticks"], pl["response"]
    S_ref, tot_ref, st = O.raster_scatter(nw, nt, pl["depos"], seed=pl["fluct_seed"], fluctuate=True,
                                          nsigma=cfg["nsigma"], want_totals=True)
    assert float(np.max(np.abs(S_ref))) < 2 ** 24  # fp32 adds of integers stay exact (reading A9)
    S, M, tot, stats = run_plane(B, pl, cfg, fluctuate=True, want_totals=True)
    flipped = int(np.count_nonzero(S.astype(np.float64) != S_ref))
    record("configs[%d] S" % idx, flipped_bins=flipped, drawn_bins=int(st["drawn"]))
    assert flipped <= FLIP_BUDGET * st["drawn"], (flipped, st["drawn"])
    assert int(np.count_nonzero(tot != tot_ref)) <= flipped
    assert stats["bins_drawn"] == st["drawn"]
    mean, var = expected_charge(pl["depos"], nw, nt)
    assert abs(float(S.astype(np.float64).sum()) - mean) <= 3.0 * math.sqrt(var) + 1.0
    # M: whole plane against the oracle's FFT route, sampled outputs against the definition
    M_ref = O.convolve_fft(S_ref, R, pl["pad_w"], pl["pad_t"])
    check_M(M, M_ref, "configs[%d] M" % idx)
    check_points(O, S_ref, R, M, np.random.default_rng(idx), 4000, "configs[%d] M at sampled outputs" % idx)
    # deterministic tiled mode gives the same integer grid
    S2, _, _, _ = run_plane(B, pl, cfg, fluctuate=True, mode=B.WCSIM_SCATTER_TILED, convolve=False)
    assert int(np.count_nonzero(S2.astype(np.float64) != S_ref)) <= FLIP_BUDGET * st["drawn"]


# ---------------------------------------------------------------------------------------------------------------
# configs[3]: three planes, own responses, per-wire noise
# ---------------------------------------------------------------------------------------------------------------
def test_config_3_full(B, O):
    from paper_2203_02479_b200 import synth
    cfg = synth.config(3)
    assert cfg["noise"] and len(cfg["planes"]) == 3
    for p, pl in enumerate(cfg["planes"]):
        nw, nt, R = pl["n_wires"], pl["n_ticks"], pl["response"]
        S_ref, _, st = O.raster_scatter(nw, nt, pl["depos"], seed=pl["fluct_seed"], fluctuate=True, nsigma=cfg["nsigma"])
        S, M, _, _ = run_plane(B, pl, cfg, fluctuate=True)
        flipped = int(np.count_nonzero(S.astype(np.float64) != S_ref))
        record("configs[3] plane %d S" % p, flipped_bins=flipped, drawn_bins=int(st["drawn"]))
        assert flipped <= FLIP_BUDGET * st["drawn"]
        M_ref = O.convolve_fft(S_ref, R, pl["pad_w"], pl["pad_t"])
        check_M(M, M_ref, "configs[3] plane %d M" % p)
        check_points(O, S_ref, R, M, np.random.default_rng(30 + p), 2000, "configs[3] plane %d points" % p)
        # signal + noise in one pass (noise rides the inverse row transform): M' = M + N within M's tolerance
        _, Mn, _, _ = run_plane(B, pl, cfg, fluctuate=True, noise=True)
        N_ref = O.noise_add(np.zeros((nw, nt)), pl["pad_t"], pl["noise_seed"])
        check_M(Mn, M_ref + N_ref, "configs[3] plane %d M + N" % p)
        # noise on its own (S = 0 => M = N): it is invisible against 1e-4 max|M| otherwise
        plan = B.Plan(nw, nt, R, pad=(pl["pad_w"], pl["pad_t"]))
        plan.clear()
        plan.arm_noise(None, seed=pl["noise_seed"])
        plan.convolve()
        plan.sync()
        N = plan.output().cpu().numpy().astype(np.float64)
        plan.destroy()
        check_M(N, N_ref, "configs[3] plane %d noise alone" % p)
        rms = float(np.sqrt(np.mean(N ** 2)))
        assert abs(rms - 0.4743) < 0.01  # reading A15


# ---------------------------------------------------------------------------------------------------------------
# configs[4]: sampled windows, both scatter modes
# ---------------------------------------------------------------------------------------------------------------
def _reach(depos, nsigma, w0, w1, k0, k1):
    """depos whose +-n sigma patch (snapped outward, reading A2) can touch the window; conservative by one bin"""
    t0, x0, st, sx = (depos[k].astype(np.float64) for k in ("t0", "x0", "sigma_t", "sigma_x"))
    sel = (t0 + nsigma * st + 2 >= k0) & (t0 - nsigma * st - 2 < k1) & (x0 + nsigma * sx + 2 >= w0) & (x0 - nsigma * sx - 2 < w1)
    return np.nonzero(sel)[0]


def test_config_4_windows_both_modes(B, O):
    from paper_2203_02479_b200 import synth
    cfg = synth.config(4)
    pl = cfg["planes"][0]
    nw, nt, R = pl["n_wires"], pl["n_ticks"], pl["response"]
    n = pl["depos"]["t0"].shape[0]
    assert (nw, nt, n, R.shape) == (2560, 9600, 10_000_000, (41, 400))
    S, M, tot, stats = run_plane(B, pl, cfg, fluctuate=True, want_totals=True)
    S2, _, _, _ = run_plane(B, pl, cfg, fluctuate=True, mode=B.WCSIM_SCATTER_TILED, convolve=False)
    # properties over the whole grid
    S64 = S.astype(np.float64)
    assert np.array_equal(S, np.rint(S)) and float(np.max(np.abs(S))) < 2 ** 24
    assert int(S64.sum()) == int(tot.astype(np.int64).sum())
    assert np.array_equal(S, S2), "atomic and tiled scatter disagree"
    mean, var = expected_charge(pl["depos"], nw, nt)
    assert abs(float(S64.sum()) - mean) <= 3.0 * math.sqrt(var) + 1.0
    # sampled windows: S bin by bin, per-depo totals of depos wholly inside, M on interior points by the double sum
    rng = np.random.default_rng(4)
    WW, WT = 192, 1280
    c = (R.shape[0] - 1) // 2
    drawn = flipped = 0
    corners = [(0, 0), (nw - WW, nt - WT), (0, nt - WT)] + [(int(rng.integers(0, nw - WW)), int(rng.integers(0, nt - WT))) for _ in range(5)]
    for w0, k0 in corners:
        w1, k1 = w0 + WW, k0 + WT
        idx = _reach(pl["depos"], cfg["nsigma"], w0, w1, k0, k1)
        sub = {k: v[idx] for k, v in pl["depos"].items()}
        S_ref, _, st = O.raster_scatter(nw, nt, sub, seed=pl["fluct_seed"], fluctuate=True, nsigma=cfg["nsigma"],
                                        ids=idx.astype(np.uint64), window=(w0, w1, k0, k1))
        drawn += st["drawn"]
        flipped += int(np.count_nonzero(S64[w0:w1, k0:k1] != S_ref))
        # interior outputs whose whole response footprint lies in the window (or beyond the grid edge, where S = 0)
        lo_w = w0 + (c if w0 > 0 else 0)
        hi_w = w1 - (c if w1 < nw else 0)
        lo_t = k0 + (R.shape[1] - 1 if k0 > 0 else 0)
        px = rng.integers(lo_w, hi_w, 600)
        pt = rng.integers(lo_t, k1, 600)
        # embed the window in a frame that keeps the grid-edge behaviour: convolve_points treats outside as zero
        ref = O.convolve_points(S_ref, R, px - w0, pt - k0)
        points_close(M[px, pt], ref, M, "configs[4] window (%d, %d)" % (w0, k0))
    assert drawn > 1_000_000
    record("configs[4] S, 8 windows", flipped_bins=flipped, drawn_bins=int(drawn))
    assert flipped <= FLIP_BUDGET * drawn, (flipped, drawn)
    assert stats["depos_skipped"] == 0


def test_config_4_whole_plane(B, O):
    """configs[4] over the WHOLE plane (north_star: "all five configs match the oracle"): the oracle rasters all 10 M
    depos (about a minute) and convolves by its FFT route on the 4096 x 16384 padded grid; S is compared bin by bin in the
    atomic and the fixed-point scatter modes (the tiled mode is compared with the atomic grid above), per-depo totals depo
    by depo, M over all 24.6 M outputs by north_star's two bounds."""
    from paper_2203_02479_b200 import synth
    cfg = synth.config(4)
    pl = cfg["planes"][0]
    nw, nt, R = pl["n_wires"], pl["n_ticks"], pl["response"]
    S_ref, tot_ref, st = O.raster_scatter(nw, nt, pl["depos"], seed=pl["fluct_seed"], fluctuate=True,
                                          nsigma=cfg["nsigma"], want_totals=True)
    assert float(np.max(np.abs(S_ref))) < 2 ** 24  # fp32 adds of integers stay exact (reading A9)
    M = None
    for mode, name in ((B.WCSIM_SCATTER_ATOMIC, "atomic"), (B.WCSIM_SCATTER_FIXED, "fixed")):
        S, Mm, tot, stats = run_plane(B, pl, cfg, fluctuate=True, mode=mode, want_totals=True,
                                      convolve=(mode == B.WCSIM_SCATTER_ATOMIC))
        flipped = int(np.count_nonzero(S.astype(np.float64) != S_ref))
        record("configs[4] S whole plane, %s" % name, flipped_bins=flipped, drawn_bins=int(st["drawn"]),
               depos_with_other_total=int(np.count_nonzero(tot != tot_ref)))
        assert flipped <= FLIP_BUDGET * st["drawn"], (name, flipped, st["drawn"])
        assert int(np.count_nonzero(tot != tot_ref)) <= flipped
        assert stats["bins_drawn"] == st["drawn"] and stats["depos_skipped"] == 0
        if Mm is not None:
            M = Mm
        del S, tot
    M_ref = O.convolve_fft(S_ref, R, pl["pad_w"], pl["pad_t"])
    check_M(M, M_ref, "configs[4] M whole plane")
