"""GPU parity of the sub-wire impact-position path (reading A25): the raster on the
n_impact-times finer wire grid against the oracle's raster of that grid, and M against the oracle's plain definition
M[x][t] = sum_k sum_dx sum_dt R_k[dx+c][dt] Sf[(x-dx) K + k][t-dt].  Tolerances are north_star's."""
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


def check_close(got, ref, what):
    got = np.asarray(got, dtype=np.float64)
    r = float(np.linalg.norm((got - ref).ravel()) / max(np.linalg.norm(ref.ravel()), 1e-300))
    m, scale = float(np.max(np.abs(got - ref))), float(np.max(np.abs(ref)))
    record(what, rel_l2=r, max_abs_over_scale=m / max(scale, 1e-300), outputs=int(got.size))
    assert r <= REL_L2, "%s: rel-L2 %.3e" % (what, r)
    assert m <= MAX_ABS * scale, "%s: max-abs %.3e vs scale %.3e" % (what, m, scale)


def fine_depos(rng, n, nw, nt, K):
    d = {"t0": rng.uniform(-3, nt + 3, n), "x0": rng.uniform(-1, nw + 1, n) * K, "sigma_t": rng.uniform(0, 2.5, n),
         "sigma_x": rng.uniform(0, 1.0, n) * K, "q": rng.lognormal(np.log(5000), 0.5, n)}
    d = {k: v.astype(np.float32) for k, v in d.items()}
    d["q"][::5] *= -1
    return d


@pytest.mark.parametrize("K", [1, 2, 4, 10])
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_impact_plan_matches_the_definition(B, O, K, mode):
    from paper_2203_02479_b200 import synth
    rng = np.random.default_rng(100 + K)
    nw, nt = 37, 300
    R = synth.response_impact(K, 5, 24) * rng.uniform(0.5, 1.5, (K, 1, 1)).astype(np.float32)
    d = fine_depos(rng, 1500, nw, nt, K)
    dev = to_dev(d)
    with B.ImpactPlan(nw, nt, R, scatter_mode=mode) as plan:
        assert plan.n_impact == K and tuple(plan.charge().shape) == (nw * K, nt) and tuple(plan.output().shape) == (nw, nt)
        for fluct in (0, 1):
            plan.clear()
            plan.raster_scatter(dev, seed=8, fluctuate=fluct)
            plan.convolve()
            plan.sync()
            S = plan.charge().cpu().numpy().astype(np.float64)
            M = plan.output().cpu().numpy()
            S_ref, _, st = O.raster_scatter(nw * K, nt, d, seed=8, fluctuate=fluct)
            if fluct:
                assert int(np.count_nonzero(S != S_ref)) <= FLIP_BUDGET * st["drawn"]
            else:
                check_close(S, S_ref, "impact K=%d mode %d S" % (K, mode))
            check_close(M, O.convolve_impact(S_ref, R, K), "impact K=%d mode %d fluct %d M" % (K, mode, fluct))
        if K > 1:  # impact positions: the wire axis is always done directly
            with pytest.raises(B.WcsimError):
                plan.set_wire_mode(B.WCSIM_WIRES_FFT)


def test_point_charge_at_impact_position_k_gives_R_k(B):
    from paper_2203_02479_b200 import synth
    K, nw, nt = 5, 30, 400
    R = synth.response_impact(K, 7, 50)
    R[:, :, :] *= np.arange(1, K + 1, dtype=np.float32)[:, None, None]  # positions must not be mixed up
    with B.ImpactPlan(nw, nt, R) as plan:
        for k in range(K):
            xs, ts = 12, 33
            f = np.float32
            d = {"t0": np.array([ts + 0.5], f), "x0": np.array([xs * K + k + 0.5], f), "sigma_t": np.zeros(1, f),
                 "sigma_x": np.zeros(1, f), "q": np.array([1000.0], f)}
            plan.clear()
            plan.raster_scatter(to_dev(d), fluctuate=0)
            plan.convolve()
            plan.sync()
            M = plan.output().cpu().numpy().astype(np.float64)
            expect = np.zeros((nw, nt))
            expect[xs - 3:xs + 4, ts:ts + 50] = 1000.0 * R[k].astype(np.float64)
            assert np.max(np.abs(M - expect)) <= MAX_ABS * np.max(np.abs(expect)), k
            assert np.linalg.norm(M - expect) <= REL_L2 * np.linalg.norm(expect), k


def test_configs1_sized_plane_with_ten_impact_positions(B, O):
    """a configs[1]-sized plane (800 wires x 6000 ticks, 21 x 200 response, 100k depos, fluctuation on) with K = 10 impact
    positions per wire: patches of ~26 fine wires x ~8 ticks ("typically O(20x20) elements")"""
    from paper_2203_02479_b200 import synth
    K = 10
    cfg = synth.config(1)
    pl = cfg["planes"][0]
    nw, nt = pl["n_wires"], pl["n_ticks"]
    R = synth.response_impact(K, 21, 200)
    d = synth.to_impact_units(pl["depos"], K)
    with B.ImpactPlan(nw, nt, R, pad_ticks=pl["pad_t"]) as plan:
        plan.clear()
        plan.raster_scatter(to_dev(d), seed=cfg["fluct_seed"], fluctuate=True)
        plan.convolve()
        plan.sync()
        S = plan.charge().cpu().numpy()
        M = plan.output().cpu().numpy()
        stats = plan.stats()
    S_ref, _, st = O.raster_scatter(nw * K, nt, d, seed=cfg["fluct_seed"], fluctuate=True)
    flipped = int(np.count_nonzero(S.astype(np.float64) != S_ref))
    record("impact K=10 configs[1]-sized S", flipped_bins=flipped, drawn_bins=int(st["drawn"]),
           bins_per_depo=st["drawn"] / d["t0"].shape[0])
    assert flipped <= FLIP_BUDGET * st["drawn"] and stats["bins_drawn"] == st["drawn"]
    assert st["drawn"] / d["t0"].shape[0] > 100  # patches of O(20 x 20) / O(26 x 8) bins
    check_close(M, O.convolve_impact(S_ref, R, K), "impact K=10 configs[1]-sized M")


def test_impact_plan_with_noise_host_buffers_and_adc(B, O):
    """the accessories on an impact-position plan: fused noise (keyed by the wire, not the fine row), the host-buffer call
    and the ADC codes"""
    from paper_2203_02479_b200 import synth
    rng = np.random.default_rng(77)
    K, nw, nt = 3, 50, 640
    R = synth.response_impact(K, 7, 40)
    d = fine_depos(rng, 2500, nw, nt, K)
    host_M = torch.empty((nw, nt), dtype=torch.float32).pin_memory()
    host_adc = torch.empty((nw, nt), dtype=torch.int16).pin_memory()
    with B.ImpactPlan(nw, nt, R) as plan:
        plan.simulate_host({k: torch.from_numpy(v) for k, v in d.items()}, host_M, seed=5, fluctuate=True, noise=True, noise_seed=8)
        S_ref, _, _ = O.raster_scatter(nw * K, nt, d, seed=5, fluctuate=True)
        M_ref = O.convolve_impact(S_ref, R, K) + O.noise_add(np.zeros((nw, nt)), plan.pad_t, 8)
        check_close(host_M.numpy(), M_ref, "impact K=3 host call M + N")
        plan.simulate_host_adc_async({k: torch.from_numpy(v) for k, v in d.items()}, host_adc, 0.02, 500.0, 12, seed=5,
                                     fluctuate=True, noise=True, noise_seed=8)
        plan.sync()
        assert np.array_equal(host_adc.numpy(), O.digitize(plan.output().cpu().numpy(), 0.02, 500.0, 12))
        assert np.array_equal(plan.output().cpu().numpy(), host_M.numpy())  # the same plane-event twice: bitwise stable
