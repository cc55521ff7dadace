"""GPU parity of the batched-planes path (Section 3.3): a multi-plane plan runs the
planes of one event through ONE launch sequence -- one raster launch with the depos of all planes, row transforms over all
stacked rows, one direct wire pass with every plane's own response -- optionally replayed from a CUDA graph.  The oracle
side is a loop over the planes: every plane's S and M must equal what that plane alone gives (north_star tolerances)."""
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


def check_close(got, ref, what):
    got = np.asarray(got, dtype=np.float64)
    r, m, scale = rel_l2(got, ref), float(np.max(np.abs(got - ref))), float(np.max(np.abs(ref)))
    record(what, rel_l2=r, max_abs_over_scale=m / max(scale, 1e-300), outputs=int(got.size))
    assert r <= REL_L2, "%s: rel-L2 %.3e" % (what, r)
    assert m <= MAX_ABS * scale, "%s: max-abs %.3e vs scale %.3e" % (what, m, scale)


def small_event(rng):
    """three planes of different widths, own responses, depos that leave the grid, invalid depos, an empty-ish plane"""
    from paper_2203_02479_b200 import synth
    n_ticks = 700
    planes = []
    for p, (nw, n) in enumerate(((40, 3000), (33, 17), (70, 5000))):
        R = (synth.response(5, 30) * (1.0 + 0.5 * p)).astype(np.float32)
        if p == 1:
            R = R[::-1].copy()  # not symmetric in wires: catches a response applied to the wrong plane or flipped
            R[0] *= 3.0
        d = {"t0": rng.uniform(-5, n_ticks + 5, n), "x0": rng.uniform(-2, nw + 2, n), "sigma_t": rng.uniform(0, 2.5, n),
             "sigma_x": rng.uniform(0, 1.2, n), "q": rng.lognormal(np.log(5000), 0.5, n)}
        d = {k: v.astype(np.float32) for k, v in d.items()}
        d["q"][::7] *= -1
        d["t0"][3] = np.nan
        d["sigma_x"][5] = -1.0
        planes.append(dict(n_wires=nw, n_ticks=n_ticks, response=R, depos=d))
    return planes


@pytest.mark.parametrize("mode", [0, 2])
@pytest.mark.parametrize("fluct", [0, 1, 2])
def test_planes_plan_equals_planes_one_by_one(B, O, mode, fluct):
    rng = np.random.default_rng(17)
    planes = small_event(rng)
    nt = planes[0]["n_ticks"]
    with B.PlanesPlan([pl["n_wires"] for pl in planes], nt, [pl["response"] for pl in planes], scatter_mode=mode) as plan:
        assert [plan.plane_rows(p) for p in range(3)] == [(0, 40), (40, 33), (73, 70)]
        dev = [to_dev(pl["depos"]) for pl in planes]
        plan.clear()
        plan.reset_stats()
        plan.raster_scatter_planes(dev, seed=5, fluctuate=fluct)
        plan.arm_noise(None, seed=9)
        plan.convolve()
        plan.sync()
        S = plan.charge().cpu().numpy().astype(np.float64)
        M = plan.output().cpu().numpy().astype(np.float64)
        st = plan.stats()
        pad_t = plan.pad_t
        drawn = skipped = 0
        for p, pl in enumerate(planes):
            r0, nw = plan.plane_rows(p)
            S_ref, _, ost = O.raster_scatter(nw, nt, pl["depos"], seed=5, fluctuate=fluct)
            drawn += ost["drawn"]
            skipped += ost["skipped"]
            if fluct:
                flipped = int(np.count_nonzero(S[r0:r0 + nw] != S_ref))
                assert flipped <= FLIP_BUDGET * ost["drawn"], (p, flipped)
            else:
                check_close(S[r0:r0 + nw], S_ref, "planes plan S, plane %d mode %d" % (p, mode))
            M_ref = O.convolve_direct(S_ref, pl["response"]) + O.noise_add(np.zeros((nw, nt)), pad_t, 9)
            check_close(M[r0:r0 + nw], M_ref, "planes plan M + N, plane %d mode %d fluct %d" % (p, mode, fluct))
        assert st["bins_drawn"] == drawn and st["depos_skipped"] == skipped == 6
        # the single-plane calls are not valid on a multi-plane plan
        with pytest.raises(B.WcsimError):
            plan.raster_scatter(dev[0], seed=5, fluctuate=fluct)
        # an empty event: nothing happens
        plan.raster_scatter_planes(dev, n=[0, 0, 0], seed=5, fluctuate=fluct)
    with pytest.raises(B.WcsimError):
        B.PlanesPlan([40, 33], nt, [planes[0]["response"]] * 2, scatter_mode=B.WCSIM_SCATTER_TILED)


def test_config_3_event_through_one_launch_sequence(B, O):
    """configs[3] at full size: the three planes (800, 800, 960 wires x 6000 ticks, 200k depos each, own responses, noise)
    through a multi-plane plan, every plane against the oracle over the whole plane"""
    from paper_2203_02479_b200 import synth
    cfg = synth.config(3)
    planes = cfg["planes"]
    nt = planes[0]["n_ticks"]
    with B.PlanesPlan([pl["n_wires"] for pl in planes], nt, [pl["response"] for pl in planes],
                      pad_ticks=planes[0]["pad_t"], nsigma=cfg["nsigma"]) as plan:
        dev = [to_dev(pl["depos"]) for pl in planes]
        plan.clear()
        fluct_seeds, noise_seeds = [pl["fluct_seed"] for pl in planes], [pl["noise_seed"] for pl in planes]
        assert len(set(noise_seeds)) == 3 and len(set(fluct_seeds)) == 3  # reading A26: a seed per plane
        plan.raster_scatter_planes(dev, seeds=fluct_seeds, fluctuate=True)
        plan.arm_noise_planes(None, seeds=noise_seeds)
        plan.convolve()
        plan.sync()
        S = plan.charge().cpu().numpy()
        M = plan.output().cpu().numpy()
        assert plan.launch_count() == 5  # clear, raster, forward rows, wire pass, inverse rows: one launch each for three planes
        for p, pl in enumerate(planes):
            r0, nw = plan.plane_rows(p)
            S_ref, _, st = O.raster_scatter(nw, nt, pl["depos"], seed=pl["fluct_seed"], fluctuate=True, nsigma=cfg["nsigma"])
            flipped = int(np.count_nonzero(S[r0:r0 + nw].astype(np.float64) != S_ref))
            record("configs[3] batched plane %d S" % p, flipped_bins=flipped, drawn_bins=int(st["drawn"]))
            assert flipped <= FLIP_BUDGET * st["drawn"]
            M_ref = O.convolve_fft(S_ref, pl["response"], pl["pad_w"], pl["pad_t"])
            M_ref += O.noise_add(np.zeros((nw, nt)), pl["pad_t"], pl["noise_seed"])
            check_close(M[r0:r0 + nw], M_ref, "configs[3] batched plane %d M + N" % p)
        # noise alone through the same plan (S = 0 => M = N): plane p equals a single-plane run with plane p's seed, and
        # wire 5 of plane 0 and wire 5 of plane 1 carry different waveforms
        plan.clear()
        plan.arm_noise_planes(None, seeds=noise_seeds)
        plan.convolve()
        plan.sync()
        N = plan.output().cpu().numpy().astype(np.float64)
        rows = [plan.plane_rows(p) for p in range(3)]
        for p, pl in enumerate(planes):
            r0, nw = rows[p]
            check_close(N[r0:r0 + nw], O.noise_add(np.zeros((nw, nt)), pl["pad_t"], pl["noise_seed"]),
                        "configs[3] batched plane %d noise alone" % p)
        assert not np.allclose(N[rows[0][0] + 5], N[rows[1][0] + 5], atol=1e-3)
        # one seed for all planes (wcsim_arm_noise on a multi-plane plan) still means what it says: identical waveforms
        plan.clear()
        plan.arm_noise(None, seed=noise_seeds[1])
        plan.convolve()
        plan.sync()
        N1 = plan.output().cpu().numpy().astype(np.float64)
        assert np.array_equal(N1[rows[0][0] + 5], N1[rows[1][0] + 5])
        assert np.array_equal(N1[rows[1][0]:rows[1][0] + rows[1][1]], N[rows[1][0]:rows[1][0] + rows[1][1]])
        # the stand-alone pass takes per-plane seeds too: M += N on top of the armed result gives 2 N for plane 1
        plan.add_noise_planes(None, seeds=noise_seeds)
        plan.sync()
        N2 = plan.output().cpu().numpy().astype(np.float64)
        r0, nw = rows[1]
        check_close(N2[r0:r0 + nw], 2.0 * N[r0:r0 + nw], "configs[3] batched add_noise_planes")


def test_graph_replays_a_plane_event(B, O):
    """clear + raster + arm_noise + convolve + digitize captured once and replayed: same results as the direct calls, and
    new depo values in the same device arrays give the new event's results"""
    from paper_2203_02479_b200 import synth
    cfg = synth.config(0)
    pl = cfg["planes"][0]
    nw, nt, R = pl["n_wires"], pl["n_ticks"], pl["response"]
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        dev = to_dev(pl["depos"])
        adc = torch.zeros((nw, nt), dtype=torch.int16, device="cuda")
    stream.synchronize()
    plan = B.Plan(nw, nt, R, pad=(pl["pad_w"], pl["pad_t"]), stream=stream)
    try:
        def sequence():
            plan.clear()
            plan.raster_scatter(dev, seed=3, fluctuate=True)
            plan.arm_noise(None, seed=4)
            plan.convolve()
            plan.digitize(0.01, 900.0, 12, out=adc)

        sequence()
        plan.sync()
        M_direct = plan.output().cpu().numpy().copy()
        adc_direct = adc.cpu().numpy().copy()
        launches0 = plan.launch_count()
        plan.graph_begin()
        sequence()
        graph = plan.graph_end()
        assert plan.launch_count() == launches0  # recording runs nothing
        plan.clear_output()
        adc.zero_()
        graph.launch()
        graph.launch()
        plan.sync()
        assert plan.launch_count() == launches0 + 2 * 6  # clear, raster, three convolution kernels, digitize
        assert np.array_equal(plan.output().cpu().numpy(), M_direct)
        assert np.array_equal(adc.cpu().numpy(), adc_direct)
        # a new event in the same arrays
        d2 = {k: v.copy() for k, v in pl["depos"].items()}
        d2["t0"] = (d2["t0"] * 0.5 + 100).astype(np.float32)
        d2["q"] = (d2["q"] * 1.7).astype(np.float32)
        with torch.cuda.stream(stream):
            for k in dev:
                dev[k].copy_(torch.from_numpy(d2[k]))
        graph.launch()
        plan.sync()
        S_ref, _, st = O.raster_scatter(nw, nt, d2, seed=3, fluctuate=True)
        assert int(np.count_nonzero(plan.charge().cpu().numpy().astype(np.float64) != S_ref)) <= FLIP_BUDGET * st["drawn"]
        M_ref = O.convolve_direct(S_ref, R) + O.noise_add(np.zeros((nw, nt)), pl["pad_t"], 4)
        check_close(plan.output().cpu().numpy(), M_ref, "graph replay M + N")
        assert np.array_equal(adc.cpu().numpy(), O.digitize(plan.output().cpu().numpy(), 0.01, 900.0, 12))
        # what cannot be captured says so instead of breaking the capture: the tiled mode's first call allocates its lists
        plan.graph_begin()
        plan.set_scatter_mode(B.WCSIM_SCATTER_TILED)
        with pytest.raises(B.WcsimError):
            plan.raster_scatter(dev, seed=3, fluctuate=True)
        plan.set_scatter_mode(B.WCSIM_SCATTER_ATOMIC)
        with pytest.raises(B.WcsimError):
            plan.arm_noise(np.ones(pl["pad_t"] // 2 + 1, dtype=np.float32), seed=1)
        g2 = plan.graph_end()
        g2.destroy()
        graph.destroy()
        # once its lists exist the tiled (sort-by-tile) mode is stream-ordered like the others and can be captured
        plan.set_scatter_mode(B.WCSIM_SCATTER_TILED)
        plan.clear()
        plan.raster_scatter(dev, seed=3, fluctuate=True)
        plan.sync()
        S_tiled = plan.charge().cpu().numpy().copy()
        assert np.array_equal(S_tiled.astype(np.float64), S_ref)
        plan.graph_begin()
        plan.clear()
        plan.raster_scatter(dev, seed=3, fluctuate=True)
        g3 = plan.graph_end()
        plan.clear()
        g3.launch()
        plan.sync()
        assert np.array_equal(plan.charge().cpu().numpy(), S_tiled)
        g3.destroy()
    finally:
        plan.destroy()
    # the legacy default stream cannot be captured
    with B.Plan(nw, nt, R, stream=0) as p0:
        with pytest.raises(B.WcsimError):
            p0.graph_begin()


def test_graph_update_gives_each_event_its_own_seeds(B, O):
    """A plain replay repeats the recorded seeds, depo count and id base (they are kernel arguments frozen in the graph), so
    consecutive events would share one Philox stream and one noise realisation.  wcsim_graph_update re-records the sequence
    with the new event's values into the existing executable graph; each replay then equals the oracle with ITS seeds."""
    from paper_2203_02479_b200 import synth
    cfg = synth.config(0)
    pl = cfg["planes"][0]
    nw, nt, R = pl["n_wires"], pl["n_ticks"], pl["response"]
    events = [dict(depos=synth.depos_uniform_box(100, gen_seed=21), n=100, seed=3, noise_seed=4, id_base=0),
              dict(depos=synth.depos_uniform_box(100, gen_seed=22), n=100, seed=0xABCDEF0123, noise_seed=99, id_base=1 << 33),
              dict(depos=synth.depos_uniform_box(100, gen_seed=23), n=61, seed=5, noise_seed=6, id_base=7)]  # fewer depos too
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        dev = to_dev(events[0]["depos"])
    stream.synchronize()
    plan = B.Plan(nw, nt, R, pad=(pl["pad_w"], pl["pad_t"]), stream=stream)
    try:
        def sequence(ev):
            plan.clear()
            plan.raster_scatter(dev, n=ev["n"], seed=ev["seed"], depo_id_base=ev["id_base"], fluctuate=True)
            plan.arm_noise(None, seed=ev["noise_seed"])
            plan.convolve()

        graph = None
        noise_of_wire5 = []
        for ev in events:
            with torch.cuda.stream(stream):
                for k in dev:
                    dev[k].copy_(torch.from_numpy(ev["depos"][k]))
            plan.graph_begin()
            sequence(ev)
            if graph is None:
                graph = plan.graph_end()
            else:
                graph.update()
            plan.clear_output()
            graph.launch()
            plan.sync()
            d = {k: v[: ev["n"]] for k, v in ev["depos"].items()}
            S_ref, _, st = O.raster_scatter(nw, nt, d, seed=ev["seed"], id_base=ev["id_base"], fluctuate=True)
            S = plan.charge().cpu().numpy().astype(np.float64)
            assert int(np.count_nonzero(S != S_ref)) <= FLIP_BUDGET * st["drawn"]
            N_ref = O.noise_add(np.zeros((nw, nt)), pl["pad_t"], ev["noise_seed"])
            check_close(plan.output().cpu().numpy(), O.convolve_direct(S_ref, R) + N_ref, "graph update M + N")
            noise_of_wire5.append(N_ref[5].copy())
        assert not np.allclose(noise_of_wire5[0], noise_of_wire5[1])
        # without the update the old values come back: a replay over event 0's depos still uses event 2's seed, count and ids
        with torch.cuda.stream(stream):
            for k in dev:
                dev[k].copy_(torch.from_numpy(events[0]["depos"][k]))
        graph.launch()
        plan.sync()
        ev = events[2]
        d = {k: v[: ev["n"]] for k, v in events[0]["depos"].items()}
        S_ref, _, st = O.raster_scatter(nw, nt, d, seed=ev["seed"], id_base=ev["id_base"], fluctuate=True)
        assert int(np.count_nonzero(plan.charge().cpu().numpy().astype(np.float64) != S_ref)) <= FLIP_BUDGET * st["drawn"]
        # a different sequence is refused and the capture is closed; a plan with a live graph is not freed from under it
        plan.graph_begin()
        plan.clear()
        with pytest.raises(B.WcsimError) as e:
            graph.update()
        assert e.value.status == B.WCSIM_ESTATE
        assert B.lib().wcsim_plan_destroy(plan.handle) == B.WCSIM_ESTATE
        graph.destroy()
    finally:
        plan.destroy()


def test_planes_plan_graph(B, O):
    rng = np.random.default_rng(3)
    planes = small_event(rng)
    nt = planes[0]["n_ticks"]
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        dev = [to_dev(pl["depos"]) for pl in planes]
    stream.synchronize()
    with B.PlanesPlan([pl["n_wires"] for pl in planes], nt, [pl["response"] for pl in planes], stream=stream) as plan:
        plan.graph_begin()
        plan.clear()
        plan.raster_scatter_planes(dev, seed=11, fluctuate=True)
        plan.convolve()
        graph = plan.graph_end()
        graph.launch()
        plan.sync()
        S = plan.charge().cpu().numpy().astype(np.float64)
        M = plan.output().cpu().numpy()
        for p, pl in enumerate(planes):
            r0, nw = plan.plane_rows(p)
            S_ref, _, st = O.raster_scatter(nw, nt, pl["depos"], seed=11, fluctuate=True)
            assert int(np.count_nonzero(S[r0:r0 + nw] != S_ref)) <= FLIP_BUDGET * st["drawn"]
            check_close(M[r0:r0 + nw], O.convolve_direct(S_ref, pl["response"]), "planes graph M, plane %d" % p)
        graph.destroy()


def test_simulate_host_adc_async_and_contiguous_depos(B, O):
    """the end-to-end call returning ADC codes (reading A23) equals digitising the oracle-checked M; the five host depo
    arrays of one pinned block go over in one copy and give the same result as five separate arrays"""
    from paper_2203_02479_b200 import synth
    cfg = synth.config(1, n_depos=5000)
    pl = cfg["planes"][0]
    nw, nt, R = pl["n_wires"], pl["n_ticks"], pl["response"]
    n = 5000
    block = torch.empty(5 * n, dtype=torch.float32).pin_memory()
    host = {}
    for a, k in enumerate(("t0", "x0", "sigma_t", "sigma_x", "q")):
        host[k] = block[a * n:(a + 1) * n]
        host[k].copy_(torch.from_numpy(pl["depos"][k]))
    host_adc = torch.empty((nw, nt), dtype=torch.int16).pin_memory()
    host_M = torch.empty((nw, nt), dtype=torch.float32).pin_memory()
    with B.Plan(nw, nt, R, pad=(pl["pad_w"], pl["pad_t"])) as plan:
        plan.simulate_host_adc_async(host, host_adc, 0.01, 900.0, 12, seed=2, fluctuate=True, noise=True, noise_seed=6)
        plan.sync()
        M = plan.output().cpu().numpy()
        assert np.array_equal(host_adc.numpy(), O.digitize(M, 0.01, 900.0, 12))
        S_ref, _, _ = O.raster_scatter(nw, nt, pl["depos"], seed=2, fluctuate=True)
        M_ref = O.convolve_fft(S_ref, R, pl["pad_w"], pl["pad_t"]) + O.noise_add(np.zeros((nw, nt)), pl["pad_t"], 6)
        check_close(M, M_ref, "simulate_host_adc M + N")
        sep = {k: torch.from_numpy(pl["depos"][k].copy()) for k in host}  # five separate (pageable) arrays
        plan.simulate_host(sep, host_M, seed=2, fluctuate=True, noise=True, noise_seed=6)
        assert np.array_equal(host_M.numpy(), M)
        with pytest.raises(ValueError):
            plan.simulate_host(sep, torch.empty(10, dtype=torch.float32), seed=2)
        with pytest.raises(ValueError):
            plan.simulate_host_adc_async(sep, torch.empty((nw, nt), dtype=torch.float32), 0.01, 900.0)


def test_armed_custom_spectrum_survives_a_later_add_noise(B, O):
    from paper_2203_02479_b200 import synth
    R = synth.response(5, 30)
    nw, nt = 24, 500
    with B.Plan(nw, nt, R) as p:
        P = p.pad_t
        amp1 = np.linspace(1.0, 0.0, P // 2 + 1).astype(np.float32)
        amp2 = np.full(P // 2 + 1, 0.25, dtype=np.float32)
        p.arm_noise(amp1, seed=5)
        p.clear_output()
        p.add_noise(amp=amp2, seed=7)   # uploads another custom spectrum while amp1 is armed
        p.sync()
        N2 = p.output().cpu().numpy()
        p.clear()
        p.convolve()                    # S = 0: M = the armed noise, which must still be amp1's
        p.sync()
        N1 = p.output().cpu().numpy()
    check_close(N2, O.noise_add(np.zeros((nw, nt)), P, seed=7, amp=amp2.astype(np.float64)), "add_noise amp2")
    check_close(N1, O.noise_add(np.zeros((nw, nt)), P, seed=5, amp=amp1.astype(np.float64)), "armed amp1 after add_noise amp2")


def test_planes_api_limits_and_single_plane(B, O):
    """wcsim_raster_scatter_planes on an ordinary (one-plane) plan equals wcsim_raster_scatter bit for bit; 8 planes are the
    limit, 9 and 0 are refused; a plane may have no depos at all"""
    from paper_2203_02479_b200 import synth
    cfg = synth.config(1, n_depos=3000)
    pl = cfg["planes"][0]
    nw, nt, R = 120, 900, synth.response(5, 24)
    d = {k: v.copy() for k, v in pl["depos"].items()}
    d["x0"] = (d["x0"] * (nw / 800.0)).astype(np.float32)
    d["t0"] = (d["t0"] * (nt / 6000.0)).astype(np.float32)
    dev = to_dev(d)
    with B.Plan(nw, nt, R) as p:
        p.clear()
        p.raster_scatter(dev, seed=3, fluctuate=True)
        p.sync()
        S1 = p.charge().cpu().numpy().copy()
        p.clear()
        p.raster_scatter_planes([dev], seed=3, fluctuate=True)
        p.sync()
        assert np.array_equal(p.charge().cpu().numpy(), S1)
    S_ref, _, st = O.raster_scatter(nw, nt, d, seed=3, fluctuate=True)
    assert int(np.count_nonzero(S1.astype(np.float64) != S_ref)) <= FLIP_BUDGET * st["drawn"]
    with B.PlanesPlan([nw] * 8, nt, [R] * 8) as p8:
        empty = {k: torch.empty(0, dtype=torch.float32, device="cuda") for k in dev}
        p8.clear()
        p8.raster_scatter_planes([dev, empty, dev, empty, empty, empty, empty, dev], seed=3, fluctuate=True)
        p8.convolve()
        p8.sync()
        S8 = p8.charge().cpu().numpy()
        M8 = p8.output().cpu().numpy()
        M_ref = O.convolve_direct(S_ref, R)
        for q in range(8):
            r0, n = p8.plane_rows(q)
            assert (r0, n) == (q * nw, nw)
            if q in (0, 2, 7):
                assert np.array_equal(S8[r0:r0 + n], S1)
                check_close(M8[r0:r0 + n], M_ref, "8-plane plan, plane %d" % q)
            else:
                assert not S8[r0:r0 + n].any() and not M8[r0:r0 + n].any()  # an empty plane stays empty: no leak across the halos
    for bad in (0, 9):
        with pytest.raises((B.WcsimError, ValueError)):
            B.PlanesPlan([nw] * bad, nt, [R] * bad)
