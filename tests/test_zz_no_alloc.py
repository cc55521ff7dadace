"""wcsim_raster_scatter_noalloc against the plan-based path it mirrors.

Some users of libwcsim cannot allocate device memory where they need the charge grid: a plug-in inside a framework that
owns the GPU's memory and forbids cudaMalloc while its event loop runs (an allocation can synchronise every stream of the
process), or an acquisition thread that may not block in the driver.  For them the library has one entry point that
takes the caller's own S and keeps the kernel's scratch (a 64-bit fixed-point grid) in a fixed 4 MiB array built into the
library.  That array is shared by every call and keeps the previous call's contents, so the thing to check is not only
that one call is right but that the NEXT one is too -- with a different grid shape, so that stale words of the first call
would land in the wrong bins if they were not cleared.

The reference here is the existing path: a plan in WCSIM_SCATTER_FIXED mode (itself checked against the oracle in
test_gpu_parity.py).  Both run the same order-independent integer accumulation, so equality is expected bit for bit; the
asserted bound is the one the parity tests use (rel-L2 <= 1e-5, max-abs <= 1e-4 max|S|; integer grids equal).

This file is named to be collected last: with `pytest -x`, a failure here must not hide the parity tests.  It passes
alone in a fresh process (the entry point's first call on the device does its own set-up) and after the other tests.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

REL_L2, MAX_ABS = 1e-5, 1e-4


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (run with -m gpu on the B200 box)")
    from paper_2203_02479_b200 import binding
    binding.lib()
    return binding


def _to_dev(depos):
    return {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in depos.items()}


def _plan_path(B, n_wires, n_ticks, dev, seed, id_base, fluctuate):
    """S of the existing path: a plan in fixed-point scatter mode (it allocates; that is the point of the other one)."""
    from paper_2203_02479_b200 import synth
    with B.Plan(n_wires, n_ticks, synth.response(3, 8), scatter_mode=B.WCSIM_SCATTER_FIXED) as p:
        p.raster_scatter(dev, seed=seed, depo_id_base=id_base, fluctuate=fluctuate)
        p.sync()
        return p.charge().cpu().numpy().astype(np.float64)


def _assert_same(got, ref, what, integer):
    got = got.astype(np.float64)
    scale = float(np.max(np.abs(ref)))
    assert scale > 0, what + ": empty reference"
    if integer:
        assert np.array_equal(got, ref), "%s: %d bins differ" % (what, int(np.count_nonzero(got != ref)))
    rel = float(np.linalg.norm(got - ref) / np.linalg.norm(ref))
    assert rel <= REL_L2, "%s: rel-L2 %.3e" % (what, rel)
    assert float(np.max(np.abs(got - ref))) <= MAX_ABS * scale, what


@pytest.mark.parametrize("fluctuate", [0, 1])
def test_two_calls_in_a_row_match_the_plan_path(B, fluctuate):
    from paper_2203_02479_b200 import synth
    # call 1: configs[0]'s grid and depo distribution; call 2: a wider, shorter grid with other depos, seed and ids
    d1 = synth.depos_uniform_box(400, gen_seed=11)
    d1["q"][::5] *= -1.0
    d2 = synth.depos_uniform_box(700, gen_seed=12)
    d2["x0"] = (d2["x0"] * 2.0).astype(np.float32)        # spread over 128 wires
    d2["t0"] = (d2["t0"] * 0.5).astype(np.float32)        # and 256 ticks
    cases = [(64, 512, d1, 5, 0), (128, 256, d2, 0xC0FFEE, (1 << 40) + 17)]
    stream = torch.cuda.current_stream()
    for call, (nw, nt, d, seed, id_base) in enumerate(cases, 1):
        dev = _to_dev(d)
        S = torch.zeros(nw * nt, dtype=torch.float32, device="cuda")
        B.wcsim_raster_scatter_noalloc(nw, nt, dev, S, seed=seed, depo_id_base=id_base, fluctuate=fluctuate, stream=stream)
        torch.cuda.synchronize()
        got = S.cpu().numpy().reshape(nw, nt)
        ref = _plan_path(B, nw, nt, dev, seed, id_base, fluctuate)
        _assert_same(got, ref, "call %d (%dx%d, fluctuate=%d)" % (call, nw, nt, fluctuate), integer=bool(fluctuate))


def test_accumulates_into_the_callers_grid_and_repeats_bit_for_bit(B):
    from paper_2203_02479_b200 import synth
    dev = _to_dev(synth.depos_uniform_box(300, gen_seed=13))
    S = torch.zeros(64 * 512, dtype=torch.float32, device="cuda")
    B.wcsim_raster_scatter_noalloc(64, 512, dev, S, seed=9, fluctuate=1)
    torch.cuda.synchronize()
    once = S.clone()
    B.wcsim_raster_scatter_noalloc(64, 512, dev, S, seed=9, fluctuate=1)  # same call again: S doubles exactly (integers)
    torch.cuda.synchronize()
    assert torch.equal(S, 2 * once)
    ref = _plan_path(B, 64, 512, dev, 9, 0, 1)
    assert np.array_equal(once.cpu().numpy().reshape(64, 512).astype(np.float64), ref)


def test_limit_and_argument_errors(B):
    from paper_2203_02479_b200 import synth
    dev = _to_dev(synth.depos_uniform_box(8, gen_seed=14))
    nw, nt = 64, B.WCSIM_NOALLOC_MAX_BINS // 64
    S = torch.zeros(nw * nt + nw, dtype=torch.float32, device="cuda")
    B.wcsim_raster_scatter_noalloc(nw, nt, dev, S, fluctuate=0)          # exactly the maximum: accepted
    torch.cuda.synchronize()
    assert float(S[: nw * nt].abs().sum()) > 0 and float(S[nw * nt:].abs().sum()) == 0
    with pytest.raises(B.WcsimError) as e:                                # one tick more: refused, and says why
        B.wcsim_raster_scatter_noalloc(nw, nt + 1, dev, S, fluctuate=0)
    assert e.value.status == B.WCSIM_ETOOBIG and "WCSIM_NOALLOC_MAX_BINS" in str(e.value)
    with pytest.raises(B.WcsimError) as e:
        B.wcsim_raster_scatter_noalloc(64, 512, dev, S, fluctuate=3)
    assert e.value.status == B.WCSIM_EINVAL
    B.wcsim_raster_scatter_noalloc(64, 512, dev, S, n=0)                  # nothing to do is not an error
