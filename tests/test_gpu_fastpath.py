"""The guarded fp32 fast path of the fluctuated raster (csrc/rng.cuh) against the fp64 routines it stands in for.

The raster decides a rounded-normal draw k = clamp(rint(mu + sd z), 0, N) (reading A6) from an fp32 estimate when
that estimate is farther from a rounding boundary than a bound on its own error, and otherwise falls back to the fp64
routine.  Two things make that exact: (1) the error of the fp32 normal quantile is measured here over ALL 2^32 words and must
stay below half the constant the guard assumes; (2) for every draw the guard accepts, k must equal the fp64 routine's."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

Z32_ERR_ASSUMED = 4.0e-6  # kZ32Err of csrc/rng.cuh


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (run with -m gpu on the B200 box)")
    from paper_2203_02479_b200 import binding
    binding.lib()
    return binding


def test_z32_error_over_all_words(B):
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    worst, zmax, accepted = 0.0, 0.0, 0
    for first in range(0, 1 << 32, 1 << 30):
        B.wcsim_debug_z32_scan(first, 1 << 30, out)
        torch.cuda.synchronize()
        raw = out.cpu().numpy()
        e_abs, z_max, e_rel = raw[0], raw[1], raw[3]
        n = int(raw[2:3].view(np.uint64)[0])
        worst, zmax, accepted = max(worst, e_abs), max(zmax, z_max), accepted + n
    print("z32: max |z32 - z64| = %.3e over %d accepted words (%.4f of all), max |z| = %.4f" % (
        worst, accepted, accepted / 2.0 ** 32, zmax))
    assert accepted > 0.99 * 2 ** 32          # only the far tails are left to the fp64 routine
    assert zmax < 2.94                        # the guard's error budget assumes |z| < 2.93 + rounding
    assert 2.0 * worst <= Z32_ERR_ASSUMED, worst


def test_fast_normal_agrees_wherever_it_accepts(B):
    rng = np.random.default_rng(17)
    n = 4_000_000
    # N and p spread over the raster's range (mu >= 16 is the binomial sampler's normal branch; smaller mu occurs with
    # the normal-approximation sampler of reading A21), plus adversarial cases: mu + sd z placed next to a half-integer
    N = np.floor(np.exp(rng.uniform(np.log(1.0), np.log(3e6), n)))
    p = np.exp(rng.uniform(np.log(1e-7), np.log(0.5), n))
    w = rng.integers(0, 2 ** 32, size=n, dtype=np.uint64).astype(np.uint32)
    from scipy.special import ndtri
    m = n // 4
    u = (w[:m].astype(np.float64) + 0.5) / 2.0 ** 32
    z = ndtri(u)
    mu_t = np.exp(rng.uniform(np.log(16.0), np.log(2e5), m))
    # choose p so that mu + sd z is (nearly) a half-integer: p = mu / N with mu solved for a target x
    x_t = np.floor(mu_t) + 0.5 + rng.normal(0.0, 1e-4, m)
    mu_s = mu_t.copy()
    for _ in range(30):  # fixed point of mu = x - sqrt(mu (1 - mu/N)) z
        mu_s = np.clip(x_t - np.sqrt(np.maximum(mu_s * (1 - mu_s / N[:m].clip(2 * mu_t)), 0)) * z, 1.0, None)
    N[:m] = np.floor(N[:m].clip(2 * mu_t) + 1)
    p[:m] = np.clip(mu_s / N[:m], 1e-9, 0.5)
    dN, dp = torch.from_numpy(N).cuda(), torch.from_numpy(p).cuda()
    dw = torch.from_numpy(w.view(np.int32)).cuda()
    k_fast = torch.zeros(n, dtype=torch.float64, device="cuda")
    ok = torch.zeros(n, dtype=torch.int32, device="cuda")
    k_ref = torch.zeros(n, dtype=torch.float64, device="cuda")
    B.wcsim_debug_fast_normal(dN, dp, dw, k_fast, ok, n)
    B.wcsim_debug_normal_draw(dN, dp, dw, k_ref, n)  # the fp64 rounded normal for every mu (reading A21)
    torch.cuda.synchronize()
    ok = ok.cpu().numpy().astype(bool)
    kf, kr = k_fast.cpu().numpy(), k_ref.cpu().numpy()
    bad = np.flatnonzero(ok & (kf != kr))
    print("fast normal: accepted %.4f of %d draws (adversarial quarter: %.4f), %d accepted draws differ" % (
        ok.mean(), n, ok[:m].mean(), bad.size))
    assert bad.size == 0, [(N[i], p[i], int(w[i]), kf[i], kr[i]) for i in bad[:5]]
    assert ok[m:].mean() > 0.95  # the fast path has to be the common case, or it is not a fast path
