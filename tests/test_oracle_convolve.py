"""Pins for the oracle's convolution (O5-O7 of SURVEY.md section 8c; north_star: "a delta-function input reproducing
R exactly", "linearity", "brute-force direct 2D convolution on tiny grids").  Eq. 1 / Eq. 2."""
import numpy as np
import pytest

import oracle
from paper_2203_02479_b200 import synth


def brute_conv(S, R):
    """M[x][t] = sum_dx sum_dt R[dx+c][dt] S[x-dx][t-dt], python loops straight from Eq. 1 (tiny grids only)."""
    nw, nt = S.shape
    nrw, nrt = R.shape
    c = (nrw - 1) // 2
    M = np.zeros_like(S, dtype=np.float64)
    for x in range(nw):
        for t in range(nt):
            acc = 0.0
            for dx in range(-c, c + 1):
                for dt in range(nrt):
                    xs, ts = x - dx, t - dt
                    if 0 <= xs < nw and 0 <= ts < nt:
                        acc += R[dx + c, dt] * S[xs, ts]
            M[x, t] = acc
    return M


def dft_naive(z, sign):
    n = len(z)
    k = np.arange(n)
    return np.exp(sign * 2j * np.pi * np.outer(k, k) / n) @ z


def test_fft_matches_naive_dft():
    rng = np.random.default_rng(0)
    for n in (1, 2, 4, 8, 64, 256):
        z = rng.standard_normal(n) + 1j * rng.standard_normal(n)
        for sign in (-1, +1):
            assert np.max(np.abs(oracle.fft(z, sign) - dft_naive(z, sign))) < 1e-11 * n
    # forward then inverse is n times the identity (unnormalised)
    z = rng.standard_normal(128) + 0j
    assert np.allclose(oracle.fft(oracle.fft(z, -1), +1), 128 * z, atol=1e-10)


def test_delta_reproduces_response_exactly():
    R = synth.response().astype(np.float64)            # 21 x 200
    nw, nt = 64, 512
    for (xs, ts) in [(30, 100), (0, 0), (63, 511), (5, 400), (60, 10)]:
        S = np.zeros((nw, nt))
        S[xs, ts] = 1.0
        M = oracle.convolve_direct(S, R)
        expect = np.zeros((nw, nt))
        for dx in range(-10, 11):
            x = xs + dx
            if 0 <= x < nw:
                n = min(200, nt - ts)
                expect[x, ts:ts + n] = R[dx + 10, :n]
        assert np.array_equal(M, expect)               # direct sum of one term: exact
        Mf = oracle.convolve_fft(S, R, 128, 1024)
        assert np.max(np.abs(Mf - expect)) <= 1e-13 * np.max(np.abs(R))


def test_response_orientation_is_not_transposed_or_flipped():
    # an asymmetric R on both axes: a flipped dx or dt index would fail here even where the delta test's R is symmetric in x
    R = np.zeros((3, 4))
    R[0, 1] = 2.0     # dx = -1, dt = 1
    R[2, 3] = -5.0    # dx = +1, dt = 3
    S = np.zeros((8, 16))
    S[4, 5] = 1.0
    M = oracle.convolve_direct(S, R)
    assert M[3, 6] == 2.0 and M[5, 8] == -5.0 and np.count_nonzero(M) == 2
    Mf = oracle.convolve_fft(S, R, 16, 32)
    assert np.allclose(Mf, M, atol=1e-14)
    assert oracle.convolve_points(S, R, [3, 5, 4], [6, 8, 5])[0] == 2.0


def test_linearity():
    rng = np.random.default_rng(1)
    R = synth.response(5, 12).astype(np.float64)
    S1, S2 = rng.standard_normal((12, 40)), rng.standard_normal((12, 40))
    a, b = 2.5, -0.75
    for conv in (oracle.convolve_direct, lambda s, r: oracle.convolve_fft(s, r, 16, 64)):
        lhs = conv(a * S1 + b * S2, R)
        rhs = a * conv(S1, R) + b * conv(S2, R)
        assert np.max(np.abs(lhs - rhs)) <= 1e-12 * np.max(np.abs(rhs))


@pytest.mark.parametrize("nw,nt,nrw,nrt,pw,pt", [(6, 20, 3, 5, 8, 32), (9, 17, 5, 8, 16, 32), (4, 8, 1, 1, 4, 8),
                                                 (16, 32, 7, 9, 32, 64)])
def test_direct_fft_brute_and_numpy_agree_on_tiny_grids(nw, nt, nrw, nrt, pw, pt):
    rng = np.random.default_rng(nw * 100 + nt)
    S = rng.standard_normal((nw, nt))
    S[rng.random((nw, nt)) < 0.5] = 0.0
    R = rng.standard_normal((nrw, nrt))
    ref = brute_conv(S, R)
    Md = oracle.convolve_direct(S, R)
    Mf = oracle.convolve_fft(S, R, pw, pt)
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(Md - ref)) <= 1e-13 * scale
    assert np.max(np.abs(Mf - ref)) <= 1e-12 * scale
    # third opinion: numpy's rfft2 on the same padded embedding
    c = (nrw - 1) // 2
    Sp = np.zeros((pw, pt)); Sp[:nw, :nt] = S
    Rp = np.zeros((pw, pt))
    for dx in range(-c, c + 1):
        Rp[dx % pw, :nrt] += R[dx + c]
    Mn = np.fft.irfft2(np.fft.rfft2(Sp) * np.fft.rfft2(Rp), s=(pw, pt))[:nw, :nt]
    assert np.max(np.abs(Mn - ref)) <= 1e-12 * scale
    # sampled points by the definition
    px = rng.integers(0, nw, 20); ptk = rng.integers(0, nt, 20)
    assert np.allclose(oracle.convolve_points(S, R, px, ptk), ref[px, ptk], rtol=0, atol=1e-13 * scale)


def test_padding_bounds_are_tight():
    # A13: exact iff pad_t >= n_t + n_rt - 1 and pad_w >= n_w + c; powers of two here, so choose sizes at the bound
    rng = np.random.default_rng(3)
    nrw, nrt = 5, 9          # c = 2
    R = rng.standard_normal((nrw, nrt))
    # tick axis: n_t + n_rt - 1 = 32 fits pad 32 exactly; n_t = 25 needs 33 > 32 -> wraps
    for nt, ok in ((24, True), (25, False)):
        S = rng.standard_normal((6, nt))
        err = np.max(np.abs(oracle.convolve_fft(S, R, 8, 32) - oracle.convolve_direct(S, R)))
        assert (err < 1e-12) == ok
    # wire axis: n_w + c = 8 fits pad 8; n_w = 7 needs 9 -> wraps
    for nw, ok in ((6, True), (7, False)):
        S = rng.standard_normal((nw, 16))
        err = np.max(np.abs(oracle.convolve_fft(S, R, 8, 32) - oracle.convolve_direct(S, R)))
        assert (err < 1e-12) == ok


def test_config0_direct_vs_fft_end_to_end():
    cfg = synth.config(0)
    pl = cfg["planes"][0]
    S, _, _ = oracle.raster_scatter(pl["n_wires"], pl["n_ticks"], pl["depos"])
    R = pl["response"].astype(np.float64)
    Md = oracle.convolve_direct(S, R)
    Mf = oracle.convolve_fft(S, R, pl["pad_w"], pl["pad_t"])
    assert np.linalg.norm(Md - Mf) <= 1e-12 * np.linalg.norm(Md)
    # the bipolar response integrates to ~0 along time per wire: sum_t R(x, t) is small against sum_t |R|
    assert abs(R.sum()) < 0.25 * np.abs(R).sum()
    # total of M = (sum S) (sum R) when nothing leaves the grid in wires... ticks are cropped, so only bound it
    assert np.isfinite(Md).all()
