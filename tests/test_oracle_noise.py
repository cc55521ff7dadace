"""Pins for the oracle's noise term N(t,x) (O11, O12 of SURVEY.md section 8c).  PAPER.md:40 names the term;
BASELINE.json configs[3] gives the model A(f) = 3 (f/f0) exp(-f/f0), f0 = 0.1 f_Nyquist, uniform random phases."""
import math

import numpy as np
import pytest

import oracle


def test_amplitude_spectrum_closed_form():
    for P in (64, 1024, 8192):
        amp = oracle.noise_amp(P)
        assert amp.shape == (P // 2 + 1,)
        assert amp[0] == 0.0
        k = np.arange(P // 2 + 1)
        r = (k / P) / 0.05                      # f / f0 with f0 = 0.1 * 0.5 cycles per tick
        assert np.allclose(amp, 3.0 * r * np.exp(-r), rtol=4e-16, atol=0)
        # maximum 3/e at f = f0, i.e. k = 0.05 P
        kmax = int(np.argmax(amp))
        assert abs(kmax - 0.05 * P) <= 1 and amp[kmax] == pytest.approx(3.0 / math.e, rel=3e-3)
        # Nyquist: f/f0 = 10
        assert amp[-1] == pytest.approx(30.0 * math.exp(-10.0), rel=1e-14)


def test_spectrum_has_the_amplitude_and_philox_phase():
    P, seed, wire = 256, 11, 7
    z = oracle.noise_spectrum(P, seed, wire)
    amp = oracle.noise_amp(P)
    assert np.allclose(np.abs(z), amp, rtol=1e-14, atol=1e-300)
    for k in (1, 2, 3, 4, 5, 77, 128):
        u = (oracle.noise_word(seed, wire, k) + 0.5) / 2.0**32
        assert z[k] == pytest.approx(amp[k] * complex(math.cos(2 * math.pi * u), math.sin(2 * math.pi * u)), abs=1e-15)
    # phases differ between wires and seeds
    assert not np.allclose(oracle.noise_spectrum(P, seed, wire + 1)[1:], z[1:])
    assert not np.allclose(oracle.noise_spectrum(P, seed + 1, wire)[1:], z[1:])


@pytest.mark.parametrize("P,expect", [(1024, 230.40), (8192, 1843.20), (16384, 3686.40)])
def test_parseval_closed_form(P, expect):
    # sum_t N^2 over the full padded window = 2 sum_{k=1}^{P/2-1} A_k^2 + (A_{P/2} cos phi)^2 (+ A_0^2 = 0),
    # independent of the phases; the value tends to P * 9 * 0.1 / 4 = 0.225 P
    amp = oracle.noise_amp(P)
    closed = 2.0 * np.sum(amp[1:P // 2] ** 2)
    assert closed == pytest.approx(expect, abs=0.02)
    assert closed / P == pytest.approx(0.225, abs=1e-4)
    M = np.zeros((3, P))
    oracle.noise_add(M, P, seed=5)
    for x in range(3):
        z = oracle.noise_spectrum(P, 5, x)
        assert np.sum(M[x] ** 2) == pytest.approx(closed + z[P // 2].real ** 2, rel=1e-12)
        assert abs(M[x].sum()) < 1e-9          # DC amplitude is zero
    # RMS 0.4743 ADC (reading A15)
    assert math.sqrt(np.mean(M ** 2)) == pytest.approx(0.4743, abs=2e-4)


def test_round_trip_recovers_the_spectrum():
    P = 512
    M = np.zeros((2, P))
    oracle.noise_add(M, P, seed=3)
    amp = oracle.noise_amp(P)
    for x in range(2):
        spec = np.fft.rfft(M[x]) / math.sqrt(P)      # independent library transform
        z = oracle.noise_spectrum(P, 3, x)
        assert np.allclose(spec[1:P // 2], z[1:P // 2], atol=1e-13)
        assert np.allclose(np.abs(spec[1:P // 2]), amp[1:P // 2], atol=1e-13)
        assert spec[P // 2].real == pytest.approx(z[P // 2].real, abs=1e-13)
        assert abs(spec[0]) < 1e-13


def test_definition_points_match_the_fft_route_and_crop():
    P, nt, nw = 256, 200, 5
    M = np.full((nw, nt), 1.5)
    oracle.noise_add(M, P, seed=9)
    rng = np.random.default_rng(0)
    wires = np.sort(rng.integers(0, nw, 40))
    ticks = rng.integers(0, nt, 40)
    pts = oracle.noise_points(P, 9, wires, ticks)
    assert np.allclose(M[wires, ticks] - 1.5, pts, atol=1e-13)
    # the cropped window is the head of the padded one
    Mfull = np.zeros((nw, P))
    oracle.noise_add(Mfull, P, seed=9)
    assert np.allclose(M - 1.5, Mfull[:, :nt], atol=1e-15)


def test_custom_amplitude_single_line():
    # one spectral line at k0 with amplitude a: N[t] = 2 a cos(2 pi k0 t / P + phi) / sqrt(P)
    P, k0, a = 128, 5, 2.0
    amp = np.zeros(P // 2 + 1)
    amp[k0] = a
    M = np.zeros((1, P))
    oracle.noise_add(M, P, seed=1, amp=amp)
    phi = 2 * math.pi * (oracle.noise_word(1, 0, k0) + 0.5) / 2.0**32
    t = np.arange(P)
    assert np.allclose(M[0], 2 * a * np.cos(2 * np.pi * k0 * t / P + phi) / math.sqrt(P), atol=1e-13)
