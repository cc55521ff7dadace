"""Pins of the oracle's ideal ADC (reading A23; M is "what is input to an analog-to-digital converter")."""
import numpy as np
import pytest

import oracle as O


def test_hand_worked_codes():
    # gain 2 codes per unit, baseline 100, 12 bits
    M = np.array([0.0, 0.24, 0.25, 0.26, 0.75, 1.25, -49.9, -50.0, -50.3, -1e9, 1997.4, 1997.6, 1e9, np.nan], dtype=np.float32)
    #             100  100.48 100.5 100.52 101.5 102.5  0.2    0.0    -0.6   clamp  4094.8  4095.2 clamp  nan
    want = [100, 100, 100, 101, 102, 102, 0, 0, 0, 0, 4095, 4095, 4095, 0]  # ties go to the even code
    assert O.digitize(M, 2.0, 100.0, 12).tolist() == want


def test_numpy_restatement_and_monotonicity():
    rng = np.random.default_rng(4)
    M = (rng.normal(0, 300, 200_000)).astype(np.float32)
    for bits, gain, base in ((12, 0.37, 900.0), (14, 4.0, 8000.0), (8, 0.01, 3.0)):
        adc = O.digitize(M, gain, base, bits)
        v = (M * np.float32(gain)).astype(np.float32) + np.float32(base)
        want = np.clip(np.rint(v.astype(np.float32)), 0, 2 ** bits - 1).astype(np.int16)
        assert np.array_equal(adc, want)
        order = np.argsort(M)
        assert np.all(np.diff(adc[order].astype(np.int32)) >= 0)  # gain > 0: monotone in M
        assert adc.min() >= 0 and adc.max() <= 2 ** bits - 1


def test_bad_arguments():
    with pytest.raises(ValueError):
        O.digitize(np.zeros(4, dtype=np.float32), 1.0, 0.0, 16)
    with pytest.raises(ValueError):
        O.digitize(np.zeros(4, dtype=np.float32), 1.0, 0.0, 0)
