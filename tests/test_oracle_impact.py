"""Pins of the oracle's sub-wire ("impact position") convolution, reading A25 of DESIGN.md (patches are
"typically O(20x20) elements"):
    M[x][t] = sum_k sum_dx sum_dt R[k][dx+c][dt] Sf[(x-dx) K + k][t-dt]
None of these re-types the C loop: K = 1 must be the already pinned Eq. (1) routine, a delta must read R_k back, the result
must be linear, a pure-python sum over the definition must agree on tiny grids, and the K sub-grids convolved one by one
with the pinned single-response routine must add up to it.  The raster on the K-times finer grid is the ordinary raster
(pinned in test_oracle_raster.py) on a grid of n_wires K rows with x in units of pitch / K; one test here checks that the
fine patch re-binned to whole wires is the coarse patch wherever both extents cover the wire."""
import numpy as np
import pytest

import oracle as O


@pytest.fixture(scope="module", autouse=True)
def _lib():
    O.lib()


def test_K1_is_the_plain_convolution():
    rng = np.random.default_rng(1)
    S = rng.normal(size=(9, 40))
    R = rng.normal(size=(5, 7))
    assert np.array_equal(O.convolve_impact(S, R[None], 1), O.convolve_direct(S, R))


@pytest.mark.parametrize("K", [2, 3, 10])
def test_delta_at_impact_position_k_reads_R_k_back(K):
    rng = np.random.default_rng(K)
    nw, nt, n_rw, n_rt = 12, 50, 5, 9
    c = (n_rw - 1) // 2
    R = rng.normal(size=(K, n_rw, n_rt))
    for k in range(K):
        xs, ts = 6, 11
        Sf = np.zeros((nw * K, nt))
        Sf[xs * K + k, ts] = 1.0
        M = O.convolve_impact(Sf, R, K)
        expect = np.zeros((nw, nt))
        # wire offsets dx = -c..c land on wires xs + dx; R_k[dx + c][dt] at tick ts + dt
        expect[xs - c:xs + c + 1, ts:ts + n_rt] = R[k]
        assert np.array_equal(M, expect), k
    # a delta near the wire and tick edges is cropped, not wrapped
    Sf = np.zeros((nw * K, nt))
    Sf[0 * K + (K - 1), nt - 2] = 2.0
    M = O.convolve_impact(Sf, R, K)
    expect = np.zeros((nw, nt))
    expect[0:c + 1, nt - 2:] = 2.0 * R[K - 1][c:, :2]
    assert np.array_equal(M, expect)


def test_linearity():
    rng = np.random.default_rng(5)
    K = 4
    S1, S2 = rng.normal(size=(2, 8 * K, 30))
    R = rng.normal(size=(K, 3, 6))
    M = O.convolve_impact(2.5 * S1 - 0.75 * S2, R, K)
    assert np.allclose(M, 2.5 * O.convolve_impact(S1, R, K) - 0.75 * O.convolve_impact(S2, R, K), rtol=0, atol=1e-12)


def test_python_brute_force_on_a_tiny_grid():
    rng = np.random.default_rng(7)
    K, nw, nt, n_rw, n_rt = 3, 5, 9, 3, 4
    c = 1
    Sf = rng.integers(-3, 4, size=(nw * K, nt)).astype(np.float64)
    R = rng.integers(-2, 3, size=(K, n_rw, n_rt)).astype(np.float64)  # small integers: every sum is exact in any order
    M = O.convolve_impact(Sf, R, K)
    for x in range(nw):
        for t in range(nt):
            acc = 0.0
            for k in range(K):
                for dx in range(-c, c + 1):
                    for dt in range(n_rt):
                        xs, ts = x - dx, t - dt
                        if 0 <= xs < nw and 0 <= ts < nt:
                            acc += R[k, dx + c, dt] * Sf[xs * K + k, ts]
            assert M[x, t] == acc, (x, t)


def test_sum_over_sub_grids_of_the_pinned_single_response_routine():
    rng = np.random.default_rng(9)
    K, nw, nt = 5, 20, 64
    Sf = rng.normal(size=(nw * K, nt)) * (rng.random((nw * K, nt)) < 0.2)
    R = rng.normal(size=(K, 7, 12))
    M = O.convolve_impact(Sf, R, K)
    parts = sum(O.convolve_direct(Sf[k::K], R[k]) for k in range(K))
    assert np.allclose(M, parts, rtol=0, atol=1e-12 * np.abs(M).max())
    # and the orientation: a response that differs between impact positions must not be applied to the wrong one
    R2 = R.copy()
    R2[[0, 1]] = R2[[1, 0]]
    assert not np.allclose(O.convolve_impact(Sf, R2, K), M)


def test_fine_patch_rebinned_to_wires_is_the_coarse_patch():
    """raster on the K-times finer wire grid (x and sigma_x in units of pitch / K) summed over the K impact positions of a
    wire equals the whole-wire raster's bin wherever both +-3 sigma extents cover that wire fully (the erf sum telescopes)"""
    K, nw, nt = 10, 30, 120
    f = np.float32
    x0, sx = 14.37, 0.8
    fine = {"t0": np.array([60.2], f), "x0": np.array([x0 * K], f), "sigma_t": np.array([1.5], f),
            "sigma_x": np.array([sx * K], f), "q": np.array([1.0e4], f)}
    coarse = dict(fine, x0=np.array([float(fine["x0"][0]) / K], np.float64).astype(f),
                  sigma_x=np.array([float(fine["sigma_x"][0]) / K], np.float64).astype(f))
    Sf, _, _ = O.raster_scatter(nw * K, nt, fine, fluctuate=False)
    Sc, _, _ = O.raster_scatter(nw, nt, coarse, fluctuate=False)
    rebinned = Sf.reshape(nw, K, nt).sum(axis=1)
    lo_f, hi_f = O.axis_extent(float(fine["x0"][0]), float(fine["sigma_x"][0]))
    full = [x for x in range(nw) if x * K >= lo_f and (x + 1) * K <= hi_f]  # wires all of whose fine bins are in the extent
    assert len(full) >= 3
    # fp32 inputs: x0 K / K is not x0 exactly, so compare at the level the input rounding allows
    assert np.allclose(rebinned[full], Sc[full], rtol=2e-5, atol=1e-9 * Sc.max())
    # the fine patch is typically O(20 x 20) bins: here 48 fine wires x 10 ticks
    assert (hi_f - lo_f) >= 4 * K
