"""Pins for oracle/background.py (NEXT-4: FAR bookkeeping P:200/P:219, training-time whitening batch P:102)."""
import numpy as np

from oracle import background as obg
from oracle import psd as opsd
from oracle import whiten as owh
from synthdata.noise import coloured_noise


def test_far_counts_hand_example_strict_inequality():
    bg = np.array([1.0, 5.0, 3.0, 3.0, 9.0], dtype=np.float32)
    ev = np.array([0.0, 3.0, 9.0, 10.0, 4.0], dtype=np.float32)
    assert obg.far_counts(bg, ev).tolist() == [5, 2, 0, 0, 2]     # ties do not count ("greater than")
    np.testing.assert_array_equal(obg.far(bg, ev, 2.0), np.array([2.5, 1.0, 0.0, 0.0, 1.0]))


def test_far_counts_equal_sorted_search_library_routine():
    rng = np.random.default_rng(3)
    bg = rng.standard_normal(5000).astype(np.float32)
    bg[::7] = bg[3]                                                # repeated values
    ev = np.concatenate([rng.standard_normal(300).astype(np.float32), bg[:20]])
    ref = bg.size - np.searchsorted(np.sort(bg), ev, side="right")
    np.testing.assert_array_equal(obg.far_counts(bg, ev), ref)


def test_far_is_monotone_and_bounded():
    rng = np.random.default_rng(4)
    bg = rng.gumbel(size=2000).astype(np.float32)
    ev = np.sort(rng.gumbel(size=100).astype(np.float32))
    n = obg.far_counts(bg, ev)
    assert np.all(np.diff(n) <= 0) and n.max() <= bg.size and n.min() >= 0
    assert obg.far_counts(bg, np.array([np.inf, -np.inf], dtype=np.float32)).tolist() == [0, bg.size]
    assert obg.far_counts(np.zeros(0, np.float32), ev).tolist() == [0] * 100


def _batch(B=3, n=21504, seed=21):
    return np.stack([coloured_noise(n, seed + b).astype(np.float64) for b in range(B)])      # [B][2][n]


def test_training_batch_element_is_the_single_segment_path_and_shapes():
    x = _batch()
    y = obg.whiten_training_batch(x, 16384)
    assert y.shape == (3, 2, 3072)                                 # 10.5 s -> 8 s PSD + 2.5 s -> 1.5 s kernel
    # direct-sum FIR (O(N L), no FFT) with taps from scipy's Welch of the first 8 s: an independent route
    import scipy.signal
    _, p = scipy.signal.welch(x[1, 0, :16384], fs=2048.0, window="hann", nperseg=4096, noverlap=2048,
                              detrend="constant", average="mean")
    h = owh.design_filter(p)
    np.testing.assert_allclose(y[1, 0], owh.whiten_fir_direct(x[1, 0, 16384:], h), rtol=0, atol=1e-9 * np.abs(y).max())


def test_training_batch_uses_each_elements_own_psd():
    """Rescaling one (element, detector) leaves ITS whitened output unchanged (its PSD rescales with it) and no other
    output moves; a mix-up of PSDs between elements or detectors fails this."""
    x = _batch()
    y = obg.whiten_training_batch(x, 16384)
    x2 = x.copy()
    x2[2, 1] *= 8.0
    y2 = obg.whiten_training_batch(x2, 16384)
    np.testing.assert_allclose(y2, y, rtol=0, atol=1e-10 * np.abs(y).max())
    x3 = x[[2, 0, 1]]
    np.testing.assert_array_equal(obg.whiten_training_batch(x3, 16384), y[[2, 0, 1]])


def test_training_batch_output_is_roughly_white():
    """7-segment PSDs are noisy, so the whitened variance is only near 1: E[1/P_hat] exceeds 1/P by about k/(k-1) for an
    estimate with k effective averages (k ~ 5-7 here)."""
    x = _batch(B=8, seed=40)
    y = obg.whiten_training_batch(x, 16384)
    band_fraction = (1000.0 - 20.0) / 1024.0
    v = y.var() / band_fraction
    assert 1.0 < v < 1.5
