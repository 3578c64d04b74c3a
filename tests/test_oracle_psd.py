"""Pins for oracle/psd.py (O-1, reading A1/A2)."""
import numpy as np
import pytest
import scipy.signal

from oracle import psd as opsd

RNG = np.random.default_rng(11)
FS = 2048.0


def test_welch_equals_scipy_library_routine():
    x = RNG.standard_normal(16 * 2048) * 3e-3 + 0.7   # non-zero mean exercises the detrend
    p = opsd.welch(x, FS, 4096, 2048)
    f, ref = scipy.signal.welch(x, fs=FS, window="hann", nperseg=4096, noverlap=2048,
                                detrend="constant", scaling="density", average="mean")
    assert p.shape == (2049,)
    np.testing.assert_allclose(p, ref, rtol=1e-10, atol=1e-22)


def test_welch_physical_units_equal_scipy():
    x = RNG.standard_normal(8 * 2048) * 7e-22
    p = opsd.welch(x, FS, 4096, 2048)
    _, ref = scipy.signal.welch(x, fs=FS, window="hann", nperseg=4096, noverlap=2048,
                                detrend="constant", scaling="density", average="mean")
    np.testing.assert_allclose(p, ref, rtol=1e-10)


def test_segment_count_closed_form():
    assert opsd.segment_count(64 * 2048, 4096, 2048) == 63    # 64 s
    assert opsd.segment_count(8 * 2048, 4096, 2048) == 7      # 8 s
    assert opsd.segment_count(4095, 4096, 2048) == 0


def test_sinusoid_peak_bin_and_power():
    amp, f0 = 2.5, 100.0                      # on a bin: df = 0.5 Hz -> k0 = 200
    t = np.arange(32 * 2048) / FS
    p = opsd.welch(amp * np.sin(2 * np.pi * f0 * t), FS, 4096, 2048)
    assert np.argmax(p) == 200
    np.testing.assert_allclose(np.sum(p) * 0.5, amp ** 2 / 2, rtol=1e-9)


def test_parseval_single_rectangular_segment():
    x = RNG.standard_normal(4096)
    x -= x.mean()
    p = opsd.periodogram(x, FS, np.ones(4096))
    np.testing.assert_allclose(np.sum(p) * (FS / 4096), np.mean(x ** 2), rtol=1e-12)


def test_white_noise_level():
    sigma = 3.0
    x = RNG.standard_normal(256 * 2048) * sigma
    p = opsd.welch(x, FS, 4096, 2048)
    np.testing.assert_allclose(p[10:-10].mean(), 2 * sigma ** 2 / FS, rtol=0.02)


def test_hann_is_periodic():
    w = opsd.hann_periodic(4096)
    np.testing.assert_allclose(w, scipy.signal.get_window("hann", 4096, fftbins=True), atol=1e-15)
    assert w[0] == 0.0 and w[2048] == 1.0


# ---- NEXT-3 variant: median-averaged Welch ----------------------------------------------------------------------
def test_median_bias_closed_forms_and_limit():
    assert opsd.median_bias(1) == 1.0
    assert abs(opsd.median_bias(3) - (1.0 - 0.5 + 1.0 / 3.0)) < 1e-15
    assert opsd.median_bias(4) == opsd.median_bias(3)          # even n: the two middle values are averaged
    assert abs(opsd.median_bias(200001) - np.log(2.0)) < 1e-5  # alternating harmonic series -> ln 2


def test_median_bias_is_the_expected_median_of_exponentials():
    """Definition check by Monte Carlo: E[median of n unit exponentials] = median_bias(n)."""
    rng = np.random.default_rng(5)
    for n in (7, 63):
        med = np.median(rng.exponential(1.0, size=(200_000, n)), axis=1)
        se = med.std() / np.sqrt(med.size)
        assert abs(med.mean() - opsd.median_bias(n)) < 5 * se


@pytest.mark.parametrize("seconds", [8, 9, 64])                # 7 (odd), 8 (even), 63 segments
def test_median_welch_equals_scipy_library_routine(seconds):
    x = RNG.standard_normal(seconds * 2048) * 3e-3 + 0.2
    p = opsd.welch(x, FS, 4096, 2048, average="median")
    _, ref = scipy.signal.welch(x, fs=FS, window="hann", nperseg=4096, noverlap=2048,
                                detrend="constant", scaling="density", average="median")
    np.testing.assert_allclose(p, ref, rtol=1e-10, atol=1e-22)


def test_median_welch_ignores_a_glitch_that_the_mean_does_not():
    x = RNG.standard_normal(64 * 2048)
    clean_med = opsd.welch(x, FS, 4096, 2048, average="median")
    clean_mean = opsd.welch(x, FS, 4096, 2048)
    x[70000] += 500.0                                         # one loud spike (flat spectrum): it lands in two segments of 63
    med = opsd.welch(x, FS, 4096, 2048, average="median")
    mean = opsd.welch(x, FS, 4096, 2048)
    band = slice(40, 2000)
    assert np.median(mean[band] / clean_mean[band]) > 3.0
    assert abs(np.median(med[band] / clean_med[band]) - 1.0) < 0.1
