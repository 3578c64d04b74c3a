"""Pins for oracle/fft.py: closed forms and library routines (none re-types the oracle's formula)."""
import numpy as np
import pytest

from oracle import fft as offt

RNG = np.random.default_rng(7)


def test_dft_naive_delta_closed_form():
    n, n0 = 64, 5
    x = np.zeros(n); x[n0] = 1.0
    k = np.arange(n)
    np.testing.assert_allclose(offt.dft_naive(x), np.exp(-2j * np.pi * k * n0 / n), atol=1e-13)


def test_dft_naive_sinusoid_lands_in_its_bin():
    n, k0, amp = 256, 19, 3.0
    x = amp * np.cos(2 * np.pi * k0 * np.arange(n) / n + 0.3)
    mag = np.abs(offt.dft_naive(x))
    assert np.argmax(mag[: n // 2]) == k0
    np.testing.assert_allclose(mag[k0], amp * n / 2, rtol=1e-12)
    mask = np.ones(n, bool); mask[[k0, n - k0]] = False
    assert mag[mask].max() < 1e-10


def test_dft_naive_sign_convention_shift_theorem():
    # x[n-1] <-> X[k] exp(-2 pi i k / N): fails for a +i kernel
    n = 32
    x = RNG.standard_normal(n)
    lhs = offt.dft_naive(np.roll(x, 1))
    rhs = offt.dft_naive(x) * np.exp(-2j * np.pi * np.arange(n) / n)
    np.testing.assert_allclose(lhs, rhs, atol=1e-12)


@pytest.mark.parametrize("n", [2, 8, 64, 1024])
def test_fft_radix2_equals_naive_dft(n):
    x = RNG.standard_normal(n) + 1j * RNG.standard_normal(n)
    np.testing.assert_allclose(offt.fft_radix2(x), offt.dft_naive(x), atol=1e-9 * n)
    np.testing.assert_allclose(offt.fft_radix2(x, inverse=True), offt.dft_naive(x, inverse=True), atol=1e-12)


@pytest.mark.parametrize("n", [4096, 8192])
def test_fft_radix2_equals_library_fft(n):
    x = RNG.standard_normal((2, n)) + 1j * RNG.standard_normal((2, n))
    np.testing.assert_allclose(offt.fft_radix2(x), np.fft.fft(x), atol=1e-9)
    np.testing.assert_allclose(offt.fft_radix2(x, inverse=True), np.fft.ifft(x), atol=1e-13)


def test_parseval():
    n = 512
    x = RNG.standard_normal(n)
    spec = offt.fft_radix2(x)
    np.testing.assert_allclose(np.sum(x ** 2), np.sum(np.abs(spec) ** 2) / n, rtol=1e-12)


def test_real_transforms_roundtrip_and_library():
    n = 2048
    x = RNG.standard_normal(n)
    spec = offt.rfft(x)
    assert spec.shape == (n // 2 + 1,)
    np.testing.assert_allclose(spec, np.fft.rfft(x), atol=1e-10)
    np.testing.assert_allclose(offt.irfft(spec, n), x, atol=1e-12)


def test_fft_rejects_non_power_of_two():
    with pytest.raises(ValueError):
        offt.fft_radix2(np.zeros(12))
