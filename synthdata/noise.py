"""Coloured Gaussian noise with a known analytic one-sided PSD.

Stand-in for the paper's GWOSC O3 strain at 2048 Hz (Sec. IV.A),
which is not available offline.  Recipe (BASELINE.json configs[0]):

    S(f) = 1e-46 * ((f/30)^-4 + 1 + (f/300)^2)   evaluated at clip(f, 20, 1000) Hz

Frequency-domain synthesis in blocks of N_b samples, 50 %-overlapped and
cross-faded with w[n] = sin(pi n / N_b) (w^2 of the two overlapping blocks sums
to 1, so the PSD is preserved and there are no block-edge steps).

This is input generation only; it uses numpy's FFT freely.
"""
from __future__ import annotations

import numpy as np

FS = 2048.0


def analytic_psd(f):
    """One-sided PSD S(f) in strain^2/Hz; f clipped to [20, 1000] Hz (reading A10)."""
    f = np.clip(np.asarray(f, dtype=np.float64), 20.0, 1000.0)
    return 1e-46 * ((f / 30.0) ** -4 + 1.0 + (f / 300.0) ** 2)


def _sigma_analytic():
    # sigma^2 = int_0^{fs/2} S(clip f) df, closed form of the piecewise integrand
    a, b = 20.0, 1000.0
    flat_lo = analytic_psd(a) * a
    flat_hi = analytic_psd(b) * (FS / 2 - b)
    mid = 1e-46 * ((30.0 ** 4) * (a ** -3 - b ** -3) / 3.0 + (b - a) + (b ** 3 - a ** 3) / (3 * 300.0 ** 2))
    return float(np.sqrt(flat_lo + mid + flat_hi))


SIGMA_X_ANALYTIC = _sigma_analytic()  # ~7.16e-22


def _block(rng, n_b, fs):
    k = np.arange(n_b // 2 + 1)
    f = k * fs / n_b
    amp = np.sqrt(analytic_psd(f) * fs * n_b / 4.0)
    spec = amp * (rng.standard_normal(k.size) + 1j * rng.standard_normal(k.size))
    spec[0] = 0.0
    spec[-1] = spec[-1].real * np.sqrt(2.0)  # Nyquist bin is real
    return np.fft.irfft(spec, n_b)


def coloured_noise(n_samples, seed, n_channels=2, fs=FS, n_block=1 << 20, dtype=np.float32):
    """[n_channels][n_samples] noise; channel c uses SeedSequence(seed).spawn(n_channels)[c]."""
    n_samples = int(n_samples)
    n_block = int(min(n_block, 1 << int(np.ceil(np.log2(max(2 * n_samples, 4096))))))
    half = n_block // 2
    fade = np.sin(np.pi * np.arange(n_block) / n_block)
    out = np.empty((n_channels, n_samples), dtype=dtype)
    children = np.random.SeedSequence(seed).spawn(n_channels)
    for c in range(n_channels):
        rng = np.random.Generator(np.random.PCG64(children[c]))
        n_half = -(-n_samples // half)  # number of half-blocks needed
        acc = np.zeros((n_half + 1) * half, dtype=np.float64)
        prev = _block(rng, n_block, fs) * fade
        for i in range(n_half):
            cur = _block(rng, n_block, fs) * fade
            acc[i * half:(i + 1) * half] = prev[half:] + cur[:half]
            prev = cur
        out[c] = acc[:n_samples].astype(dtype)
    return out
