"""Discrete Fourier transforms, float64/complex128.  (Oracle: test infrastructure only.)

Conventions: forward transforms are unnormalised,
X[k] = sum_n x[n] exp(-2 pi i n k / N); the inverse carries the 1/N factor.

``dft_naive`` is the definition written out (O(N^2)).  ``fft_radix2`` is the oracle's own
power-of-two FFT; tests prove the two equal, after which the rest of the oracle may use
either (or numpy's FFT as a library primitive, which the tests also compare).
"""
from __future__ import annotations

import numpy as np


def dft_naive(x, inverse=False):
    """X[k] = sum_n x[n] exp(-/+ 2 pi i n k / N), O(N^2), evaluated row by row."""
    x = np.asarray(x, dtype=np.complex128)
    n = x.shape[-1]
    sign = 2.0 if inverse else -2.0
    idx = np.arange(n)
    out = np.empty_like(x)
    for k in range(n):
        # reduce n*k mod N in integers so the phase stays accurate for large N
        ph = (idx * k) % n
        out[..., k] = np.sum(x * np.exp(1j * sign * np.pi * ph / n), axis=-1)
    return out / n if inverse else out


def fft_radix2(x, inverse=False):
    """Iterative decimation-in-time radix-2 FFT along the last axis (N a power of two)."""
    x = np.array(x, dtype=np.complex128)
    n = x.shape[-1]
    if n & (n - 1):
        raise ValueError("fft_radix2 needs a power-of-two length")
    bits = n.bit_length() - 1
    rev = np.zeros(n, dtype=np.int64)
    for b in range(bits):
        rev |= ((np.arange(n) >> b) & 1) << (bits - 1 - b)
    x = x[..., rev]
    sign = 2.0 if inverse else -2.0
    half = 1
    while half < n:
        w = np.exp(1j * sign * np.pi * np.arange(half) / (2 * half))
        x = x.reshape(x.shape[:-1] + (n // (2 * half), 2, half))
        even = x[..., 0, :]
        odd = x[..., 1, :] * w
        x = np.concatenate([even + odd, even - odd], axis=-1).reshape(x.shape[:-3] + (n,))
        half *= 2
    return x / n if inverse else x


def rfft(x):
    """One-sided spectrum X[0..N/2] of a real sequence."""
    x = np.asarray(x, dtype=np.float64)
    return fft_radix2(x)[..., : x.shape[-1] // 2 + 1]


def irfft(spec, n):
    """Real sequence of length n from its one-sided spectrum (Hermitian extension, 1/n on the inverse)."""
    spec = np.asarray(spec, dtype=np.complex128)
    full = np.empty(spec.shape[:-1] + (n,), dtype=np.complex128)
    full[..., : n // 2 + 1] = spec
    full[..., n // 2 + 1:] = np.conj(spec[..., 1: n // 2][..., ::-1])
    full[..., 0] = full[..., 0].real
    full[..., n // 2] = full[..., n // 2].real
    return fft_radix2(full, inverse=True).real
