"""O-1  Welch power spectral density.  (Oracle: test infrastructure only.)

Paper: "The first 8 s is used to estimate the power spectral density (PSD) used for
whitening" (Sec. IV.B); "the whitening module uses the first 64 seconds of the
snapshotter state to estimate the PSD" (Sec. VI).  The paper does not state the
estimator's parameters; BASELINE.json fixes "Welch PSD estimate with a Hann window and
50% overlap", fftlength 2 s.  Reading A1 adds: periodic Hann, per-segment
mean removal, one-sided density scaling, mean over segments.
"""
from __future__ import annotations

import numpy as np

from .fft import fft_radix2


def hann_periodic(n):
    """w[m] = 0.5 - 0.5 cos(2 pi m / n), m = 0..n-1."""
    return 0.5 - 0.5 * np.cos(2.0 * np.pi * np.arange(n) / n)


def segment_count(n_samples, nfft, hop):
    """J = floor((N - nfft)/hop) + 1 (63 for 64 s, 7 for 8 s at nfft 4096, hop 2048; reading A2)."""
    return (n_samples - nfft) // hop + 1 if n_samples >= nfft else 0


def periodogram(seg, fs, window):
    """One Welch segment: remove the mean, window, DFT, |X|^2 / (fs sum w^2), doubled for 0 < k < N/2."""
    seg = np.asarray(seg, dtype=np.float64)
    n = seg.shape[-1]
    seg = (seg - seg.mean(axis=-1, keepdims=True)) * window
    spec = fft_radix2(seg)[..., : n // 2 + 1]
    p = (spec.real ** 2 + spec.imag ** 2) / (fs * np.sum(window ** 2))
    p[..., 1: n // 2] *= 2.0
    return p


def median_bias(n):
    """NEXT-3 variant (the paper does not name its averaging, reading A1 is the mean): the median of
    n periodogram values of Gaussian noise (chi-squared with 2 degrees of freedom, i.e. exponential) underestimates
    their mean by sum_{i=1}^{m} (-1)^(i+1) / i, m = n for odd n and n - 1 for even n (-> ln 2)."""
    m = n if n % 2 else n - 1
    return sum((1.0 if i % 2 else -1.0) / i for i in range(1, m + 1))


def welch(x, fs=2048.0, nfft=4096, hop=2048, average="mean"):
    """P[k], k = 0..nfft/2, in x-units^2/Hz: mean (reading A1) over the J segments x[hop j : hop j + nfft], or, for
    average="median", their per-bin median divided by median_bias(J)."""
    x = np.asarray(x, dtype=np.float64)
    j_total = segment_count(x.shape[-1], nfft, hop)
    if j_total < 1:
        raise ValueError("need at least one full segment")
    w = hann_periodic(nfft)
    if average == "median":
        pg = np.stack([periodogram(x[..., hop * j: hop * j + nfft], fs, w) for j in range(j_total)])
        return np.median(pg, axis=0) / median_bias(j_total)
    if average != "mean":
        raise ValueError("average must be 'mean' or 'median'")
    acc = np.zeros(x.shape[:-1] + (nfft // 2 + 1,), dtype=np.float64)
    for j in range(j_total):
        acc += periodogram(x[..., hop * j: hop * j + nfft], fs, w)
    return acc / j_total
