"""O-2 whitening-filter design and O-3 whitening.  (Oracle: test infrastructure only.)

Paper: "The remaining 2.5 s of the window is whitened in the frequency-domain, and
transformed back to time-domain.  Due to whitening filter settle-in, 0.5 s of data is
corrupted on both ends of the window and removed"; "build a whitening filter.
The remaining data is whitened, and half a second is cropped from both edges".
BASELINE.json: "divide by the square root of the interpolated PSD, band-limit, irFFT
with tapering".  The paper gives no formulas; readings A3-A6:

  design grid  f_d[k] = k fs / N_d, k = 0..N_d/2                               (A4)
  P_d          = linear interpolation of the Welch PSD (grid k fs/nfft_w) at f_d (A4)
  A[k]         = 1 / sqrt(P_d[k] fs / 2)  if f_lo <= f_d[k] <= f_hi else 0      (A3, A6)
  g[n]         = (1/N_d) (A[0] + (-1)^n A[N_d/2] + 2 sum_{k=1}^{N_d/2-1} A[k] cos(2 pi k n / N_d))
  h[j]         = g[|j|] cos^2(pi j / L),  j = -L/2..L/2  (h[+-L/2] = 0, zero phase)   (A5)
  y[m]         = sum_{j=-(L/2-1)}^{L/2-1} h[j] x[m - j],   L/2 <= m < N - L/2      (O-3)

Output index m' = m - L/2; the output has N - L samples (0.5 s removed per edge for L = 1 s).
"""
from __future__ import annotations

import numpy as np


def interp_psd_linear(psd, fs, nfft_w, n_design):
    """Linear interpolation of P (bin spacing fs/nfft_w) onto k fs / n_design, k = 0..n_design/2."""
    psd = np.asarray(psd, dtype=np.float64)
    out = np.empty(n_design // 2 + 1, dtype=np.float64)
    for k in range(n_design // 2 + 1):
        pos_num = k * nfft_w            # position in source bins = k * nfft_w / n_design (exact rational)
        i = pos_num // n_design
        frac = (pos_num - i * n_design) / n_design
        if i >= psd.shape[-1] - 1:
            out[k] = psd[-1]
        else:
            out[k] = (1.0 - frac) * psd[i] + frac * psd[i + 1]
    return out


def inverse_asd(psd_d, fs, n_design, f_lo, f_hi):
    """A[k] = 1/sqrt(P_d fs/2) inside [f_lo, f_hi] (inclusive), 0 outside."""
    k = np.arange(n_design // 2 + 1)
    f = k * fs / n_design
    band = (f >= f_lo) & (f <= f_hi)
    a = np.zeros_like(f)
    a[band] = 1.0 / np.sqrt(psd_d[band] * fs / 2.0)
    return a


def impulse_response(a, n_design, n_lags):
    """g[n], n = 0..n_lags: inverse real DFT (1/N_d on the inverse) of the real, even spectrum A."""
    k = np.arange(1, n_design // 2)
    g = np.empty(n_lags + 1, dtype=np.float64)
    for n in range(n_lags + 1):
        ph = (k * n) % n_design
        g[n] = (a[0] + (-1.0) ** n * a[n_design // 2]
                + 2.0 * np.sum(a[1: n_design // 2] * np.cos(2.0 * np.pi * ph / n_design))) / n_design
    return g


def design_filter(psd, fs=2048.0, nfft_w=4096, n_design=8192, filter_len=2048, f_lo=20.0, f_hi=1000.0):
    """Taps h[j + L/2], j = -L/2..L/2 (length L+1, both end taps exactly 0)."""
    half = filter_len // 2
    p_d = interp_psd_linear(psd, fs, nfft_w, n_design)
    a = inverse_asd(p_d, fs, n_design, f_lo, f_hi)
    g = impulse_response(a, n_design, half)
    j = np.arange(-half, half + 1)
    taper = np.cos(np.pi * j / filter_len) ** 2
    taper[0] = taper[-1] = 0.0
    return g[np.abs(j)] * taper


def whiten_fir_direct(x, h):
    """O-3 by direct summation, O(N L).  x: [..., N] -> [..., N - L]."""
    x = np.asarray(x, dtype=np.float64)
    half = (h.shape[-1] - 1) // 2
    n = x.shape[-1]
    n_out = n - 2 * half
    if n_out <= 0:
        return np.zeros(x.shape[:-1] + (0,), dtype=np.float64)
    y = np.zeros(x.shape[:-1] + (n_out,), dtype=np.float64)
    for j in range(-(half - 1), half):
        # y[m'] += h[j] x[m' + half - j]
        y += h[j + half] * x[..., half - j: half - j + n_out]
    return y


def whiten_fft(x, h):
    """The paper's wording: FFT the segment, multiply by DFT(h), inverse FFT, discard L/2 per
    edge.  numpy's FFT is the library primitive; tests prove this equals ``whiten_fir_direct``."""
    x = np.asarray(x, dtype=np.float64)
    half = (h.shape[-1] - 1) // 2
    n = x.shape[-1]
    if n - 2 * half <= 0:
        return np.zeros(x.shape[:-1] + (0,), dtype=np.float64)
    hc = np.zeros(n, dtype=np.float64)
    for j in range(-(half - 1), half):
        hc[j % n] += h[j + half]
    y = np.fft.irfft(np.fft.rfft(x, axis=-1) * np.fft.rfft(hc), n, axis=-1)
    return y[..., half: n - half]
