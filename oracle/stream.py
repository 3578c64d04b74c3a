"""O-4 window unfold, O-6 streaming / rolling-PSD rule, timeslides.  (Oracle: test infrastructure only.)

Paper: "Clients send streaming updates of strain data to a snapshotter [...] the whitening module
uses the first 64 seconds of the snapshotter state to estimate the PSD and build a whitening
filter.  The remaining data is whitened, and half a second is cropped from both edges [...] The
whitened data is then unfolded into a batch of overlapping windows" (Sec. VI);
"the Hanford strain data is held fixed and the Livingston data is shifted in 1 s increments"
(Sec. IX).  BASELINE.json configs[2]: "PSD re-estimated every 8 s from trailing 64 s; 1.5 s
windows at 16 Hz stride (128 samples)".  Readings C1-C3, A7 fix what the paper leaves open:

  update u delivers raw samples [s u, s u + s); n = s (u + 1)
  if n >= psd_len and (n - psd_len) mod psd_update == 0:  P <- Welch(x[n - psd_len : n]); h <- design(P)
  if a filter exists: whitened samples m in [n - s - L/2, n - L/2) are produced with the CURRENT h and
     appended; they are never recomputed
  once >= K whitened samples exist, the newest K per channel form the window -> one score

The offline rule is the same rule applied to a stored segment, so stream and batch agree sample for
sample: sample m uses the filter of epoch e(m) = floor((n(m) - psd_len) / psd_update),
n(m) = s (floor((m + L/2) / s) + 1).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import psd as _psd
from . import whiten as _wh
from . import network as _net


@dataclass
class StreamConfig:
    fs: float = 2048.0
    welch_nfft: int = 4096
    welch_hop: int = 2048
    filter_len: int = 2048
    n_design: int = 8192
    f_lo: float = 20.0
    f_hi: float = 1000.0
    kernel_len: int = 3072
    stride: int = 128
    psd_len: int = 131072
    psd_update: int = 16384
    welch_average: str = "mean"      # NEXT-3 variant: "median" (oracle/psd.py)


def unfold(y, kernel_len, stride, first=0, shifts=None, n_windows=None):
    """O-4: win[i][c][n] = y[c][first + i*stride + shift_c + n]."""
    y = np.asarray(y)
    c_tot, n_y = y.shape
    shifts = [0] * c_tot if shifts is None else list(shifts)
    avail = min((n_y - first - sh - kernel_len) // stride + 1 for sh in shifts)
    if n_windows is None:
        n_windows = max(avail, 0)
    if n_windows > avail:
        raise ValueError("not enough whitened samples for the requested windows")
    out = np.empty((n_windows, c_tot, kernel_len), dtype=y.dtype)
    for i in range(n_windows):
        for c in range(c_tot):
            a = first + i * stride + shifts[c]
            out[i, c] = y[c, a: a + kernel_len]
    return out


def timeslide_window_count(n_y, kernel_len, stride, shift):
    """Reading C3: no wrap-around; slide with L1 shift `shift` has floor((N_y - shift - K)/s) + 1 windows."""
    v = (n_y - shift - kernel_len) // stride + 1
    return max(v, 0)


def first_whitened_index(cfg: StreamConfig):
    """Raw-sample index of the first whitened sample: psd_len - stride - L/2 (reading C1)."""
    return cfg.psd_len - cfg.stride - cfg.filter_len // 2


def epoch_of_sample(m, cfg: StreamConfig):
    n_m = cfg.stride * ((m + cfg.filter_len // 2) // cfg.stride + 1)
    return (n_m - cfg.psd_len) // cfg.psd_update


def epoch_filter(x, e, cfg: StreamConfig):
    """Filter of PSD epoch e: Welch over x[n_e - psd_len : n_e], n_e = psd_len + e psd_update."""
    n_e = cfg.psd_len + e * cfg.psd_update
    p = _psd.welch(x[n_e - cfg.psd_len: n_e], cfg.fs, cfg.welch_nfft, cfg.welch_hop, cfg.welch_average)
    return _wh.design_filter(p, cfg.fs, cfg.welch_nfft, cfg.n_design, cfg.filter_len, cfg.f_lo, cfg.f_hi)


def whiten_rolling(x, cfg: StreamConfig, m_lo=None, m_hi=None, filters=None):
    """Offline form of O-6 for one channel x[N]: whitened samples for raw indices [m_lo, m_hi)
    (defaults: everything the streaming rule would have produced).  Returns (y, m_lo).
    filters: optional dict {epoch: taps} of THIS channel, filled on first use, so that many short requests on
    one record design each epoch's filter once (memoisation only; the arithmetic is epoch_filter's)."""
    x = np.asarray(x, dtype=np.float64)
    half = cfg.filter_len // 2
    n_eff = (x.shape[0] // cfg.stride) * cfg.stride
    lo_all, hi_all = first_whitened_index(cfg), n_eff - half
    m_lo = lo_all if m_lo is None else m_lo
    m_hi = hi_all if m_hi is None else m_hi
    if m_lo < lo_all or m_hi > hi_all:
        raise ValueError("requested samples are outside what the streaming rule produces")
    y = np.empty(max(m_hi - m_lo, 0), dtype=np.float64)
    m = m_lo
    while m < m_hi:
        e = epoch_of_sample(m, cfg)
        m_next = min(cfg.psd_len + (e + 1) * cfg.psd_update - cfg.stride - half, m_hi)  # first sample of epoch e+1
        if filters is None:
            h = epoch_filter(x, e, cfg)
        else:
            if e not in filters:
                filters[e] = epoch_filter(x, e, cfg)
            h = filters[e]
        y[m - m_lo: m_next - m_lo] = _wh.whiten_fir_direct(x[m - half: m_next + half], h)
        m = m_next
    return y, m_lo


class StreamOracle:
    """O-6 as a state machine fed ``stride`` samples per channel at a time."""

    def __init__(self, cfg: StreamConfig, net=None, n_channels=2):
        self.cfg, self.net, self.c = cfg, net, n_channels
        self.raw = np.zeros((n_channels, 0), dtype=np.float64)
        self.white = np.zeros((n_channels, 0), dtype=np.float64)
        self.h = None
        self.n = 0
        self.n_psd_updates = 0

    def step(self, new_samples):
        cfg = self.cfg
        new_samples = np.asarray(new_samples, dtype=np.float64)
        assert new_samples.shape == (self.c, cfg.stride)
        self.raw = np.concatenate([self.raw, new_samples], axis=1)
        self.n += cfg.stride
        n, half = self.n, cfg.filter_len // 2
        if n >= cfg.psd_len and (n - cfg.psd_len) % cfg.psd_update == 0:
            self.h = [
                _wh.design_filter(_psd.welch(self.raw[c, n - cfg.psd_len: n], cfg.fs, cfg.welch_nfft, cfg.welch_hop,
                                             cfg.welch_average),
                                  cfg.fs, cfg.welch_nfft, cfg.n_design, cfg.filter_len, cfg.f_lo, cfg.f_hi)
                for c in range(self.c)]
            self.n_psd_updates += 1
        if self.h is None:
            return None
        seg = self.raw[:, n - cfg.stride - 2 * half: n]            # exactly stride outputs
        new_w = np.stack([_wh.whiten_fir_direct(seg[c], self.h[c]) for c in range(self.c)])
        self.white = np.concatenate([self.white, new_w], axis=1)
        if self.white.shape[1] < cfg.kernel_len:
            return None
        win = self.white[:, -cfg.kernel_len:]
        if self.net is None:
            return win.copy()
        return float(_net.forward(self.net, win[None])[0])
