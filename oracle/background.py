"""NEXT-4  background bookkeeping and the training-time whitening batch.  (Oracle: test infrastructure only.)

False-alarm rate.  Paper: "the Hanford strain data is held fixed and the Livingston data is shifted in 1 s increments
until the required background livetime is accumulated.  Then, a false alarm rate (FAR) can be assigned to injected
events by dividing the number of background events with detection statistic greater than the event of interest, with
livetime analyzed." (Sec. VI).  So FAR(e) = #{b in background : b > e} / T_bg, with a STRICT inequality
(the paper's "greater than"); an event as loud as the loudest background trigger gets FAR 0 (the paper quotes such events
as "less than 1 per year", the minimum its one year of background resolves).

Training-time whitening batch.  Paper: "The length of each noise window sampled from disk is 10.5 s.  The first 8 s is
used to estimate the power spectral density (PSD) used for whitening.  The remaining 2.5 s of the window is whitened in
the frequency-domain, and transformed back to time-domain.  Due to whitening filter settle-in, 0.5 s of data is
corrupted on both ends of the window and removed.  Thus, only 1.5 s of data is actually analyzed by the neural-network.
[...] We use a training batch size of 384" (Sec. IV.B).  Every batch element and detector has its OWN PSD and
filter; the steps are O-1, O-2, O-3 of the hot path (readings A1-A6) applied per (element, detector).
"""
from __future__ import annotations

import numpy as np

from . import psd as _psd
from . import whiten as _wh


def far_counts(background, events):
    """n[i] = number of background statistics strictly greater than events[i] (plain double loop)."""
    background = np.asarray(background)
    events = np.asarray(events)
    out = np.zeros(events.shape[0], dtype=np.int64)
    for i in range(events.shape[0]):
        n = 0
        for b in background:
            if b > events[i]:
                n += 1
        out[i] = n
    return out


def far(background, events, livetime_s):
    """FAR in 1/s: far_counts / T_bg (float64 division)."""
    return far_counts(background, events).astype(np.float64) / np.float64(livetime_s)


def whiten_training_batch(x, n_psd, fs=2048.0, nfft=4096, hop=2048, n_design=8192, filter_len=2048, f_lo=20.0,
                          f_hi=1000.0):
    """x: [B][C][n] raw strain.  Per (b, c): PSD from x[b, c, :n_psd], taps from that PSD, whitening of x[b, c, n_psd:],
    filter_len/2 samples dropped per edge.  Returns [B][C][n - n_psd - filter_len]."""
    x = np.asarray(x, dtype=np.float64)
    B, C, n = x.shape
    out = np.empty((B, C, n - n_psd - filter_len), dtype=np.float64)
    for b in range(B):
        for c in range(C):
            p = _psd.welch(x[b, c, :n_psd], fs=fs, nfft=nfft, hop=hop)
            h = _wh.design_filter(p, fs=fs, nfft_w=nfft, n_design=n_design, filter_len=filter_len, f_lo=f_lo, f_hi=f_hi)
            out[b, c] = _wh.whiten_fft(x[b, c, n_psd:], h)
    return out
