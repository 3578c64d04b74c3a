"""Analytic Newtonian inspiral chirps (stand-in for the paper's IMRPhenomPv2
injections; recipe SURVEY.md 8(d)).

With tau = t_c - t > 0 and Mc_s = M_c * 4.925491e-6 s:

    f(tau)   = (1/pi) (5 / (256 tau))^{3/8} Mc_s^{-5/8}
    phi(tau) = -2 (tau / (5 Mc_s))^{5/8} + phi0
    h(t)     ~ f^{2/3} cos(phi)     for 20 Hz <= f <= 300 Hz, 64-sample cos^2 ramps at both ends

The L1 copy is evaluated analytically at t - delta, |delta| <= 10 ms (light travel
time between the LIGO sites).  The pair is scaled to a network SNR rho:

    sum_det 4 sum_k |h~(f_k)|^2 / S(f_k) df = rho^2   over 20-1000 Hz.

Input generation only (uses numpy FFT for the SNR normalisation).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .noise import analytic_psd, FS

MSUN_S = 4.925491e-6
F_START, F_END = 20.0, 300.0


@dataclass
class ChirpParams:
    t_c: float        # coalescence time in seconds from sample 0 (H1 frame)
    m_chirp: float    # solar masses
    phi0: float
    delta_l1: float   # seconds, L1 arrival offset
    snr: float        # network SNR


def _tau_of_f(f, mc_s):
    return (5.0 / 256.0) * (np.pi * f) ** (-8.0 / 3.0) * mc_s ** (-5.0 / 3.0)


def newtonian_chirp(n_samples, t_c, m_chirp, phi0, fs=FS):
    """Unit-amplitude-law chirp on sample grid 0..n_samples-1 (float64) and its support [i0, i1)."""
    mc_s = m_chirp * MSUN_S
    tau_start = _tau_of_f(F_START, mc_s)
    tau_end = _tau_of_f(F_END, mc_s)
    i0 = int(np.ceil((t_c - tau_start) * fs))
    i1 = int(np.floor((t_c - tau_end) * fs)) + 1
    lo, hi = max(i0, 0), min(i1, n_samples)
    h = np.zeros(n_samples, dtype=np.float64)
    if hi <= lo:
        return h, (lo, lo)
    idx = np.arange(i0, i1)
    tau = t_c - idx / fs
    f = (1.0 / np.pi) * (5.0 / (256.0 * tau)) ** 0.375 * mc_s ** -0.625
    phi = -2.0 * (tau / (5.0 * mc_s)) ** 0.625 + phi0
    wave = f ** (2.0 / 3.0) * np.cos(phi)
    ramp = min(64, idx.size // 2)
    if ramp > 0:
        r = np.sin(0.5 * np.pi * (np.arange(ramp) + 0.5) / ramp) ** 2
        wave[:ramp] *= r
        wave[-ramp:] *= r[::-1]
    h[lo:hi] = wave[lo - i0:hi - i0]
    return h, (lo, hi)


def _snr_sq(h, fs=FS):
    """4 sum |h~|^2 / S df over 20-1000 Hz, h~ the continuous-FT approximation (dt * DFT)."""
    n = h.size
    spec = np.fft.rfft(h) / fs
    f = np.fft.rfftfreq(n, 1.0 / fs)
    band = (f >= 20.0) & (f <= 1000.0)
    return float(4.0 * np.sum(np.abs(spec[band]) ** 2 / analytic_psd(f[band])) * (fs / n))


def inject_chirps(strain, params, fs=FS):
    """Add chirps to strain [2][N] in float64 and return (float32 strain, per-chirp templates).

    templates[i] = (lo, hi, h_H1[lo:hi], h_L1[lo:hi]) after SNR scaling (float64), so tests can
    check the SNR pin without re-deriving anything.
    """
    out = np.asarray(strain, dtype=np.float64).copy()
    n = out.shape[1]
    templates = []
    for p in params:
        h0, (a0, b0) = newtonian_chirp(n, p.t_c, p.m_chirp, p.phi0, fs)
        h1, (a1, b1) = newtonian_chirp(n, p.t_c + p.delta_l1, p.m_chirp, p.phi0, fs)
        lo, hi = min(a0, a1), max(b0, b1)
        if hi <= lo:
            templates.append((lo, lo, np.zeros(0), np.zeros(0)))
            continue
        seg0, seg1 = h0[lo:hi], h1[lo:hi]
        # zero-pad to a power of two for the SNR integral
        npad = 1 << int(np.ceil(np.log2(max(hi - lo, 2) * 2)))
        z0 = np.zeros(npad); z0[:hi - lo] = seg0
        z1 = np.zeros(npad); z1[:hi - lo] = seg1
        rho2 = _snr_sq(z0, fs) + _snr_sq(z1, fs)
        scale = p.snr / np.sqrt(rho2) if rho2 > 0 else 0.0
        out[0, lo:hi] += scale * seg0
        out[1, lo:hi] += scale * seg1
        templates.append((lo, hi, scale * seg0, scale * seg1))
    return out.astype(np.float32), templates


def draw_chirp_params(n_chirps, duration_s, seed, slot_s=17.6, t_first=70.0):
    """Config-2 style draws: one chirp per ``slot_s`` slot, t_c uniform in the slot's middle 10 s."""
    rng = np.random.Generator(np.random.PCG64(seed))
    out = []
    for i in range(n_chirps):
        slot0 = t_first + i * slot_s
        if slot0 + slot_s > duration_s:
            break
        t_c = slot0 + 0.5 * (slot_s - 10.0) + 10.0 * rng.random()
        out.append(ChirpParams(
            t_c=float(t_c),
            m_chirp=float(rng.uniform(10.0, 60.0)),
            phi0=float(rng.uniform(0.0, 2 * np.pi)),
            delta_l1=float(rng.uniform(-0.010, 0.010)),
            snr=float(rng.uniform(4.0, 20.0)),
        ))
    return out
