"""Checks of the seeded input generators (shapes, spectra, SNR scaling, determinism)."""
import numpy as np

from oracle import psd as opsd
from oracle import whiten as owh
from synthdata import analytic_psd, coloured_noise, SIGMA_X_ANALYTIC, inject_chirps, ChirpParams
from synthdata.chirps import draw_chirp_params, newtonian_chirp

FS = 2048.0


def test_noise_matches_analytic_psd_and_sigma():
    x = coloured_noise(256 * 2048, seed=1001)
    assert x.shape == (2, 256 * 2048) and x.dtype == np.float32
    np.testing.assert_allclose(x.astype(np.float64).std(), SIGMA_X_ANALYTIC, rtol=0.03)
    assert abs(SIGMA_X_ANALYTIC - 7.16e-22) < 0.02e-22
    p = opsd.welch(x[0].astype(np.float64), FS, 4096, 2048)
    f = np.arange(2049) * 0.5
    ratio = p[60:1990] / analytic_psd(f[60:1990])
    np.testing.assert_allclose(ratio.mean(), 1.0, rtol=0.03)
    # channels independent
    c = np.corrcoef(x[0], x[1])[0, 1]
    assert abs(c) < 0.02


def test_noise_is_deterministic_in_the_seed():
    a = coloured_noise(8192, seed=5); b = coloured_noise(8192, seed=5); c = coloured_noise(8192, seed=6)
    np.testing.assert_array_equal(a, b)
    assert not np.array_equal(a, c)


def test_chirp_frequency_sweep_and_duration():
    h, (lo, hi) = newtonian_chirp(16 * 2048, t_c=10.0, m_chirp=10.0, phi0=0.0)
    np.testing.assert_allclose((hi - lo) / FS, 4.73, atol=0.05)       # 4.73 s from 20 Hz at Mc = 10
    h2, (lo2, hi2) = newtonian_chirp(16 * 2048, t_c=10.0, m_chirp=60.0, phi0=0.0)
    np.testing.assert_allclose((hi2 - lo2) / FS, 0.24, atol=0.02)
    assert h[:lo].max() == 0 and h[hi:].max() == 0


def test_injection_snr_pin_whitened_template_energy():
    # pin: per-detector whitened-template energy sums to rho^2/2 each (equal amplitudes)
    n = 32 * 2048
    p = ChirpParams(t_c=20.0, m_chirp=30.0, phi0=1.0, delta_l1=0.004, snr=10.0)
    _, tmpl = inject_chirps(np.zeros((2, n)), [p])
    lo, hi, h0, h1 = tmpl[0]
    h = owh.design_filter(analytic_psd(np.arange(2049) * 0.5))
    e = []
    for seg in (h0, h1):
        z = np.zeros(n); z[lo:hi] = seg
        e.append(np.sum(owh.whiten_fft(z, h) ** 2))
    np.testing.assert_allclose(e[0] + e[1], 100.0, rtol=0.02)
    np.testing.assert_allclose(e[0], 50.0, rtol=0.03)


def test_draw_chirp_params_ranges():
    ps = draw_chirp_params(200, 3600.0, seed=2002)
    assert len(ps) == 200
    assert all(10 <= p.m_chirp <= 60 and 4 <= p.snr <= 20 and abs(p.delta_l1) <= 0.01 for p in ps)
