"""Pins for oracle/whiten.py (O-2, O-3; readings A3-A6, A9)."""
import numpy as np
import scipy.signal

from oracle import psd as opsd
from oracle import whiten as owh
from synthdata import analytic_psd, coloured_noise

RNG = np.random.default_rng(13)
FS = 2048.0


def _psd_grid(nfft=4096):
    return analytic_psd(np.arange(nfft // 2 + 1) * FS / nfft)


def test_interp_is_identity_on_the_welch_grid():
    p = RNG.random(2049) + 0.5
    np.testing.assert_array_equal(owh.interp_psd_linear(p, FS, 4096, 4096), p)


def test_interp_midpoints_closed_form():
    p = RNG.random(2049) + 0.5
    q = owh.interp_psd_linear(p, FS, 4096, 8192)
    assert q.shape == (4097,)
    np.testing.assert_array_equal(q[0::2], p)
    np.testing.assert_allclose(q[1::2], 0.5 * (p[:-1] + p[1:]), rtol=1e-15)


def test_band_mask_bin_indices():
    for n_d, lo, hi in [(8192, 80, 4000), (4096, 40, 2000)]:
        a = owh.inverse_asd(np.ones(n_d // 2 + 1), FS, n_d, 20.0, 1000.0)
        nz = np.nonzero(a)[0]
        assert nz[0] == lo and nz[-1] == hi and nz.size == hi - lo + 1


def test_flat_psd_gives_one_over_sigma():
    sigma = 4.0
    p = np.full(4097, 2 * sigma ** 2 / FS)
    a = owh.inverse_asd(p, FS, 8192, 20.0, 1000.0)
    np.testing.assert_allclose(a[80:4001], 1.0 / sigma, rtol=1e-15)
    assert a[79] == 0 and a[4001] == 0


def test_impulse_response_equals_library_irfft():
    a = owh.inverse_asd(owh.interp_psd_linear(_psd_grid(), FS, 4096, 8192), FS, 8192, 20.0, 1000.0)
    g = owh.impulse_response(a, 8192, 1024)
    ref = np.fft.irfft(a, 8192)
    np.testing.assert_allclose(g, ref[:1025], rtol=1e-9, atol=1e-9 * np.abs(ref).max())


def test_taps_shape_symmetry_and_zero_ends():
    h = owh.design_filter(_psd_grid())
    assert h.shape == (2049,)
    assert h[0] == 0.0 and h[-1] == 0.0
    np.testing.assert_array_equal(h, h[::-1])
    assert np.count_nonzero(h) <= 2047 and np.count_nonzero(h) > 2000


def test_taper_is_cos_squared_hann():
    # with A == 1 everywhere in band the taper can be read back: h[j]/g[|j|]
    p = np.full(2049, 2.0 / FS)
    a = owh.inverse_asd(owh.interp_psd_linear(p, FS, 4096, 8192), FS, 8192, 20.0, 1000.0)
    g = owh.impulse_response(a, 8192, 1024)
    h = owh.design_filter(p)
    np.testing.assert_allclose(h[1024], g[0], rtol=1e-15)                       # centre tap untouched
    np.testing.assert_allclose(h[1024 + 512], g[512] * 0.5, rtol=1e-12)         # cos^2(pi/4) = 1/2
    hann_sym = scipy.signal.get_window("hann", 2049, fftbins=False)             # library Hann, 2049 points
    np.testing.assert_allclose(h, g[np.abs(np.arange(-1024, 1025))] * hann_sym, atol=1e-15)


def test_fir_direct_equals_library_convolution():
    h = owh.design_filter(_psd_grid())
    x = RNG.standard_normal(6000)
    y = owh.whiten_fir_direct(x, h)
    ref = np.convolve(x, h, mode="valid")       # full taps incl. the two zero end taps
    assert y.shape == (6000 - 2048,)
    np.testing.assert_allclose(y, ref, atol=1e-12 * np.abs(ref).max())


def test_fir_index_convention_with_asymmetric_taps():
    # asymmetric taps expose a flipped / off-by-one index: y[m] = sum_j h[j] x[m-j]
    half = 4
    h = np.zeros(2 * half + 1); h[half + 2] = 1.0     # h[j=+2] = 1  ->  y[m] = x[m-2]
    x = np.arange(40.0)
    y = owh.whiten_fir_direct(x, h)
    np.testing.assert_array_equal(y, x[half - 2: half - 2 + y.size])


def test_fft_whitening_equals_direct_sum_and_is_segment_invariant():
    h = owh.design_filter(_psd_grid())
    x = RNG.standard_normal(20000)
    y_long = owh.whiten_fir_direct(x, h)                    # long-stream FIR output
    np.testing.assert_allclose(owh.whiten_fft(x, h), y_long, atol=1e-11)
    # reading A5: a 5120-sample segment whitened alone (circular FFT, crop 1024 per edge)
    a = 7000
    seg = owh.whiten_fft(x[a: a + 5120], h)
    assert seg.shape == (3072,)
    np.testing.assert_allclose(seg, y_long[a: a + 3072], atol=1e-11)


def test_scale_invariance_power_of_two():
    x = coloured_noise(16 * 2048, seed=5, n_channels=1)[0].astype(np.float64)
    def run(v):
        return owh.whiten_fir_direct(v[:8192], owh.design_filter(opsd.welch(v, FS, 4096, 2048)))
    y0, y1 = run(x), run(x * 2.0 ** 70)
    np.testing.assert_allclose(y1, y0, rtol=0, atol=4e-15 * np.abs(y0).max())


def test_whitened_coloured_noise_is_flat_unit_variance():
    # BASELINE.json north_star pin: noise coloured by the analytic S(f), whitened with the filter
    # designed from that same analytic PSD -> in-band PSD*fs/2 = 1, variance = band fraction 980/1024
    x = coloured_noise(128 * 2048, seed=21, n_channels=1)[0].astype(np.float64)
    h = owh.design_filter(_psd_grid())
    y = owh.whiten_fft(x, h)
    p = opsd.welch(y, FS, 4096, 2048) * FS / 2
    inband = p[2 * 25: 2 * 990]
    np.testing.assert_allclose(inband.mean(), 1.0, rtol=0.02)
    assert np.abs(np.log(inband)).max() < 0.6            # flat: 127 averages -> ~9 % scatter per bin
    np.testing.assert_allclose(y.var(), 980.0 / 1024.0, rtol=0.02)
    assert p[4: 2 * 15].max() < 1e-6 and p[2 * 1010:].max() < 1e-6   # band-limited (bins 0-1: detrend leakage)


def test_self_estimated_psd_whitening_statistics():
    # reading A6 tolerance: E[1/P_hat] bias ~ +1.7 % with 63 overlapped Hann averages
    x = coloured_noise(64 * 2048, seed=1000)[0].astype(np.float64)
    h = owh.design_filter(opsd.welch(x, FS, 4096, 2048))
    y = owh.whiten_fft(x, h)
    np.testing.assert_allclose(y.var(), 980.0 / 1024.0, rtol=0.03)


def test_frequency_response_tracks_inverse_asd():
    p = _psd_grid()
    h = owh.design_filter(p)
    hc = np.zeros(8192); hc[np.arange(-1024, 1025) % 8192] = h
    resp = np.fft.rfft(hc)
    assert np.abs(resp.imag).max() < 1e-9 * np.abs(resp.real).max()          # zero phase
    a = owh.inverse_asd(owh.interp_psd_linear(p, FS, 4096, 8192), FS, 8192, 20.0, 1000.0)
    k = np.arange(4 * 40, 4 * 900)
    np.testing.assert_allclose(resp.real[k], a[k], rtol=0.02)
