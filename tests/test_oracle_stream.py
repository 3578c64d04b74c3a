"""Pins for oracle/stream.py (O-4, O-6; readings C1-C3) and the paper's geometry constants."""
import numpy as np

from oracle import stream as ost
from oracle import whiten as owh
from oracle import psd as opsd
from synthdata import coloured_noise

FS = 2048


def _golden():
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                name, value = line.split()[:2]
                out[name] = float(value)
    return out


def test_golden_paper_constants_are_mutually_consistent_and_match_the_defaults():
    g = _golden()
    assert g["training_window"] == g["training_psd_length"] + g["training_whitened_length"]          # 10.5 = 8 + 2.5
    assert g["training_whitened_length"] - 2 * g["whitening_crop_per_edge"] == g["kernel_length"]    # 2.5 - 1 = 1.5
    assert g["window_shift"] == 1.0 / g["inference_rate"]
    assert g["kernel_length"] - g["window_shift"] == g["window_overlap"]
    cfg = ost.StreamConfig()
    assert cfg.fs == g["sample_rate"] and cfg.kernel_len == g["kernel_length"] * cfg.fs
    assert cfg.filter_len == 2 * g["whitening_crop_per_edge"] * cfg.fs and cfg.psd_len == g["inference_psd_length"] * cfg.fs


def test_paper_geometry_constants():
    # 10.5 s = 8 s PSD + 2.5 s whitened; 0.5 s cropped per edge -> 1.5 s analysed
    assert 10.5 * FS == 8 * FS + 2.5 * FS
    assert int(2.5 * FS) - 2 * (FS // 2) == int(1.5 * FS) == 3072
    # 1.5 s windows shifted 0.25 s overlap by 1.25 s; batch 128 at 4 Hz
    assert 3072 - 512 == int(1.25 * FS)
    # snapshotter state: PSD length + (batch-1) strides + kernel + filter
    assert 64 * FS + 127 * 512 + 3072 + 2048 == 201216


def test_unfold_definition():
    y = np.arange(2 * 100).reshape(2, 100)
    w = ost.unfold(y, kernel_len=10, stride=4, first=3, shifts=[0, 8], n_windows=5)
    assert w.shape == (5, 2, 10)
    np.testing.assert_array_equal(w[2, 0], y[0, 3 + 8: 3 + 18])
    np.testing.assert_array_equal(w[2, 1], y[1, 3 + 8 + 8: 3 + 8 + 18])
    assert ost.unfold(y, 10, 4).shape[0] == (100 - 10) // 4 + 1


def test_timeslide_window_count_closed_form():
    assert ost.timeslide_window_count(100000, 3072, 128, 2048) == (100000 - 2048 - 3072) // 128 + 1
    assert ost.timeslide_window_count(4000, 3072, 128, 2048) == 0


def _small_cfg():
    # scaled-down geometry (same rule, 16x shorter) so the state machine runs in seconds
    return ost.StreamConfig(welch_nfft=256, welch_hop=128, filter_len=128, n_design=512, f_lo=20.0, f_hi=1000.0,
                            kernel_len=192, stride=8, psd_len=2048, psd_update=512)


def test_first_index_and_epoch_closed_forms():
    cfg = ost.StreamConfig()
    assert ost.first_whitened_index(cfg) == 131072 - 128 - 1024 == 129920
    assert ost.epoch_of_sample(129920, cfg) == 0
    assert ost.epoch_of_sample(129920 + 16383, cfg) == 0
    assert ost.epoch_of_sample(129920 + 16384, cfg) == 1


def test_stream_equals_batch_sample_for_sample():
    cfg = _small_cfg()
    x = coloured_noise(2048 + 3 * 512 + 64, seed=77).astype(np.float64) * 2.0 ** 70
    so = ost.StreamOracle(cfg, net=None)
    n_updates = x.shape[1] // cfg.stride
    first_window_update, wins = None, []
    for u in range(n_updates):
        r = so.step(x[:, u * cfg.stride: (u + 1) * cfg.stride])
        if r is not None:
            if first_window_update is None:
                first_window_update = u
            wins.append(r)
    # C1: first PSD at n = psd_len (update psd_len/s - 1); first window K/s - 1 updates later
    assert first_window_update == cfg.psd_len // cfg.stride - 1 + cfg.kernel_len // cfg.stride - 1
    assert so.n_psd_updates == 1 + (n_updates * cfg.stride - cfg.psd_len) // cfg.psd_update
    for c in range(2):
        y, m_lo = ost.whiten_rolling(x[c], cfg)
        assert m_lo == ost.first_whitened_index(cfg)
        np.testing.assert_allclose(so.white[c], y, rtol=0, atol=1e-12)
    # windows are the unfold of the whitened stream
    yb = np.stack([ost.whiten_rolling(x[c], cfg)[0] for c in range(2)])
    ub = ost.unfold(yb, cfg.kernel_len, cfg.stride)
    assert len(wins) == ub.shape[0]
    np.testing.assert_allclose(np.stack(wins), ub, atol=1e-12)


def test_epoch_switch_uses_new_filter_from_the_specified_sample():
    cfg = _small_cfg()
    x = coloured_noise(2048 + 2 * 512, seed=78, n_channels=1)[0].astype(np.float64) * 2.0 ** 70
    y, m_lo = ost.whiten_rolling(x, cfg)
    half = cfg.filter_len // 2
    m_sw = cfg.psd_len + cfg.psd_update - cfg.stride - half        # first sample of epoch 1
    h0, h1 = ost.epoch_filter(x, 0, cfg), ost.epoch_filter(x, 1, cfg)
    y0 = owh.whiten_fir_direct(x[m_sw - 1 - half: m_sw + half], h0)[0]
    y1 = owh.whiten_fir_direct(x[m_sw - half: m_sw + 1 + half], h1)[0]
    np.testing.assert_allclose(y[m_sw - 1 - m_lo], y0, atol=1e-12)
    np.testing.assert_allclose(y[m_sw - m_lo], y1, atol=1e-12)
    assert not np.allclose(h0, h1)


def test_timeslide_commutes_with_whitening():
    # A8/C3: whitening is per channel, so shifting whitened L1 == whitening shifted L1 (fixed filter)
    x = coloured_noise(16 * 2048, seed=79).astype(np.float64)
    h = [owh.design_filter(opsd.welch(x[c], 2048.0, 4096, 2048)) for c in range(2)]
    y = np.stack([owh.whiten_fft(x[c], h[c]) for c in range(2)])
    shift = 2048
    a = ost.unfold(y, 3072, 128, shifts=[0, shift], n_windows=8)
    y_shifted = owh.whiten_fft(x[1, shift:], h[1])
    b = ost.unfold(np.stack([y[0, : y_shifted.size], y_shifted]), 3072, 128, n_windows=8)
    np.testing.assert_allclose(a, b, atol=1e-10)
