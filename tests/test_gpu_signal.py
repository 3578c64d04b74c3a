"""GPU parity (through the C ABI) of the signal path against the float64 oracle: O-1 Welch PSD,
O-2 filter taps, O-3 whitening, O-6 rolling whitening.  Tolerances: rules T1 of DESIGN.md."""
import numpy as np
import pytest
import torch

from oracle import psd as opsd
from oracle import stream as ost
from oracle import whiten as owh
from synthdata import coloured_noise
from synthdata.configs import config0_strain

pytestmark = pytest.mark.gpu
FS = 2048.0
SCALE2 = 2.0 ** 140


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


@pytest.fixture(scope="module")
def cfg0(af):
    x = config0_strain()
    return dict(x=x, xd=torch.from_numpy(x).cuda(), x64=x.astype(np.float64))


def test_welch_psd_matches_oracle_config0(af, cfg0):
    ctx = af.Context(n_design=4096, kernel_len=2048, precision=af.FP32)
    p = ctx.psd_welch(cfg0["xd"]).cpu().numpy().astype(np.float64) / SCALE2
    ref = np.stack([opsd.welch(cfg0["x64"][c]) for c in range(2)])
    band = slice(40, 2001)                                       # 20-1000 Hz at df = 0.5 Hz
    rel = np.abs(p[:, band] - ref[:, band]) / ref[:, band]
    assert rel.max() <= 1e-4, rel.max()
    # outside the band only the level matters (bins near DC are detrend leakage)
    assert np.abs(p[:, 4:] - ref[:, 4:]).max() <= 1e-3 * ref[:, 4:].max()


@pytest.mark.parametrize("n_samples", [4096, 4096 + 2047, 10 * 2048 + 5])
def test_welch_ragged_lengths(af, cfg0, n_samples):
    ctx = af.Context(precision=af.FP32)
    p = ctx.psd_welch(cfg0["xd"][:, :n_samples].contiguous()).cpu().numpy().astype(np.float64) / SCALE2
    ref = np.stack([opsd.welch(cfg0["x64"][c, :n_samples]) for c in range(2)])
    rel = np.abs(p[:, 40:2001] - ref[:, 40:2001]) / ref[:, 40:2001]
    assert rel.max() <= 1e-4


@pytest.mark.parametrize("n_design", [4096, 8192])
def test_filter_taps_and_whitening_match_oracle(af, cfg0, n_design):
    ctx = af.Context(n_design=n_design, kernel_len=2048, precision=af.FP32)
    psd = ctx.psd_welch(cfg0["xd"])
    white = ctx.whiten(cfg0["xd"], psd).cpu().numpy().astype(np.float64)
    taps = ctx.filter_taps().cpu().numpy().astype(np.float64) * 2.0 ** 70      # scaled units -> physical
    assert white.shape == (2, 64 * 2048 - 2048)
    for c in range(2):
        h = owh.design_filter(opsd.welch(cfg0["x64"][c]), n_design=n_design)
        assert np.abs(taps[c] - h).max() <= 2e-5 * np.abs(h).max()
        assert taps[c][0] == 0 and taps[c][-1] == 0
        y = owh.whiten_fft(cfg0["x64"][c], h)
        rms = np.sqrt(np.mean(y ** 2))
        assert np.abs(white[c] - y).max() <= 1e-4 * rms, np.abs(white[c] - y).max() / rms      # T1


def test_whitening_direct_sum_samples_and_ragged_tail(af, cfg0):
    # length that is not a multiple of the overlap-save hop: several blocks and a ragged tail
    n = 6144 * 3 + 2048 + 777
    ctx = af.Context(precision=af.FP32)
    xd = cfg0["xd"][:, 5000:5000 + n].contiguous()
    psd = ctx.psd_welch(cfg0["xd"])
    white = ctx.whiten(xd, psd).cpu().numpy().astype(np.float64)
    assert white.shape == (2, n - 2048)
    for c in range(2):
        h = owh.design_filter(opsd.welch(cfg0["x64"][c]))
        y = owh.whiten_fir_direct(cfg0["x64"][c, 5000:5000 + n], h)              # the O(N L) definition
        assert np.abs(white[c] - y).max() <= 1e-4 * np.sqrt(np.mean(y ** 2))


def test_whitening_bf16_output_and_degenerate_lengths(af, cfg0):
    ctx = af.Context(precision=af.FP32)
    psd = ctx.psd_welch(cfg0["xd"])
    w32 = ctx.whiten(cfg0["xd"][:, :20000].contiguous(), psd)
    w16 = ctx.whiten(cfg0["xd"][:, :20000].contiguous(), psd, out_dtype=torch.bfloat16)
    assert torch.equal(w16, w32.to(torch.bfloat16))                              # one RNE rounding, nothing else
    assert ctx.whiten(cfg0["xd"][:, :2048].contiguous(), psd).shape == (2, 0)    # nothing survives the crop
    assert ctx.whiten(cfg0["xd"][:, :2049].contiguous(), psd).shape == (2, 1)


def test_status_codes(af, cfg0):
    ctx = af.Context(precision=af.FP32)
    with pytest.raises(af.AframeError) as e:
        ctx.psd_welch(cfg0["xd"][:, :4095].contiguous())
    assert e.value.status == af.ESHAPE
    with pytest.raises(af.AframeError) as e:
        ctx.load_weights(b"\0" * 64)
    assert e.value.status == af.EINVAL


def test_rolling_whitening_matches_oracle_across_epochs(af):
    # 64 s warm-up + 3 PSD epochs (+ ragged tail that is not a multiple of the stride)
    n = 131072 + 3 * 16384 + 5000 + 77
    x = coloured_noise(n, seed=1002)
    ctx = af.Context(precision=af.FP32)
    white = ctx.whiten_rolling(torch.from_numpy(x).cuda()).cpu().numpy().astype(np.float64)
    cfg = ost.StreamConfig()
    m0 = ost.first_whitened_index(cfg)
    n_eff = (n // 128) * 128
    assert white.shape == (2, n_eff - 1024 - m0)
    x64 = x.astype(np.float64)
    # oracle on sampled stretches: start, both sides of each epoch switch, ragged end
    spots = [m0, m0 + 16384 - 300, m0 + 2 * 16384 - 300, m0 + 3 * 16384 - 300, n_eff - 1024 - 600]
    for c in range(2):
        for a in spots:
            y, _ = ost.whiten_rolling(x64[c], cfg, m_lo=a, m_hi=a + 600)
            got = white[c, a - m0: a - m0 + 600]
            assert np.abs(got - y).max() <= 1e-4, (c, a, np.abs(got - y).max())   # rms(y) ~ 0.98


def test_rolling_whitening_shorter_than_warmup_writes_nothing(af):
    x = coloured_noise(100000, seed=3)
    ctx = af.Context(precision=af.FP32)
    assert ctx.whiten_rolling(torch.from_numpy(x).cuda()).shape == (2, 0)


@pytest.mark.parametrize("batch", [1, 2, 7, 600])
def test_batched_rfft_and_irfft_of_the_overlap_save_block(af, batch):
    """aframe_rfft8192 / aframe_irfft8192 (the two halves of the whitening kernel without the spectral multiply) against
    the oracle's radix-2 FFT (itself pinned to the naive DFT): one-sided spectrum incl. DC, Nyquist and the self-mirrored
    bin 2048; the inverse on a spectrum with non-zero imaginary parts at DC / Nyquist (ignored); round trip."""
    from oracle import fft as offt
    rng = np.random.default_rng(batch)
    x = rng.standard_normal((batch, 8192)).astype(np.float32)
    x[0, :] += 3.0                                               # a DC term
    ctx = af.Context(precision=af.FP32)
    xd = torch.from_numpy(x).cuda()
    spec = ctx.rfft8192(xd)
    got = spec.cpu().numpy().astype(np.float64)
    got = got[..., 0] + 1j * got[..., 1]
    rows = list(range(min(batch, 3))) + ([batch - 1] if batch > 3 else [])
    ref = offt.rfft(x[rows].astype(np.float64))
    scale = np.sqrt(np.mean(np.abs(ref) ** 2))
    # fp32 transform of 8192 points: 2e-6 of the spectrum's rms, plus one fp32 ulp of the row's LARGEST bin (the DC bin of row
    # 0 is 3 * 8192 = 2.4e4, whose ulp alone is 2e-3, and partial sums of that size pass through the butterflies the Nyquist
    # bin shares with it: measured 1.1e-3 at DC, 8.9e-4 at Nyquist; with one row the rms does not hide it)
    assert (np.abs(got[rows] - ref) <= 2e-6 * scale + 1.2e-7 * np.abs(ref).max(axis=-1, keepdims=True)).all()
    back = ctx.irfft8192(spec).cpu().numpy()
    assert np.abs(back - x).max() <= 2e-6 * np.abs(x).max()
    s = (rng.standard_normal((len(rows), 4097)) + 1j * rng.standard_normal((len(rows), 4097)))
    sd = torch.from_numpy(np.stack([s.real, s.imag], axis=-1).astype(np.float32)).cuda().contiguous()
    y = ctx.irfft8192(sd).cpu().numpy().astype(np.float64)
    s32 = sd.cpu().numpy().astype(np.float64)
    yref = offt.irfft(s32[..., 0] + 1j * s32[..., 1], 8192)
    assert np.abs(y - yref).max() <= 2e-6 * np.sqrt(np.mean(yref ** 2)) * 10
