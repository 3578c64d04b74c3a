"""GPU parity (through the C ABI) of the NEXT-3/NEXT-4 rows against the float64 oracle: median-averaged Welch,
the training-time whitening batch and FAR bookkeeping."""
import numpy as np
import pytest
import torch

from oracle import background as obg
from oracle import psd as opsd
from synthdata import coloured_noise

pytestmark = pytest.mark.gpu
SCALE2 = 2.0 ** 140


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


@pytest.mark.parametrize("seconds", [8, 9, 64])                 # 7, 8 (even: two middle values), 63 segments
def test_median_welch_matches_oracle(af, seconds):
    x = coloured_noise(seconds * 2048, 77)
    x[0, 5000] += 3e-19                                          # a glitch the median should shrug off
    ctx = af.Context(precision=af.FP32, welch_average=1)
    p = ctx.psd_welch(torch.from_numpy(x).cuda()).cpu().numpy().astype(np.float64) / SCALE2
    ref = np.stack([opsd.welch(x[c].astype(np.float64), average="median") for c in range(2)])
    band = slice(40, 2001)
    rel = np.abs(p[:, band] - ref[:, band]) / ref[:, band]
    assert rel.max() <= 1e-4, rel.max()
    mean = np.stack([opsd.welch(x[c].astype(np.float64)) for c in range(2)])
    assert np.abs(p[:, band] / mean[:, band] - 1.0).max() > 1e-2  # and it is not the mean


def test_median_welch_rejects_too_many_segments(af):
    ctx = af.Context(precision=af.FP32, welch_average=1)
    x = torch.zeros((2, 300 * 2048), device="cuda")
    with pytest.raises(af.AframeError) as e:
        ctx.psd_welch(x)
    assert e.value.status == af.EUNSUPPORTED
    with pytest.raises(af.AframeError):
        af.Context(welch_average=2)


@pytest.mark.parametrize("batch", [1, 5, 384])                   # 384: the paper's training batch
def test_training_whitening_batch_matches_oracle(af, batch):
    n = 21504                                                    # 10.5 s: 8 s PSD + 2.5 s whitened -> 1.5 s kept
    x = np.stack([coloured_noise(n, 300 + b) for b in range(min(batch, 6))])
    if batch > 6:
        x = np.concatenate([x] * (batch // 6))[:batch]
        x = x * (1.0 + np.arange(batch, dtype=np.float32)[:, None, None] % 7)   # own PSD per row: scale drops out
    ctx = af.Context(precision=af.FP32)
    y = ctx.whiten_batch(torch.from_numpy(np.ascontiguousarray(x)).cuda(), 16384)
    assert y.shape == (batch, 2, 3072)
    y = y.cpu().numpy().astype(np.float64)
    picks = sorted({0, batch // 2, batch - 1})
    ref = obg.whiten_training_batch(x[picks].astype(np.float64), 16384)
    for k, b in enumerate(picks):
        for c in range(2):
            rms = np.sqrt(np.mean(ref[k, c] ** 2))
            assert np.abs(y[b, c] - ref[k, c]).max() <= 1e-4 * rms       # rule T1
    if batch > 6:                                                # rows that differ only by scale whiten alike
        assert np.abs(y[6] - y[0]).max() <= 1e-4 * np.sqrt(np.mean(y[0] ** 2))
    yb = ctx.whiten_batch(torch.from_numpy(np.ascontiguousarray(x)).cuda(), 16384, out_dtype=torch.bfloat16)
    assert np.abs(yb.float().cpu().numpy() - y).max() <= 2.0 ** -8 * np.abs(y).max()      # one bf16 rounding


def test_training_whitening_batch_rejects_bad_shapes(af):
    ctx = af.Context(precision=af.FP32)
    x = torch.zeros((2, 2, 21504), device="cuda")
    for n_psd in (2048, 21504 - 2048):
        with pytest.raises(af.AframeError) as e:
            ctx.whiten_batch(x, n_psd)
        assert e.value.status == af.ESHAPE


@pytest.mark.parametrize("n_bg,n_ev", [(0, 5), (1, 1), (5000, 333), (100_003, 2049), (3_000_000, 1)])
def test_far_counts_bit_exact(af, n_bg, n_ev):
    rng = np.random.default_rng(n_bg + n_ev)
    bg = rng.gumbel(size=n_bg).astype(np.float32)
    ev = rng.gumbel(size=n_ev).astype(np.float32)
    if n_bg > 10 and n_ev > 10:
        bg[::5] = bg[1]                                          # ties: "greater than" is strict
        ev[:4] = [bg[1], np.inf, -np.inf, np.nan]
    ctx = af.Context(precision=af.FP32)
    counts, far = ctx.far(torch.from_numpy(bg).cuda(), torch.from_numpy(ev).cuda(), 86400.0 * 365)
    if n_bg * n_ev <= 2_000_000:
        ref = obg.far_counts(bg, ev)
    else:                                                        # the oracle's double loop on a sample of the events
        idx = np.unique(np.concatenate([np.arange(min(n_ev, 8)), rng.integers(0, n_ev, 24)]))
        ref = np.full(n_ev, -1, dtype=np.int64)
        ref[idx] = [int(np.count_nonzero(bg > ev[i])) for i in idx]
        assert np.array_equal(obg.far_counts(bg[:2000], ev[idx[:3]]), [np.count_nonzero(bg[:2000] > ev[i]) for i in idx[:3]])
    got = counts.cpu().numpy()
    sel = ref >= 0
    assert np.array_equal(got[sel], ref[sel])
    assert np.array_equal(far.cpu().numpy()[sel], ref[sel].astype(np.float64) / np.float64(86400.0 * 365))


def test_far_rejects_bad_livetime(af):
    ctx = af.Context(precision=af.FP32)
    z = torch.zeros(4, device="cuda")
    with pytest.raises(af.AframeError) as e:
        ctx.far(z, z, 0.0)
    assert e.value.status == af.EINVAL
