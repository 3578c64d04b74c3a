"""BASELINE.json configs[2] as it is written: one hour of two-detector coloured noise with 200 Newtonian chirps, PSD
re-estimated every 8 s from the trailing 64 s, 1.5 s windows at stride 128, config-1 network on the tensor-core path.

(a) batched: the whole hour through aframe_score_timeslides (zero lag: one "slide" with shift 0), 4096 windows per launch
    sequence -- the shared-stage path, with chirp-bearing windows;
(b) streamed: the first ~3000 updates through aframe_stream_step (64 s of warm-up, then > 2000 scored updates that cross
    15 PSD updates and 6 chirps), compared with (a) window by window;
(c) the float64 oracle on SURVEY 8(d)'s subsample: every 64th window + the 48 windows around 10 chirps + the 32 windows
    around 5 PSD updates (rules T3 and T4 over the whole subsample).
P:170-172 (snapshotter -> whitener -> network), P:108 / P:145 (signals sit 0.25-1.25 s into the window)."""
import numpy as np
import pytest
import scipy.stats
import torch

from oracle import network as onet
from oracle import stream as ost
from synthdata import full_config, make_weight_blob
from synthdata.configs import config2_strain

pytestmark = pytest.mark.gpu
FS, S, K = 2048, 128, 3072


def rel_err(g, o):
    g, o = np.asarray(g, np.float64), np.asarray(o, np.float64)
    return float(np.max(np.abs(g - o) / np.maximum(np.abs(o), 1e-3 * np.abs(o).max())))


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


def subsample(n_win, params, cfg, m0):
    """every 64th window, 48 windows around each of 10 chirps (24 of them hold the coalescence
    time), 32 windows around each of 5 PSD-epoch switches (8 before, 24 after)."""
    picks = set(range(0, n_win, 64))
    for p in params[:: len(params) // 10][:10]:
        i_c = (int(round(p.t_c * FS)) - m0) // S               # last window that still holds t_c ... 23 windows earlier
        picks.update(range(i_c - 35, i_c + 13))
    for e in (1, 2, 57, 230, 431):
        m_switch = cfg.psd_len + e * cfg.psd_update - S - cfg.filter_len // 2
        i = (m_switch - m0) // S
        picks.update(range(i - 8, i + 24))
    return np.array(sorted(i for i in picks if 0 <= i < n_win), dtype=np.int64)


def test_config2_hour_batched_streamed_and_oracle_subsample(af):
    x, params = config2_strain()
    assert x.shape == (2, 3600 * FS) and len(params) == 200
    cfg = ost.StreamConfig()
    m0 = ost.first_whitened_index(cfg)
    n_white = x.shape[1] - m0 - cfg.filter_len // 2
    n_win = (n_white - K) // S + 1
    assert n_win == 56554
    blob = make_weight_blob(**full_config())
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ctx = af.Context(precision=af.F16, stream=stream)
        w = ctx.load_weights(blob)
        # (a) the hour in one call
        batched = ctx.score_timeslides(w, torch.from_numpy(x).cuda(), 0, n_win, [0], batch=4096)
        stream.synchronize()
        batched = batched[0].cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(batched))
        # (b) the first updates one by one: update u scores window u - 1046 (first PSD at update 1023, window full 23 later)
        n_updates = 1046 + 2050
        st = ctx.stream_create(w)
        upd = torch.from_numpy(np.ascontiguousarray(x[:, : n_updates * S].reshape(2, n_updates, S).transpose(1, 0, 2))).cuda()
        buf = torch.empty((2, S), dtype=torch.float32, device="cuda")
        out = torch.zeros((n_updates, 2), dtype=torch.float32, device="cuda")
        for u in range(n_updates):
            buf.copy_(upd[u], non_blocking=True)
            st.step(buf)
            out[u, 0].copy_(st.score[0], non_blocking=True)
            out[u, 1].copy_(st.n_scores[0], non_blocking=True)
        stream.synchronize()
        assert st.uses_graph
        st.close()
    out = out.cpu().numpy()
    assert np.all(out[:1046, 1] == 0) and np.all(out[1046:, 1] == 1)
    streamed = out[1046:, 0].astype(np.float64)
    n_s = len(streamed)
    t_last = (m0 + (n_s - 1) * S + K) / FS
    assert n_s == 2050 and sum(1 for p in params if p.t_c < t_last - 0.25) >= 6
    assert (n_updates * S - cfg.psd_len) // cfg.psd_update >= 15
    # Stream and batch whiten every sample with the same filter (reading C2) but not with the same arithmetic -- 2047-tap
    # direct sums in fp32 kept as fp32, against fp32 FFT overlap-save stored as fp16 -- so their scores agree to the size
    # of that fp16 rounding of the network input (measured 3e-4), not bit for bit.
    assert rel_err(streamed, batched[:n_s]) <= 1.5e-3

    # (c) oracle on the subsample
    picks = subsample(n_win, params, cfg, m0)
    assert 1400 <= len(picks) <= 1600
    x64 = x.astype(np.float64)
    filters = [{}, {}]
    wins = np.empty((len(picks), 2, K))
    for j, i in enumerate(picks):
        a = m0 + int(i) * S
        for c in range(2):
            wins[j, c], _ = ost.whiten_rolling(x64[c], cfg, m_lo=a, m_hi=a + K, filters=filters[c])
    want = onet.forward(onet.parse_blob(blob), wins)
    got = batched[picks]
    err, rho = rel_err(got, want), scipy.stats.spearmanr(got, want).statistic
    in_stream = picks < n_s
    err_s = rel_err(streamed[picks[in_stream]], want[in_stream])
    print(f"configs[2]: {len(picks)} oracle windows; batched rel err {err:.3e}, spearman {rho:.5f}; "
          f"streamed ({int(in_stream.sum())} of them) rel err {err_s:.3e}")
    assert err <= 2e-2 and err_s <= 2e-2                         # T3
    assert rho >= 0.999                                          # T4 over the subsample (chirps included)
