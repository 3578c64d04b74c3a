"""The paper's detection-statistic flow end to end on the device: whiten both detectors
once, score the zero-lag stream and 8 timeslides, integrate with the 1 s top hat, cluster over 8 s, and assign each
zero-lag trigger a false-alarm rate from the timeslide background.  The oracle recomputes every stage after the scores
from the SAME float32 scores (readings D1-D3, E1), so triggers, counts and rates must agree exactly; the scores themselves
are checked against the oracle in test_gpu_stream.py / test_gpu_network.py."""
import numpy as np
import pytest
import torch

from oracle import background as obg
from oracle import postprocess as opp
from synthdata import coloured_noise, full_config, make_weight_blob
from synthdata.chirps import draw_chirp_params, inject_chirps

pytestmark = pytest.mark.gpu
FS, S = 2048, 128


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


def test_zero_lag_triggers_get_far_from_timeslide_background(af):
    import bench
    seconds = 512
    n_win, n_raw = bench.block_geometry(seconds)
    noise = coloured_noise(n_raw, seed=4242)
    x, _ = inject_chirps(noise, draw_chirp_params(20, n_raw / FS, seed=7))
    shifts = [0] + [k * FS for k in range(1, 9)]                 # series 0 = zero lag, 1..8 = background
    ctx = af.Context(precision=af.F16)
    w = ctx.load_weights(make_weight_blob(**full_config()))
    scores = ctx.score_timeslides(w, torch.from_numpy(x).cuda(), 0, n_win, shifts, batch=4096)
    assert scores.shape == (9, n_win) and bool(torch.isfinite(scores).all())
    integ, val, idx = ctx.postprocess(scores, n_int=16, n_cluster=128)      # 1 s top hat, 8 s clusters at 16 Hz
    livetime = 8 * n_win * S / FS                                           # seconds of background analysed
    counts, far = ctx.far(val[1:].reshape(-1).contiguous(), val[0].contiguous(), livetime)

    s = scores.cpu().numpy()
    ref_val, ref_idx = [], []
    for k in range(9):
        ri = opp.integrate_tophat(s[k], 16, dtype=np.float32)
        np.testing.assert_array_equal(integ[k].cpu().numpy(), ri)
        i, v = opp.cluster_max(ri, 128)
        ref_idx.append(i); ref_val.append(v)
    ref_val, ref_idx = np.asarray(ref_val), np.asarray(ref_idx)
    np.testing.assert_array_equal(idx.cpu().numpy(), ref_idx)
    np.testing.assert_array_equal(val.cpu().numpy(), ref_val)
    ref_counts = obg.far_counts(ref_val[1:].reshape(-1), ref_val[0])
    np.testing.assert_array_equal(counts.cpu().numpy(), ref_counts)
    np.testing.assert_array_equal(far.cpu().numpy(), obg.far(ref_val[1:].reshape(-1), ref_val[0], livetime))
    n_trig = n_win // 128
    assert val.shape == (9, n_trig) and int(counts.max()) <= 8 * n_trig
    nz = far[far > 0]
    assert nz.numel() == 0 or float(nz.min()) >= 1.0 / livetime             # the resolution of this background
