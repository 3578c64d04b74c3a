"""GPU parity of NEXT-1 (aframe_postprocess) against the oracle: integrated series bit for bit (same float32 arithmetic
in the same order, reading D3), trigger indices and values exactly; float64 oracle within rounding."""
import numpy as np
import pytest
import torch

from oracle import postprocess as opp

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


@pytest.mark.parametrize("n", [1, 15, 16, 129, 128 * 7 + 53])
def test_postprocess_matches_oracle(af, n):
    rng = np.random.default_rng(n)
    s = rng.standard_normal((3, n)).astype(np.float32)
    s[1, n // 2:] = s[1, n // 2]                                # a run of equal scores: ties in the argmax
    ctx = af.Context(precision=af.F16)
    integ, val, idx = ctx.postprocess(torch.from_numpy(s).cuda(), n_int=16, n_cluster=128)
    integ, val, idx = integ.cpu().numpy(), val.cpu().numpy(), idx.cpu().numpy()
    for k in range(3):
        ref32 = opp.integrate_tophat(s[k], 16, dtype=np.float32)
        np.testing.assert_array_equal(integ[k], ref32)
        ri, rv = opp.cluster_max(ref32, 128)
        np.testing.assert_array_equal(idx[k], ri)
        np.testing.assert_array_equal(val[k], rv)
        ref64 = opp.integrate_tophat(s[k].astype(np.float64), 16)
        np.testing.assert_allclose(integ[k], ref64, rtol=2e-6, atol=2e-7)


def test_postprocess_on_timeslide_scores_and_errors(af):
    ctx = af.Context(precision=af.F16)
    s = torch.randn(8, 4096, device="cuda")
    integ, val, idx = ctx.postprocess(s[:, :4000].contiguous()[:, :4000])
    assert integ.shape == (8, 4000) and val.shape == (8, 32) and idx.dtype == torch.int64
    assert bool((idx >= 0).all()) and bool((idx < 4000).all())
    assert torch.equal(integ.gather(1, idx), val)
    with pytest.raises(af.AframeError) as e:
        ctx.postprocess(s, n_int=0)
    assert e.value.status == af.EINVAL


def test_postprocess_nan_propagates_like_the_oracle(af):
    """A NaN score makes NaN integrated values; a cluster window that holds one yields its FIRST NaN (value and index),
    wherever it sits relative to the warp's lanes -- numpy.argmax's rule in the oracle."""
    rng = np.random.default_rng(99)
    s = rng.standard_normal((2, 128 * 5)).astype(np.float32)
    s[0, 200] = np.nan                                           # integrated values 200..215 are NaN (window 1)
    s[1, 3] = np.nan; s[1, 128 * 3 + 77] = np.nan                # first lane; a middle lane of window 3
    ctx = af.Context(precision=af.F16)
    integ, val, idx = ctx.postprocess(torch.from_numpy(s).cuda(), n_int=16, n_cluster=128)
    integ, val, idx = integ.cpu().numpy(), val.cpu().numpy(), idx.cpu().numpy()
    for k in range(2):
        ref32 = opp.integrate_tophat(s[k], 16, dtype=np.float32)
        np.testing.assert_array_equal(integ[k], ref32)           # (assert_array_equal treats NaNs in the same place as equal)
        ri, rv = opp.cluster_max(ref32, 128)
        np.testing.assert_array_equal(idx[k], ri)
        np.testing.assert_array_equal(val[k], rv)
    assert idx[0, 1] == 200 and np.isnan(val[0, 1]) and idx[1, 0] == 3 and idx[1, 3] == 128 * 3 + 77
