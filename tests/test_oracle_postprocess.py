"""Pins for oracle/postprocess.py (NEXT-1): closed forms, a library routine and brute force."""
import numpy as np
import scipy.signal

from oracle import postprocess as opp


def test_tophat_of_a_constant_is_the_constant():
    np.testing.assert_allclose(opp.integrate_tophat(np.full(50, 3.25), 16), 3.25, rtol=0, atol=1e-15)


def test_tophat_of_an_impulse_is_a_box_of_height_one_over_n():
    s = np.zeros(64); s[20] = 1.0
    out = opp.integrate_tophat(s, 16)
    expect = np.zeros(64); expect[20:36] = 1.0 / 16
    np.testing.assert_allclose(out, expect, atol=1e-15)
    assert abs(out.sum() - 1.0) < 1e-12                       # unit DC gain away from the start


def test_tophat_equals_library_fir_filter_after_the_ramp():
    rng = np.random.default_rng(0)
    s = rng.standard_normal(300)
    ref = scipy.signal.lfilter(np.full(16, 1 / 16), [1.0], s)   # causal moving average, zero initial state
    np.testing.assert_allclose(opp.integrate_tophat(s, 16)[15:], ref[15:], atol=1e-13)
    # ramp-in: mean of what exists
    assert abs(opp.integrate_tophat(s, 16)[4] - s[:5].mean()) < 1e-14


def test_cluster_max_brute_force_ties_and_partial_window():
    x = np.array([0., 5., 5., 1.,   2., 2., 9., 9.,   7.])
    idx, val = opp.cluster_max(x, 4)
    np.testing.assert_array_equal(idx, [1, 6, 8])            # first maximum wins; trailing partial window counted
    np.testing.assert_array_equal(val, [5., 9., 7.])
    rng = np.random.default_rng(1)
    y = rng.standard_normal(128 * 5)
    idx, val = opp.cluster_max(y, 128)
    np.testing.assert_array_equal(idx, y.reshape(5, 128).argmax(axis=1) + 128 * np.arange(5))
    np.testing.assert_array_equal(val, y.reshape(5, 128).max(axis=1))


def test_float32_variant_is_what_the_kernel_computes():
    rng = np.random.default_rng(2)
    s = rng.standard_normal(100).astype(np.float32)
    a = opp.integrate_tophat(s, 16, dtype=np.float32)
    assert a.dtype == np.float32
    np.testing.assert_allclose(a, opp.integrate_tophat(s.astype(np.float64), 16), rtol=2e-6, atol=2e-7)


def test_cluster_max_propagates_nan_as_its_first_occurrence():
    """Hand example: a window holding NaNs yields the first NaN; windows without are unaffected."""
    x = np.array([1.0, np.nan, 5.0, np.nan, 2.0, 7.0, 3.0, 0.0])
    idx, val = opp.cluster_max(x, 4)
    assert list(idx) == [1, 5] and np.isnan(val[0]) and val[1] == 7.0
