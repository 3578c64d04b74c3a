"""aframe_psd_welch_static: the Welch PSD (O-1) with its periodogram scratch in a fixed file-scope device array, for callers
that may not allocate device memory (CUDA-graph capture, serving loops).  Checked against aframe_psd_welch -- the existing,
allocating path, itself checked against the oracle in tests/test_gpu_signal.py -- on two calls in a row that share the
array (the second shorter than the first, so a stale periodogram read by mistake would show), plus the size limit.
This file sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide the parity tests."""
import numpy as np
import pytest
import torch

from synthdata import coloured_noise

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


def test_static_scratch_psd_equals_the_allocating_path_on_two_calls_in_a_row(af):
    ctx = af.Context(precision=af.FP32)
    assert int(ctx.lib.aframe_psd_welch_static_max_floats()) == 2 * 64 * 2049
    x1 = torch.from_numpy(coloured_noise(64 * 2048, seed=11)).cuda()            # 63 segments: the 64 s PSD of P:172
    x2 = torch.from_numpy(coloured_noise(8 * 2048 + 517, seed=12)).cuda()       # 7 segments and a ragged tail (P:102's 8 s)
    out1 = torch.empty((2, ctx.n_freq), dtype=torch.float32, device="cuda")
    out2 = torch.empty_like(out1)
    ctx.psd_welch_static(x2, out2)                                              # (first use loads the kernels' module)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]                                  # the driver's count: sees any cudaMalloc
    launches = ctx.launch_count()
    ctx.psd_welch_static(x1, out1)                                              # two calls in a row on the shared array
    ctx.psd_welch_static(x2, out2)
    torch.cuda.synchronize()
    assert ctx.launch_count() - launches == 4 and torch.cuda.mem_get_info()[0] == free_before
    for x, got in ((x1, out1), (x2, out2)):
        want = ctx.psd_welch(x).cpu().numpy().astype(np.float64)
        got = got.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(got)) and want.max() > 0
        # tolerance of the PSD parity tests (1e-4 relative, tests/test_gpu_signal.py); the kernels are the same, so it is met exactly
        assert np.abs(got - want).max() <= 1e-4 * np.abs(want).max()
        np.testing.assert_array_equal(got, want)
    # again after the allocating path has run, from a second context (the array belongs to the device, not to a context)
    ctx2 = af.Context(precision=af.FP32, welch_average=1)
    out3 = torch.empty_like(out1)
    ctx2.psd_welch_static(x2, out3)
    np.testing.assert_array_equal(out3.cpu().numpy(), ctx2.psd_welch(x2).cpu().numpy())


def test_static_scratch_psd_rejects_sizes_beyond_its_array(af):
    ctx = af.Context(precision=af.FP32)
    out = torch.empty((2, ctx.n_freq), dtype=torch.float32, device="cuda")
    x = torch.zeros((2, 66 * 2048), dtype=torch.float32, device="cuda")         # 65 segments: one more than the array holds
    with pytest.raises(af.AframeError) as e:
        ctx.psd_welch_static(x, out)
    assert e.value.status == af.ESHAPE and "exceeds the static scratch" in str(e.value)
    ctx.psd_welch_static(x[:, : 65 * 2048].contiguous(), out)                   # 64 segments: the maximum
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
    with pytest.raises(af.AframeError):
        ctx.psd_welch_static(x[:, :1000].contiguous(), out)                                  # shorter than one segment, as aframe_psd_welch
