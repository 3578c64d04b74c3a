"""Pins for oracle/network.py (O-5; readings B1-B8)."""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle import network as onet
from synthdata import weights as sw

RNG = np.random.default_rng(17)


@pytest.mark.parametrize("c_in,c_out,k,stride,pad,t", [
    (2, 3, 7, 2, 3, 19), (3, 4, 3, 1, 1, 11), (3, 4, 3, 2, 1, 12), (4, 2, 1, 2, 0, 9), (1, 1, 3, 2, 1, 7)])
def test_conv_matmul_form_equals_brute_force_definition(c_in, c_out, k, stride, pad, t):
    x = RNG.standard_normal((2, c_in, t))
    w = RNG.standard_normal((c_out, c_in, k))
    fast = onet.conv1d(x, w, stride, pad)
    for b in range(2):
        np.testing.assert_allclose(fast[b], onet.conv1d_direct(x[b], w, stride, pad), atol=1e-13)


def test_conv_asymmetric_kernel_orientation():
    # cross-correlation orientation: a single tap at d=0 reads in[t*stride - pad]
    x = np.arange(10.0)[None, None, :]
    w = np.zeros((1, 1, 3)); w[0, 0, 0] = 1.0
    y = onet.conv1d(x, w, 1, 1)[0, 0]
    np.testing.assert_array_equal(y, np.concatenate([[0.0], np.arange(9.0)]))


@pytest.mark.parametrize("k,stride,pad,t", [(7, 2, 3, 64), (3, 1, 1, 33), (3, 2, 1, 32), (1, 2, 0, 31)])
def test_conv_equals_torch_library(k, stride, pad, t):
    x = RNG.standard_normal((3, 5, t)); w = RNG.standard_normal((6, 5, k))
    ref = F.conv1d(torch.from_numpy(x), torch.from_numpy(w), stride=stride, padding=pad).numpy()
    np.testing.assert_allclose(onet.conv1d(x, w, stride, pad), ref, atol=1e-12)


def test_maxpool_equals_torch_library_and_padding_never_wins():
    x = RNG.standard_normal((2, 3, 17)) - 5.0        # all negative: zero padding would win if used
    ref = F.max_pool1d(torch.from_numpy(x), 3, 2, 1).numpy()
    np.testing.assert_array_equal(onet.maxpool1d(x, 3, 2, 1), ref)


def _net(cfg):
    return onet.parse_blob(sw.make_weight_blob(**cfg))


def test_fold_is_identity_tiny_and_full_shapes():
    tiny = _net(sw.tiny_config())
    x = RNG.standard_normal((2, 2, 256))
    np.testing.assert_allclose(onet.forward(tiny, x, folded=True), onet.forward(tiny, x, folded=False), rtol=1e-12)
    # group statistics (config-1 style) on a narrow net so it runs fast
    cfg = dict(table=sw.resnet_layer_table(2, 16, 7, [1, 1], [16, 32]), norm_kind=sw.NORM_GROUP, n_groups=8, seed=3)
    net = _net(cfg)
    np.testing.assert_allclose(onet.forward(net, x, folded=True), onet.forward(net, x, folded=False), rtol=1e-12)


def test_per_channel_norm_equals_torch_batchnorm_eval():
    net = _net(sw.tiny_config())
    l = net["layers"][0]
    x = RNG.standard_normal((2, 2, 64))
    z = F.conv1d(torch.from_numpy(x), torch.from_numpy(l["W"].copy()), stride=l["stride"], padding=l["pad"])
    ref = F.batch_norm(z, torch.from_numpy(l["mean"].copy()), torch.from_numpy(l["var"].copy()),
                       torch.from_numpy(l["gamma"].copy()), torch.from_numpy(l["beta"].copy()),
                       training=False, eps=net["eps"]).numpy()
    w, b = onet.fold_norm(l, net["norm_kind"], net["n_groups"], net["eps"])
    np.testing.assert_allclose(onet.conv1d(x, w, l["stride"], l["pad"]) + b[None, :, None], ref, atol=1e-12)


def test_group_statistics_index():
    np.testing.assert_array_equal(onet.stat_index(64, 1, 8), np.repeat(np.arange(8), 8))
    np.testing.assert_array_equal(onet.stat_index(8, 0, 0), np.arange(8))


def _torch_forward(net, x):
    """Independent re-assembly of the network from torch library ops (conv1d, max_pool1d)."""
    outs, x0 = [], torch.from_numpy(x)
    for l in net["layers"]:
        src = x0 if l["input_from"] < 0 else outs[l["input_from"]]
        if l["kind"] == 0:
            g = onet.stat_index(l["c_out"], net["norm_kind"], net["n_groups"])
            z = F.conv1d(src, torch.from_numpy(l["W"].copy()), stride=l["stride"], padding=l["pad"])
            y = F.batch_norm(z, torch.from_numpy(l["mean"][g].copy()), torch.from_numpy(l["var"][g].copy()),
                             torch.from_numpy(l["gamma"].copy()), torch.from_numpy(l["beta"].copy()),
                             training=False, eps=net["eps"])
            if l["residual_from"] >= 0:
                y = y + outs[l["residual_from"]]
            if l["relu"]:
                y = F.relu(y)
        elif l["kind"] == 1:
            y = F.max_pool1d(src, l["k"], l["stride"], l["pad"])
        else:
            y = F.adaptive_avg_pool1d(src, 1)[:, :, 0] @ torch.from_numpy(l["w"].copy()) + l["b"]
        outs.append(y)
    return outs[-1].numpy()


def test_forward_equals_torch_library_assembly_tiny():
    net = _net(sw.tiny_config())
    x = RNG.standard_normal((3, 2, 2048))
    np.testing.assert_allclose(onet.forward(net, x), _torch_forward(net, x), rtol=1e-10)


def test_full_network_shape_closed_forms():
    cfg = sw.full_config()
    net = _net(cfg)
    convs = [l for l in net["layers"] if l["kind"] == 0]
    assert len(convs) == 36                                        # 1 stem + 32 + 3 shortcuts (B1)
    n_params = sum(l["W"].size + l["c_out"] for l in convs) + 512 + 1
    assert n_params == 7_210_689
    lens = onet.output_length(net, 3072)
    assert lens[0] == 1536 and lens[1] == 768 and lens[-2] == 96   # B2: 3072 -> 1536 -> 768 ... -> 96
    macs = sum(l["W"].size * lens[i] for i, l in enumerate(net["layers"]) if l["kind"] == 0) + 512
    assert abs(macs / 1e6 - 1070.92) < 0.01
    tiny = _net(sw.tiny_config())
    tl = onet.output_length(tiny, 2048)
    assert tl[0] == 1024 and tl[1] == 512 and tl[-2] == 64
    tconvs = [l for l in tiny["layers"] if l["kind"] == 0]
    assert sum(l["W"].size + l["c_out"] for l in tconvs) + 64 + 1 == 27_801


def test_he_normal_variance_and_head():
    net = _net(sw.full_config())
    l = [l for l in net["layers"] if l["kind"] == 0 and l["c_in"] == 256 and l["k"] == 3][0]
    np.testing.assert_allclose(l["W"].var(), 2.0 / (256 * 3), rtol=0.02)
    head = net["layers"][-1]
    np.testing.assert_allclose(head["w"].var(), 1.0 / 512, rtol=0.2)
    assert head["b"] == 0.0


def test_residual_is_added_before_relu():
    # hand-built 2-layer net: y = relu(conv_b(relu(conv_a(x))) + x); identity-free closed form on 1 channel
    table = [sw.LayerSpec(0, 1, 1, 1, 1, 0, 1, -1, -1), sw.LayerSpec(0, 1, 1, 1, 1, 0, 1, 0, 0),
             sw.LayerSpec(2, 1, 1, 1, 1, 0, 0, 1, -1)]
    net = onet.parse_blob(sw.make_weight_blob(table, 0, 0, seed=5, in_channels=1))
    for l in net["layers"][:2]:
        l["W"][:] = -1.0; l["gamma"][:] = 1.0; l["beta"][:] = 0.0; l["mean"][:] = 0.0; l["var"][:] = 1.0 - net["eps"]
    net["layers"][2]["w"][:] = 1.0
    x = np.array([[[-2.0, 3.0]]])
    # conv_a: -x = [2,-3] -> relu [2,0]; conv_b: -[2,0] = [-2,0]; + residual [2,0] -> [0,0]; mean 0
    # if the residual were added after the ReLU the result would be mean([2,0]) = 1
    np.testing.assert_allclose(onet.forward(net, x), [0.0], atol=1e-12)


def test_round_bf16_matches_torch():
    x = RNG.standard_normal(1000) * 10
    ref = torch.from_numpy(x).float().bfloat16().double().numpy()
    np.testing.assert_array_equal(onet.round_bf16(x), ref)


def test_round_f16_matches_torch_spacing_and_saturation():
    """Pins of round_f16 (activation storage of the tensor-core path, reading B10): the library conversion, the format's
    spacing (2^-10 relative in the normal range, 2^-24 absolute below 2^-14: hand values), saturation at +-65504."""
    x = np.concatenate([RNG.standard_normal(1000) * 10, RNG.standard_normal(200) * 1e-6, RNG.standard_normal(200) * 3e3])
    ref = torch.from_numpy(x).float().half().double().numpy()
    np.testing.assert_array_equal(onet.round_f16(x), ref)
    np.testing.assert_array_equal(onet.round_f16([1.0 + 2.0 ** -11, 1.0 + 3 * 2.0 ** -11, 2048.0 + 1.0, 2.0 ** -25 * 1.5]),
                                  [1.0, 1.0 + 2.0 ** -9, 2048.0, 2.0 ** -24])        # ties to even; subnormal spacing
    np.testing.assert_array_equal(onet.round_f16([1e5, -7e4, 65504.0, 65519.9]), [65504.0, -65504.0, 65504.0, 65504.0])
    assert np.isnan(onet.round_f16([np.nan]))[0]
    # eight times finer than bf16 in the normal range
    v = np.linspace(1.0, 2.0, 4097)[:-1]
    assert np.abs(onet.round_f16(v) - v).max() == 2.0 ** -11 and np.abs(onet.round_bf16(v) - v).max() == 2.0 ** -8


def test_live_group_norm_matches_library_and_is_scale_invariant():
    """NEXT-2 pin: oracle.group_norm_live = torch.nn.functional.group_norm (library routine); the normalised output does
    not change when the window's pre-norm tensor is rescaled (eps -> 0)."""
    import torch
    from oracle import network as onet
    rng = np.random.default_rng(5)
    z = rng.standard_normal((3, 16, 40))
    gamma, beta = rng.standard_normal(16), rng.standard_normal(16)
    got = onet.group_norm_live(z, gamma, beta, 8, 1e-5)
    ref = torch.nn.functional.group_norm(torch.from_numpy(z), 8, torch.from_numpy(gamma), torch.from_numpy(beta), 1e-5).numpy()
    np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(onet.group_norm_live(z * 37.0, gamma, beta, 8, 0.0), onet.group_norm_live(z, gamma, beta, 8, 0.0),
                               rtol=1e-10, atol=1e-10)


def test_live_group_norm_network_runs_and_differs_from_folded():
    from oracle import network as onet
    from synthdata import make_weight_blob, tiny_config_live_gn
    cfg = tiny_config_live_gn()
    net = onet.parse_blob(make_weight_blob(**cfg))
    assert net["norm_kind"] == 2 and net["layers"][0]["mean"].size == 0
    rng = np.random.default_rng(6)
    x = rng.standard_normal((2, 2, 2048))
    s = onet.forward(net, x)
    assert s.shape == (2,) and np.all(np.isfinite(s))
    # per-window statistics: scaling one window's input leaves its score (almost) unchanged, unlike a frozen norm
    s2 = onet.forward(net, x * np.array([1.0, 8.0])[:, None, None])
    assert abs(s2[1] - s[1]) < 1e-3 * max(1.0, abs(s[1])) and s2[0] == s[0]


def test_overlapping_windows_share_every_row_out_of_reach_of_their_padding():
    """The identity the CUDA path's shared stages rest on, checked on the float64 oracle alone: two
    windows cut 128 samples apart from one stream have identical activations, layer by layer, except in the rows within
    reach of each window's own zero padding.  The reach follows from the conv definition (O-5): stem + pool leave rows
    {0, 1} / {T - 1}; a k3 s1 conv adds one row per side; a k3 s2 conv maps e -> e // 2 + 1 and f -> T_out - (T_in - f - 1 + 1) // 2;
    a k1 s2 conv e -> ceil(e / 2); a residual takes the larger reach.  Stage ends: 8/7, 12/11, 18/17, 15/14 rows."""
    from synthdata import make_weight_blob, full_config
    net = onet.parse_blob(make_weight_blob(**full_config()))
    rng = np.random.default_rng(5)
    stream = rng.standard_normal((2, 3072 + 128))
    wins = np.stack([stream[:, :3072], stream[:, 128:128 + 3072]])
    _, outs = onet.forward(net, wins, keep=True)
    lens = onet.output_length(net, 3072)
    reach = {}                                     # layer -> (rows at the start, rows at the end) that see the padding
    stage_end = {}
    for i, l in enumerate(net["layers"]):
        if l["kind"] == onet.KIND_HEAD:
            break
        t_out = lens[i]
        if l["input_from"] < 0:                    # stem conv k7 s2 p3: rows 0, 1 / the last row see the padding
            e, f = 2, 1
        else:
            ei, fi = reach[l["input_from"]]
            t_in = lens[l["input_from"]]
            k, s, p = l["k"], l["stride"], l["pad"]
            # output row t reads input rows s t - p ... s t - p + k - 1
            e = max([t + 1 for t in range(t_out) if s * t - p < ei] + [0])
            f = max([t_out - t for t in range(t_out) if s * t - p + k - 1 >= t_in - fi] + [0])
            if l["kind"] == onet.KIND_CONV and l["residual_from"] >= 0:
                er, fr = reach[l["residual_from"]]
                e, f = max(e, er), max(f, fr)
        reach[i] = (e, f)
        stage_end[l["c_out"] if l["kind"] == onet.KIND_CONV else 64] = (e, f)
        shift = 128 * t_out // 3072                # rows between the two windows at this resolution
        if i == 0 or (128 * t_out) % 3072:
            continue
        a = outs[i][0][:, shift + e: t_out - f]    # window 0, the rows that are window 1's rows e ... t_out - shift - f
        b = outs[i][1][:, e: t_out - shift - f]
        scale = np.abs(outs[i]).max()
        assert np.abs(a - b).max() <= 1e-10 * scale, (i, e, f)
        # the bound is tight: the last row inside the reach does differ (checked where the padding's influence, which decays
        # with every layer, is still far above rounding: the 64- and 128-channel stages)
        if e > 0 and l["kind"] == onet.KIND_CONV and l["c_out"] <= 128:
            assert np.abs(outs[i][0][:, shift + e - 1] - outs[i][1][:, e - 1]).max() > 1e-9 * scale, (i, e)
    assert stage_end[64] == (8, 7) and stage_end[128] == (12, 11) and stage_end[256] == (18, 17) and stage_end[512] == (15, 14)
