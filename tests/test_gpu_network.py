"""GPU parity (through the C ABI) of the network forward pass against the float64 oracle.
fp32 path: rule T2 (<= 1e-4); tensor-core path (fp16 weights and activations, fp32 accumulation): rules T3 (<= 2e-2) and T4 (Spearman
>= 0.999), both asserted outright."""
import numpy as np
import pytest
import scipy.stats
import torch

from oracle import network as onet
from oracle import psd as opsd
from oracle import whiten as owh
from synthdata import make_weight_blob, tiny_config, full_config
from synthdata.configs import config0_strain, config1_raw, gather_windows

pytestmark = pytest.mark.gpu


def rel_err(g, o):
    """T2/T3: max_i |g_i - o_i| / max(|o_i|, 1e-3 max_j |o_j|)."""
    g, o = np.asarray(g, np.float64), np.asarray(o, np.float64)
    return float(np.max(np.abs(g - o) / np.maximum(np.abs(o), 1e-3 * np.abs(o).max())))


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


@pytest.fixture(scope="module")
def config0():
    x = config0_strain().astype(np.float64)
    y = np.stack([owh.whiten_fft(x[c], owh.design_filter(opsd.welch(x[c]), n_design=4096)) for c in range(2)])
    tail = y[:, -(63 * 128 + 2048):]                  # reading A7: windows from the last 12 160 raw samples
    wins = np.stack([tail[:, i * 128: i * 128 + 2048] for i in range(64)]).astype(np.float32)
    blob = make_weight_blob(**tiny_config())
    return dict(wins=wins, blob=blob, ref=onet.forward(onet.parse_blob(blob), wins), white_tail=tail.astype(np.float32))


@pytest.fixture(scope="module")
def config1():
    strain, starts, _ = config1_raw(128)
    x = strain.astype(np.float64)
    y = np.stack([owh.whiten_fft(x[c], owh.design_filter(opsd.welch(x[c, : 64 * 2048]))) for c in range(2)])
    wins = gather_windows(y, starts, 3072, offset=1024).astype(np.float32)
    blob = make_weight_blob(**full_config())
    net = onet.parse_blob(blob)
    return dict(wins=wins, blob=blob, net=net, ref=onet.forward(net, wins))


def test_config0_fp32_scores(af, config0):
    ctx = af.Context(n_design=4096, kernel_len=2048, precision=af.FP32)
    w = ctx.load_weights(config0["blob"])
    got = ctx.forward(w, torch.from_numpy(config0["wins"]).cuda()).cpu().numpy()
    assert rel_err(got, config0["ref"]) <= 1e-4


def test_config0_strided_equals_explicit_windows(af, config0):
    ctx = af.Context(n_design=4096, kernel_len=2048, precision=af.FP32)
    w = ctx.load_weights(config0["blob"])
    a = ctx.forward(w, torch.from_numpy(config0["wins"]).cuda())
    b = ctx.forward_strided(w, torch.from_numpy(config0["white_tail"]).cuda().contiguous(), 0, 64)
    assert torch.equal(a, b)                                    # O-4: same samples, same arithmetic
    with pytest.raises(af.AframeError) as e:
        ctx.forward_strided(w, torch.from_numpy(config0["white_tail"]).cuda().contiguous(), 0, 65)
    assert e.value.status == af.ESHAPE


@pytest.mark.parametrize("batch", [1, 5, 128])
def test_config1_fp32_scores(af, config1, batch):
    ctx = af.Context(precision=af.FP32)
    w = ctx.load_weights(config1["blob"])
    got = ctx.forward(w, torch.from_numpy(config1["wins"][:batch]).cuda()).cpu().numpy()
    assert rel_err(got, config1["ref"][:batch]) <= 1e-4            # T2 at every batch size (measured: 2e-7 .. 9e-7)


def test_config1_tensor_core_scores_and_rank(af, config1):
    ctx = af.Context(precision=af.F16)
    w = ctx.load_weights(config1["blob"])
    got = ctx.forward(w, torch.from_numpy(config1["wins"]).cuda()).cpu().numpy().astype(np.float64)
    ref = config1["ref"]
    err = rel_err(got, ref)
    rho = scipy.stats.spearmanr(got, ref).statistic
    # the oracle with the CUDA path's storage roundings (B10): fp16 weights, fp16 after every stored activation
    ideal = onet.forward(config1["net"], config1["wins"], act_round=onet.round_f16, weight_round=onet.round_f16)
    rho_ideal = scipy.stats.spearmanr(ideal, ref).statistic
    err_vs_ideal = rel_err(got, ideal)
    print(f"tensor-core path: rel err {err:.3e}, spearman {rho:.5f}; same roundings in float64 {rho_ideal:.5f}; vs that {err_vs_ideal:.3e}")
    assert err <= 2e-2                                           # T3
    assert err_vs_ideal <= 1e-3                                  # kernels reproduce the rounded-storage arithmetic
    assert rho >= 0.999                                          # T4, outright


@pytest.mark.parametrize("batch", [1, 3, 7])
def test_config1_tensor_core_small_and_ragged_batches(af, config1, batch):
    ctx = af.Context(precision=af.F16)
    w = ctx.load_weights(config1["blob"])
    got = ctx.forward(w, torch.from_numpy(config1["wins"][:batch]).cuda()).cpu().numpy()
    assert rel_err(got, config1["ref"][:batch]) <= 2e-2


def test_tensor_core_path_refuses_tables_it_cannot_run(af, config0):
    ctx = af.Context(n_design=4096, kernel_len=2048, precision=af.F16)
    w = ctx.load_weights(config0["blob"])                        # widths 8..64: not UMMA shapes
    with pytest.raises(af.AframeError) as e:
        ctx.forward(w, torch.from_numpy(config0["wins"]).cuda())
    assert e.value.status == af.EUNSUPPORTED                     # fails loudly, no silent fallback


def test_full_batch_launch_configuration_sampled_against_oracle(af, config1):
    """The launch configuration bench.py times (4096-window chunks, ragged tail, windows taken in place from a bf16
    whitened stream (any of the three stream types may be handed in) at stride 128): sampled scores against the float64 oracle (rule T3), and the big batch against the
    same windows scored in small batches (bit for bit: a window's score does not depend on its batch)."""
    n_win = 4096 + 37
    rng = np.random.default_rng(7)
    white = rng.standard_normal((2, (n_win - 1) * 128 + 3072)).astype(np.float32)
    wd = torch.from_numpy(white).cuda().to(torch.bfloat16).contiguous()
    ctx = af.Context(precision=af.F16)
    w = ctx.load_weights(config1["blob"])
    big = ctx.forward_strided(w, wd, 0, n_win)
    assert big.shape == (n_win,) and bool(torch.isfinite(big).all())
    picks = [0, 1, 2047, 4095, 4096, n_win - 1]
    for i in picks:
        small = ctx.forward_strided(w, wd, i * 128, 1)
        assert torch.equal(small[0], big[i])
    w64 = wd.float().cpu().numpy().astype(np.float64)
    wins = np.stack([w64[:, i * 128: i * 128 + 3072] for i in picks])
    ref = onet.forward(config1["net"], wins)
    assert rel_err(big[picks].cpu().numpy(), ref) <= 2e-2


def test_forward_rejects_bad_arguments(af, config1):
    ctx = af.Context(precision=af.F16)
    w = ctx.load_weights(config1["blob"])
    with pytest.raises(af.AframeError) as e:
        ctx.forward(w, torch.empty((0, 2, 3072), device="cuda"))
    assert e.value.status == af.EINVAL
    other = af.Context(precision=af.F16)
    with pytest.raises(af.AframeError) as e:
        other.forward(w, torch.zeros((1, 2, 3072), device="cuda"))
    assert e.value.status == af.ESTATE


def test_true_group_norm_fp32_matches_oracle(af, config0):
    """NEXT-2: GroupNorm statistics computed per window at inference (blob norm_kind 2) on the fp32 path against
    the oracle (rule T2); the tensor-core path refuses such a table loudly."""
    from synthdata import tiny_config_live_gn
    cfg = tiny_config_live_gn()
    blob = make_weight_blob(**cfg)
    wins = config0["wins"][:16].copy()
    wins[3] *= 5.0                                              # statistics are per window: a rescaled window is fine
    ref = onet.forward(onet.parse_blob(blob), wins)
    ctx = af.Context(n_design=4096, kernel_len=2048, precision=af.FP32)
    w = ctx.load_weights(blob)
    got = ctx.forward(w, torch.from_numpy(wins).cuda()).cpu().numpy()
    assert rel_err(got, ref) <= 1e-4
    ctx16 = af.Context(n_design=4096, kernel_len=2048, precision=af.F16)
    w16 = ctx16.load_weights(blob)
    with pytest.raises(af.AframeError) as e:                    # widths 8..64 do not tile onto the tensor-core kernel
        ctx16.forward(w16, torch.from_numpy(wins).cuda())
    assert e.value.status == af.EUNSUPPORTED


def test_true_group_norm_full_size_fp32_and_tensor_core(af, config1):
    """NEXT-2 at configs[1] size: the ResNet54 table with live GroupNorm.  fp32 path within T2 of the oracle; tensor-core
    path (plain conv output stored as fp16, statistics + affine + residual + ReLU in the GroupNorm kernels) within T3 and
    T4 (Spearman >= 0.999, outright); smaller ragged batches give the same scores bit for bit."""
    from synthdata import full_config_live_gn
    blob = make_weight_blob(**full_config_live_gn())
    wins = config1["wins"][:48].copy()
    wins[5] *= 7.0                                              # per-window statistics: the scale of a window drops out ...
    wins[6] = wins[5] / 7.0                                     # ... up to eps, so these two score (almost) alike
    ref = onet.forward(onet.parse_blob(blob), wins)
    assert abs(ref[5] - ref[6]) <= 1e-3 * np.abs(ref).max()
    x = torch.from_numpy(wins).cuda()
    ctx = af.Context(precision=af.FP32)
    got32 = ctx.forward(ctx.load_weights(blob), x[:8]).cpu().numpy()
    assert rel_err(got32, ref[:8]) <= 1e-4
    ctx16 = af.Context(precision=af.F16)
    w16 = ctx16.load_weights(blob)
    got = ctx16.forward(w16, x).cpu().numpy().astype(np.float64)
    err = rel_err(got, ref)
    rho = scipy.stats.spearmanr(got, ref).statistic
    # the oracle with the CUDA path's storage roundings (fp16 weights, fp16 after every stored tensor), for the record
    net = onet.parse_blob(blob)
    ideal = onet.forward(net, wins, act_round=onet.round_f16, weight_round=onet.round_f16)
    rho_ideal = scipy.stats.spearmanr(ideal, ref).statistic
    print(f"live GroupNorm, tensor-core path: rel err {err:.3e}, spearman {rho:.5f} (same roundings in float64 {rho_ideal:.5f}, "
          f"its rel err {rel_err(ideal, ref):.3e})")
    assert err <= 2e-2                                           # T3 (measured 1.0e-3)
    assert rho >= 0.999                                          # T4, outright (measured 0.99957 on these 48 windows)
    assert rel_err(got, ideal) <= 5e-3
    for nb in (1, 37):
        part = ctx16.forward(w16, x[:nb]).cpu().numpy()
        assert np.array_equal(part, got[:nb].astype(np.float32))


@pytest.mark.parametrize("kernel_len", [2048, 4096, 2560])
def test_tensor_core_path_other_window_lengths(af, kernel_len):
    """The tensor-core path is not specialised to K = 3072: the config-1 table on 1 s, 2 s and 1.25 s windows (stage lengths
    512..64, 1024..128 and 640..80: other tile shapes, windows-per-tile counts and fused-block tile counts)."""
    cfg = dict(full_config(), kernel_len=kernel_len)
    blob = make_weight_blob(**cfg)
    rng = np.random.default_rng(kernel_len)
    wins = rng.standard_normal((5, 2, kernel_len)).astype(np.float32)
    ref = onet.forward(onet.parse_blob(blob), wins)
    ctx = af.Context(kernel_len=kernel_len, precision=af.F16)
    got = ctx.forward(ctx.load_weights(blob), torch.from_numpy(wins).cuda()).cpu().numpy()
    assert rel_err(got, ref) <= 2e-2
    ctx32 = af.Context(kernel_len=kernel_len, precision=af.FP32)
    got32 = ctx32.forward(ctx32.load_weights(blob), torch.from_numpy(wins[:2]).cuda()).cpu().numpy()
    assert rel_err(got32, ref[:2]) <= 1e-4


def test_live_group_norm_tensor_core_fallback_statistics_path(af):
    """True GroupNorm on 1.25 s windows: the last stage has 80 rows per window (16-row tiles, 8 windows per tile), where
    the conv epilogue cannot emit per-window partial sums and the statistics are read back from z instead."""
    from synthdata import full_config_live_gn
    cfg = dict(full_config_live_gn(), kernel_len=2560)
    blob = make_weight_blob(**cfg)
    rng = np.random.default_rng(5)
    wins = rng.standard_normal((11, 2, 2560)).astype(np.float32)
    ref = onet.forward(onet.parse_blob(blob), wins)
    ctx = af.Context(kernel_len=2560, precision=af.F16)
    got = ctx.forward(ctx.load_weights(blob), torch.from_numpy(wins).cuda()).cpu().numpy()
    assert rel_err(got, ref) <= 2e-2


@pytest.mark.parametrize("stride,n_win", [(128, 2), (128, 3), (128, 37), (128, 301), (512, 5), (512, 64), (32, 150), (64, 33),
                                          (4, 40), (100, 21), (8, 500)])
def test_shared_stages_equal_the_per_window_path_bit_for_bit(af, config1, stride, n_win):
    """Overlapping in-place windows run in shared form (each stage once over the stream + two short edge windows per window,
    DESIGN.md section 5) when their spacing allows it; explicit [B][2][K] windows always take the per-window path.  Same
    kernels, same per-row arithmetic: the scores must be identical bit for bit, for chunk sizes 2, 3, odd, ragged, and for
    spacings that allow all stages (128, 512, 64, 32), only some (8), none but the stem (4) or nothing at all (100)."""
    rng = np.random.default_rng(stride * 1000 + n_win)
    white = torch.from_numpy(rng.standard_normal((2, (n_win - 1) * stride + 3072 + 2048)).astype(np.float32)).cuda().bfloat16()
    import math
    unit = math.lcm(2048, stride)                                # the configuration wants PSD lengths in whole strides and hops
    ctx = af.Context(precision=af.F16, stride=stride, psd_update=unit * -(-16384 // unit), psd_len=unit * -(-131072 // unit))
    w = ctx.load_weights(config1["blob"])
    shared = ctx.forward_strided(w, white.contiguous(), 0, n_win, chan_shift=[0, 2048])
    wins = torch.stack([torch.stack([white[0, i * stride: i * stride + 3072], white[1, 2048 + i * stride: 2048 + i * stride + 3072]])
                        for i in range(n_win)]).float().contiguous()
    ref = ctx.forward(w, wins)
    assert bool(torch.isfinite(shared).all())
    assert torch.equal(shared, ref)


@pytest.mark.parametrize("kernel_len", [512, 768, 1024, 1280, 2048, 2560, 4096])
def test_shared_stages_at_other_window_lengths(af, kernel_len):
    """Windows in place at stride 128 for short and long windows: the planner shares fewer stages where a stage's rows are
    too few for its edge rows (at 512 / 768 samples a window's first and last edge rows would meet in the 256- / 512-channel
    stage); what it shares must equal the per-window path -- bit for bit where both run the same kernel variant per layer
    (128-channel stage of a multiple of 128 rows: resident-weight halo tiles on both paths), else to rounding, because the
    per-window tiles of a shorter stage go through the tap-major kernel, which adds the same products in another order --
    and the oracle within rule T3."""
    cfg = dict(full_config(), kernel_len=kernel_len)
    blob = make_weight_blob(**cfg)
    n_win = 70
    rng = np.random.default_rng(kernel_len + 1)
    white = torch.from_numpy(rng.standard_normal((2, (n_win - 1) * 128 + kernel_len + 2048)).astype(np.float32)).cuda().half()
    ctx = af.Context(precision=af.F16, kernel_len=kernel_len)
    w = ctx.load_weights(blob)
    shared = ctx.forward_strided(w, white.contiguous(), 0, n_win, chan_shift=[0, 2048])
    wins = torch.stack([torch.stack([white[0, i * 128: i * 128 + kernel_len], white[1, 2048 + i * 128: 2048 + i * 128 + kernel_len]])
                        for i in range(n_win)]).float().contiguous()
    ref = ctx.forward(w, wins)
    assert bool(torch.isfinite(shared).all())
    if (kernel_len // 8) % 128 == 0:
        assert torch.equal(shared, ref)
    else:
        assert rel_err(shared.cpu().numpy(), ref.cpu().numpy()) <= 2e-3     # (measured 1e-3: one fp16 ulp is 5e-4)
    picks = [0, 1, n_win // 2, n_win - 1]
    want = onet.forward(onet.parse_blob(blob), wins[picks].cpu().numpy().astype(np.float64))
    assert rel_err(shared[picks].cpu().numpy(), want) <= 2e-2


def test_tensor_mac_counter_matches_the_layer_table(af, config1):
    """aframe_tensor_macs (bench.py's roofline numerator) counts, per launch, tile rows x C_out x K.  On the per-window path
    (explicit windows, 128 of them: every conv's rows fill whole 128-row tiles) that is the layer table's own MAC count,
    except for the 64-channel basic blocks, whose fused kernel computes 128-row MMAs per 126-row tile.  In shared form
    (overlapping in-place windows) the count must be well below the per-window figure and above the stream-only bound."""
    net = config1["net"]
    ctx = af.Context(precision=af.F16)
    w = ctx.load_weights(config1["blob"])
    B = 128
    m0 = ctx.tensor_macs()
    ctx.forward(w, torch.from_numpy(config1["wins"]).cuda())
    torch.cuda.synchronize()
    per_window = 0.0
    t_of = {-1: 3072}                                            # rows of every layer's output (layer table order)
    for i, layer in enumerate(net["layers"]):
        t_in = t_of[layer["input_from"]]
        if layer["kind"] == 2:                                   # head
            break
        t_of[i] = (t_in + 2 * layer["pad"] - layer["k"]) // layer["stride"] + 1
        if i < 2 or layer["kind"] != 0:                          # stem conv and max-pool run on CUDA cores
            continue
        t_out = t_of[i]
        rows = -(-t_out // 126) * 128 if (layer["c_in"] == 64 and layer["c_out"] == 64) else t_out
        per_window += rows * layer["c_out"] * layer["c_in"] * layer["k"]
    got = ctx.tensor_macs() - m0
    assert got == pytest.approx(B * per_window, rel=1e-12)
    # shared form: 4096 overlapping windows taken in place
    n_win = 4096
    white = torch.randn(2, (n_win - 1) * 128 + 3072 + 2048, device="cuda").bfloat16().contiguous()
    m1 = ctx.tensor_macs()
    ctx.forward_strided(w, white, 0, n_win, chan_shift=[0, 2048])
    torch.cuda.synchronize()
    shared = (ctx.tensor_macs() - m1) / n_win
    algorithmic = 1069.5e6
    assert 0.04 * algorithmic < shared < 0.5 * algorithmic      # stream alone: 128 of 3072 samples per window = 1/24
