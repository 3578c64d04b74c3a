"""GPU parity (through the C ABI) of the streaming state (O-6, BASELINE.json configs[2]/[4]) and of the offline
timeslide driver (configs[3]) against the float64 oracle."""
import numpy as np
import pytest
import torch

from oracle import network as onet
from oracle import stream as ost
from synthdata import coloured_noise, make_weight_blob, tiny_config, full_config

pytestmark = pytest.mark.gpu
FS = 2048
S = 128


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


def rel_err(g, o):
    g, o = np.asarray(g, np.float64), np.asarray(o, np.float64)
    return float(np.max(np.abs(g - o) / np.maximum(np.abs(o), 1e-3 * np.abs(o).max())))


def _run_stream(af, ctx, w, x, n_updates):
    st = ctx.stream_create(w)
    upd = torch.from_numpy(np.ascontiguousarray(x[:, : n_updates * S].reshape(2, n_updates, S).transpose(1, 0, 2))).cuda()
    flags, scores = [], []
    for u in range(n_updates):
        st.step(upd[u])
        flags.append(int(st.n_scores.item()))
        scores.append(float(st.score.item()))
    st.close()
    return np.asarray(flags), np.asarray(scores)


def test_stream_fp32_matches_oracle_through_warmup_and_a_psd_update(af):
    """configs[2]/[4] geometry (64 s PSD, update every 8 s, stride 128) with the tiny network in fp32: warm-up flags
    (reading C1), every score up to and across the second PSD epoch (reading C2), rule T2."""
    tc = tiny_config()
    n_updates = (131072 + 16384) // S + 12                      # past the second PSD (n = 147456)
    x = coloured_noise(n_updates * S, seed=1002)
    cfg = ost.StreamConfig(kernel_len=tc["kernel_len"], n_design=4096)
    blob = make_weight_blob(**tc)
    so = ost.StreamOracle(cfg, net=onet.parse_blob(blob))
    ref = [so.step(x[:, u * S:(u + 1) * S].astype(np.float64)) for u in range(n_updates)]
    assert so.n_psd_updates == 2

    ctx = af.Context(n_design=4096, kernel_len=tc["kernel_len"], precision=af.FP32)
    w = ctx.load_weights(blob)
    flags, scores = _run_stream(af, ctx, w, x, n_updates)
    exp_flags = np.array([0 if r is None else 1 for r in ref])
    np.testing.assert_array_equal(flags, exp_flags)
    first = int(np.argmax(exp_flags))
    assert first == 131072 // S - 1 + tc["kernel_len"] // S - 1   # first PSD at update 1023, window full 15 updates later
    got = scores[first:]
    want = np.array([r for r in ref if r is not None])
    assert rel_err(got, want) <= 1e-4


def test_stream_tensor_core_full_network_scores(af):
    """configs[4]: config-1 network on the fp16 tensor-core path at batch 1; rule T3 on the first scored updates."""
    fc = full_config()
    n_updates = 131072 // S + 3072 // S + 6
    x = coloured_noise(n_updates * S, seed=1002)
    blob = make_weight_blob(**fc)
    so = ost.StreamOracle(ost.StreamConfig(), net=onet.parse_blob(blob))
    ref = [so.step(x[:, u * S:(u + 1) * S].astype(np.float64)) for u in range(n_updates)]
    ctx = af.Context(precision=af.F16)
    w = ctx.load_weights(blob)
    flags, scores = _run_stream(af, ctx, w, x, n_updates)
    np.testing.assert_array_equal(flags, [0 if r is None else 1 for r in ref])
    want = np.array([r for r in ref if r is not None])
    assert len(want) == n_updates - (131072 // S - 1 + 3072 // S - 1)
    assert rel_err(scores[flags == 1], want) <= 2e-2


def test_stream_reset_reproduces_the_same_scores(af):
    tc = tiny_config()
    n_updates = 131072 // S + tc["kernel_len"] // S + 3
    x = coloured_noise(n_updates * S, seed=5)
    ctx = af.Context(n_design=4096, kernel_len=tc["kernel_len"], precision=af.FP32)
    w = ctx.load_weights(make_weight_blob(**tc))
    st = ctx.stream_create(w)
    upd = torch.from_numpy(np.ascontiguousarray(x.reshape(2, n_updates, S).transpose(1, 0, 2))).cuda()
    runs = []
    for _ in range(2):
        out = []
        for u in range(n_updates):
            st.step(upd[u])
            if u >= n_updates - 3:
                out.append((int(st.n_scores.item()), float(st.score.item())))
        runs.append(out)
        st.reset()
    assert runs[0] == runs[1] and all(f == 1 for f, _ in runs[0])


def test_stream_graph_replay_equals_direct_launches(af):
    """On a non-default stream one update is one CUDA-graph launch (configs[4]); the scores must be the same bits as
    the direct launch sequence of a context bound to the default stream."""
    fc = full_config()
    n_updates = 131072 // S + 3072 // S + 4
    x = coloured_noise(n_updates * S, seed=11)
    blob = make_weight_blob(**fc)
    upd = torch.from_numpy(np.ascontiguousarray(x.reshape(2, n_updates, S).transpose(1, 0, 2))).cuda()
    buf = torch.empty((2, S), dtype=torch.float32, device="cuda")
    out = {}
    for name, stream in (("direct", None), ("graph", torch.cuda.Stream())):
        ctx = af.Context(precision=af.F16, stream=stream)
        w = ctx.load_weights(blob)
        st = ctx.stream_create(w)
        scores = []
        with torch.cuda.stream(stream if stream is not None else torch.cuda.current_stream()):
            for u in range(n_updates):
                buf.copy_(upd[u], non_blocking=True)           # same device buffer every update -> one captured graph
                st.step(buf)
                if u >= n_updates - 5:
                    torch.cuda.current_stream().synchronize()
                    scores.append((int(st.n_scores.item()), float(st.score.item())))
            torch.cuda.current_stream().synchronize()
        out[name] = (scores, st.uses_graph)
        st.close()
    # a large forward on the graph context re-allocates its activation workspace: the next update must re-capture
    big = ctx.forward(w, torch.randn(64, 2, 3072, device="cuda"))
    st2 = ctx.stream_create(w)
    with torch.cuda.stream(stream):
        for u in range(3):
            buf.copy_(upd[u], non_blocking=True)
            st2.step(buf)
        ctx.forward(w, torch.randn(700, 2, 3072, device="cuda"))       # grows the workspace
        for u in range(3, 6):
            buf.copy_(upd[u], non_blocking=True)
            st2.step(buf)
        stream.synchronize()
    assert int(st2.n_scores.item()) == 0 and bool(torch.isfinite(big).all())
    st2.close()
    assert out["graph"][1] and not out["direct"][1]
    assert out["graph"][0] == out["direct"][0] and all(f == 1 for f, _ in out["graph"][0])


def test_score_timeslides_device_host_and_oracle(af):
    """configs[3] in one call: whiten once, score every timeslide.  (a) equals aframe_forward_strided on the rolling-
    whitened stream, bit for bit; (b) the host-buffer entry point returns the same bits; (c) sampled windows match the
    float64 oracle (rolling whitening + network) within rule T3; (d) windows past the segment are refused."""
    fc = full_config()
    n_win, shifts, batch = 200, [2048, 3 * 2048], 96           # ragged last batch
    m0 = 131072 - S - 1024
    n_white = (n_win - 1) * S + max(shifts) + 3072
    n_raw = -(-(m0 + n_white + 1024) // S) * S + 16384          # crosses a PSD epoch
    x = coloured_noise(n_raw, seed=1003)
    blob = make_weight_blob(**fc)
    ctx = af.Context(precision=af.F16)
    w = ctx.load_weights(blob)
    xd = torch.from_numpy(x).cuda()
    dev = ctx.score_timeslides(w, xd, 0, n_win, shifts, batch=batch)
    assert dev.shape == (2, n_win) and dev.is_cuda
    white = ctx.whiten_rolling(xd, out_dtype=torch.float16).contiguous()   # the call keeps its whitened stream as fp16
    for k, sh in enumerate(shifts):
        ref = ctx.forward_strided(w, white, 0, n_win, chan_shift=[0, sh])
        assert torch.equal(dev[k], ref)
    host = ctx.score_timeslides(w, torch.from_numpy(x).pin_memory(), 0, n_win, shifts, batch=batch)
    assert not host.is_cuda and torch.equal(host, dev.cpu())

    cfg = ost.StreamConfig()
    net = onet.parse_blob(blob)
    x64 = x.astype(np.float64)
    picks = [(0, 0), (0, n_win - 1), (1, 17), (1, n_win - 1), (1, 128)]
    wins = []
    for k, i in picks:
        a = m0 + i * S
        h1, _ = ost.whiten_rolling(x64[0], cfg, m_lo=a, m_hi=a + 3072)
        l1, _ = ost.whiten_rolling(x64[1], cfg, m_lo=a + shifts[k], m_hi=a + shifts[k] + 3072)
        wins.append(np.stack([h1, l1]))
    want = onet.forward(net, np.stack(wins))
    got = np.array([float(dev[k, i]) for k, i in picks])
    assert rel_err(got, want) <= 2e-2

    with pytest.raises(af.AframeError) as e:
        ctx.score_timeslides(w, xd, 0, n_win + 2000, shifts, batch=batch)
    assert e.value.status == af.ESHAPE


@pytest.mark.parametrize("stride", [512, 32])
def test_other_inference_rates(af, stride):
    """NEXT-3 (the paper infers at 4 Hz = stride 512; P:174 studies 1..64 Hz): the streaming state and the strided
    forward at other strides, tiny network in fp32, against the oracle (flags exactly, scores to rule T2)."""
    tc = tiny_config()
    n_updates = 131072 // stride + tc["kernel_len"] // stride + (4 if stride == 512 else 40)
    x = coloured_noise(n_updates * stride, seed=1002)
    cfg = ost.StreamConfig(kernel_len=tc["kernel_len"], n_design=4096, stride=stride)
    blob = make_weight_blob(**tc)
    so = ost.StreamOracle(cfg, net=onet.parse_blob(blob))
    ref = [so.step(x[:, u * stride:(u + 1) * stride].astype(np.float64)) for u in range(n_updates)]
    ctx = af.Context(n_design=4096, kernel_len=tc["kernel_len"], stride=stride, precision=af.FP32)
    w = ctx.load_weights(blob)
    st = ctx.stream_create(w)
    upd = torch.from_numpy(np.ascontiguousarray(x.reshape(2, n_updates, stride).transpose(1, 0, 2))).cuda()
    flags, scores = [], []
    for u in range(n_updates):
        st.step(upd[u])
        flags.append(int(st.n_scores.item())); scores.append(float(st.score.item()))
    st.close()
    flags, scores = np.asarray(flags), np.asarray(scores)
    np.testing.assert_array_equal(flags, [0 if r is None else 1 for r in ref])
    want = np.array([r for r in ref if r is not None])
    assert len(want) >= 4 and rel_err(scores[flags == 1], want) <= 1e-4
    # offline: rolling whitening + windows in place at this stride = the streamed windows
    white = ctx.whiten_rolling(torch.from_numpy(x).cuda()).contiguous()
    n_win = (white.shape[1] - tc["kernel_len"]) // stride + 1
    off = ctx.forward_strided(w, white, 0, n_win).cpu().numpy()
    assert n_win == len(want) and rel_err(off, want) <= 1e-4


@pytest.mark.parametrize("average", ["mean", "median"])
def test_eight_second_psd_and_median_variants_in_the_streaming_state(af, average):
    """NEXT-3: the 8 s PSD of P:102 (psd_len 16384 = 7 segments) refreshed every 2 s, with the mean or the median over the
    segments, through the streaming state and the rolling offline call, tiny network in fp32, against the oracle."""
    tc = tiny_config()
    psd_len, psd_update = 16384, 4096
    n_updates = (psd_len + tc["kernel_len"] + 3 * psd_update) // S + 5
    x = coloured_noise(n_updates * S, seed=1003)
    x[1, 20000] += 2e-19                                          # a glitch inside several PSD epochs
    cfg = ost.StreamConfig(kernel_len=tc["kernel_len"], n_design=4096, psd_len=psd_len, psd_update=psd_update,
                           welch_average=average)
    blob = make_weight_blob(**tc)
    so = ost.StreamOracle(cfg, net=onet.parse_blob(blob))
    ref = [so.step(x[:, u * S:(u + 1) * S].astype(np.float64)) for u in range(n_updates)]
    assert so.n_psd_updates >= 4
    ctx = af.Context(n_design=4096, kernel_len=tc["kernel_len"], psd_len=psd_len, psd_update=psd_update,
                     welch_average=1 if average == "median" else 0, precision=af.FP32)
    w = ctx.load_weights(blob)
    flags, scores = _run_stream(af, ctx, w, x, n_updates)
    np.testing.assert_array_equal(flags, [0 if r is None else 1 for r in ref])
    want = np.array([r for r in ref if r is not None])
    assert len(want) > 3 * psd_update // S and rel_err(scores[flags == 1], want) <= 1e-4
    white = ctx.whiten_rolling(torch.from_numpy(x).cuda()).contiguous()
    n_win = (white.shape[1] - tc["kernel_len"]) // S + 1
    off = ctx.forward_strided(w, white, 0, n_win).cpu().numpy()
    assert n_win == len(want) and rel_err(off, want) <= 1e-4


def test_stride_one_windows_offline(af):
    """NEXT-3 ("2048 Hz" online inference = one window per sample): rolling whitening and in-place windows at
    stride 1, tiny network in fp32, against the oracle."""
    tc = tiny_config()
    K = tc["kernel_len"]
    x = coloured_noise(131072 + 4096 + K, seed=1004)
    cfg = ost.StreamConfig(kernel_len=K, n_design=4096, stride=1)
    blob = make_weight_blob(**tc)
    ctx = af.Context(n_design=4096, kernel_len=K, stride=1, precision=af.FP32)
    w = ctx.load_weights(blob)
    white = ctx.whiten_rolling(torch.from_numpy(x).cuda()).contiguous()
    y = np.stack([ost.whiten_rolling(x[c].astype(np.float64), cfg)[0] for c in range(2)])
    assert white.shape[1] == y.shape[1]
    rms = np.sqrt(np.mean(y ** 2))
    assert np.abs(white.cpu().numpy() - y).max() <= 1e-4 * rms                 # rule T1
    n_win = 333
    got = ctx.forward_strided(w, white, 0, n_win).cpu().numpy()
    wins = ost.unfold(y, K, 1, n_windows=n_win)
    ref = onet.forward(onet.parse_blob(blob), wins)
    assert rel_err(got, ref) <= 1e-4


def test_bench_step_at_full_size_sampled_against_oracle(af):
    """BASELINE.json configs[3] in the launch configuration bench.py times: one 4096 s block of two-detector strain with
    232 injected chirps (plus its 64 s PSD history), 8 timeslides x 65 536 windows, batches of 4096 windows, through aframe_score_timeslides.
    The float64 oracle (rolling whitening with the epoch's own Welch PSD + network) recomputes a seeded sample of the
    524 288 scores one by one: the first and last valid window of each slide, windows on both sides of PSD-epoch
    boundaries, windows that hold a chirp's coalescence in H1 (slides misalign L1: background) and pseudo-random ones
    (rule T3); all scores must be finite."""
    import bench
    fc = full_config()
    n_win, n_raw = bench.block_geometry(4096)
    shifts = [k * FS for k in range(1, bench.N_SLIDES + 1)]
    from synthdata.configs import config3_block
    x, params = config3_block(7, n_raw)
    assert np.array_equal(x, bench.make_block(7, n_raw)) and len(params) > 200
    blob = make_weight_blob(**fc)
    ctx = af.Context(precision=af.F16)
    w = ctx.load_weights(blob)
    scores = ctx.score_timeslides(w, torch.from_numpy(x).cuda(), 0, n_win, shifts, batch=4096)
    assert scores.shape == (bench.N_SLIDES, n_win) and bool(torch.isfinite(scores).all())
    scores = scores.cpu().numpy()

    cfg = ost.StreamConfig()
    m0 = cfg.psd_len - S - cfg.filter_len // 2                  # raw index of whitened sample 0 (reading C1)
    rng = np.random.default_rng(20240318)
    picks = [(k, 0) for k in (0, 7)] + [(k, n_win - 1) for k in (0, 3, 7)]
    # windows whose samples straddle the switch to PSD epoch e (raw index where epoch e starts: reading C2)
    for e in (1, 97, 255):
        m_switch = cfg.psd_len + e * cfg.psd_update - S - cfg.filter_len // 2
        i = (m_switch - m0) // S
        picks += [(2, i - 30), (5, i - 1), (5, i)]
    for j, p in enumerate(params[3:60:8]):                      # H1 coalescence 0.25 .. 1.25 s into the window
        i_c = (int(round(p.t_c * FS)) - m0) // S
        picks += [(j % 8, i_c - 4 - 2 * j)]
    picks += [(int(rng.integers(0, 8)), int(rng.integers(0, n_win))) for _ in range(32)]
    x64 = x.astype(np.float64)
    net = onet.parse_blob(blob)
    wins = []
    for k, i in picks:
        a = m0 + i * S
        h1, _ = ost.whiten_rolling(x64[0], cfg, m_lo=a, m_hi=a + 3072)
        l1, _ = ost.whiten_rolling(x64[1], cfg, m_lo=a + shifts[k], m_hi=a + shifts[k] + 3072)
        wins.append(np.stack([h1, l1]))
    want = onet.forward(net, np.stack(wins))
    got = np.array([scores[k, i] for k, i in picks], dtype=np.float64)
    assert rel_err(got, want) <= 2e-2


def test_configurations_the_streaming_state_or_the_path_cannot_honour_are_refused(af):
    """(a) a stride that does not divide the Welch hop would leave Welch segments that end between two updates uncomputed
    (the PSD would silently come out low): aframe_stream_create refuses it; the offline calls, which compute every segment
    from the stored record, accept it.  (b) bf16 is a stream storage type only: as the network precision it is refused."""
    tc = tiny_config()
    ctx = af.Context(n_design=4096, kernel_len=tc["kernel_len"], stride=3072, psd_len=129024, psd_update=18432, precision=af.FP32)
    w = ctx.load_weights(make_weight_blob(**tc))
    with pytest.raises(af.AframeError) as e:
        ctx.stream_create(w)
    assert e.value.status == af.ESHAPE
    x = torch.from_numpy(coloured_noise(129024 + 2 * 18432, seed=3)).cuda()
    assert ctx.whiten_rolling(x).shape[1] > 0
    with pytest.raises(af.AframeError) as e:
        af.Context(precision=af.BF16)
    assert e.value.status == af.EUNSUPPORTED


def test_objects_may_be_destroyed_in_any_order_and_graphs_are_kept_per_buffer(af):
    """Lifetime (aframe.h): closing the context first, or freeing the weights under a live stream state, leaves dead shells
    that only accept their own free / destroy call; a caller that alternates between buffers keeps one graph per buffer
    (all but the first update per buffer are replays) and gets the same scores as with a single buffer."""
    tc = tiny_config()
    blob = make_weight_blob(**tc)
    n_updates = 131072 // S + tc["kernel_len"] // S + 6
    x = coloured_noise(n_updates * S, seed=21)
    upd = torch.from_numpy(np.ascontiguousarray(x.reshape(2, n_updates, S).transpose(1, 0, 2))).cuda()
    stream = torch.cuda.Stream()
    out = {}
    with torch.cuda.stream(stream):
        for n_buf in (1, 3):
            ctx = af.Context(n_design=4096, kernel_len=tc["kernel_len"], precision=af.FP32, stream=stream)
            w = ctx.load_weights(blob)
            st = ctx.stream_create(w)
            bufs = [torch.empty((2, S), dtype=torch.float32, device="cuda") for _ in range(n_buf)]
            scores = []
            for u in range(n_updates):
                b = bufs[u % n_buf]
                b.copy_(upd[u], non_blocking=True)
                st.step(b)
                if u >= n_updates - 6:
                    stream.synchronize()
                    scores.append((int(st.n_scores.item()), float(st.score.item())))
            stream.synchronize()
            replays = int(ctx.lib.aframe_stream_graph_replays(st.handle))
            assert replays == n_updates                         # every update went through a graph; captures: n_buf
            out[n_buf] = scores
            if n_buf == 1:
                ctx.close()                                     # context first: children become dead shells
                st.close(); w.free()
            else:
                w.free()                                        # weights under a live state: the state is released
                with pytest.raises(af.AframeError) as e:
                    st.step(bufs[0])
                assert e.value.status == af.ESTATE
                st.close(); ctx.close()
    assert out[1] == out[3] and all(f == 1 for f, _ in out[1])


@pytest.mark.parametrize("stride", [128, 64, 32])
def test_incremental_network_equals_a_full_forward_per_update_and_the_oracle(af, stride):
    """configs[4] with the incremental network (stream_net.cu: per update and layer only the new stream rows and the window's
    head / tail rows, one cluster kernel) against (a) the same state running one full forward of the window per update
    (cfg.stream_full_forward = 1: same fp16 roundings, other summation order) on every scored update, through two PSD updates
    and a reset, and (b) the float64 oracle (rule T3) on a sample of the updates.  8 s PSD refreshed every 2 s keeps
    the warm-up short."""
    fc = full_config()
    psd_len, psd_update, K = 16384, 4096, fc["kernel_len"]
    n_updates = (psd_len + K + 2 * psd_update) // stride + 40
    x = coloured_noise(n_updates * stride, seed=1004)
    x[0, psd_len + 3000: psd_len + 3400] += 4e-21 * np.sin(np.arange(400) * 0.3)      # something that is not noise
    blob = make_weight_blob(**fc)
    upd = torch.from_numpy(np.ascontiguousarray(x.reshape(2, n_updates, stride).transpose(1, 0, 2))).cuda()
    res = {}
    stream = torch.cuda.Stream()                                 # (the legacy default stream cannot be captured into a graph)
    for full in (0, 1, 2):                                       # 2: the incremental network on the portable cluster size 8
        if full == 2 and stride != 128:
            continue
        with torch.cuda.stream(stream):
            ctx = af.Context(precision=af.F16, stride=stride, psd_len=psd_len, psd_update=psd_update, stream_full_forward=full,
                             stream=stream)
            w = ctx.load_weights(blob)
            st = ctx.stream_create(w)
            assert (st.incremental == 0) == (full == 1) and st.incremental in (0, 8, 16) and (full != 2 or st.incremental == 8)
            out = torch.zeros((2, n_updates, 2), dtype=torch.float32, device="cuda")
            buf = torch.empty((2, stride), dtype=torch.float32, device="cuda")
            for rep in range(2 if full == 0 else 1):             # the incremental state again after a reset
                if rep:
                    st.reset()
                for u in range(n_updates):
                    buf.copy_(upd[u], non_blocking=True)
                    st.step(buf)
                    out[rep, u, 0].copy_(st.score[0], non_blocking=True)
                    out[rep, u, 1].copy_(st.n_scores[0], non_blocking=True)
            stream.synchronize()
            assert st.uses_graph
            res[full] = out.cpu().numpy()
            st.close()
    inc, ful = res[0], res[1]
    if 2 in res:                                                 # 8 or 16 CTAs: other K split, same roundings
        np.testing.assert_array_equal(res[2][0, :, 1], inc[0, :, 1])
        assert rel_err(res[2][0, inc[0, :, 1] == 1, 0], inc[0, inc[0, :, 1] == 1, 0]) <= 2e-3
    np.testing.assert_array_equal(inc[0, :, 1], ful[0, :, 1])
    scored = inc[0, :, 1] == 1
    np.testing.assert_array_equal(inc[0, :, 1], inc[1, :, 1])    # reset reproduces the run bit for bit
    np.testing.assert_array_equal(inc[0, scored, 0], inc[1, scored, 0])
    first = int(np.argmax(scored))
    assert first == psd_len // stride - 1 + K // stride - 1 and scored[first:].all()
    assert rel_err(inc[0, scored, 0], ful[0, scored, 0]) <= 2e-3
    # oracle on every 8th scored update and on the updates around the PSD switches
    cfg = ost.StreamConfig(stride=stride, psd_len=psd_len, psd_update=psd_update)
    m0 = ost.first_whitened_index(cfg)
    picks = sorted(set(range(first, n_updates, 8)) | {u for u in range(first, n_updates) if ((u + 1) * stride) % psd_update < 3 * stride})
    x64 = x.astype(np.float64)
    filters = [{}, {}]
    wins = np.empty((len(picks), 2, K))
    for j, u in enumerate(picks):
        a = m0 + (u - first) * stride
        for c in range(2):
            wins[j, c], _ = ost.whiten_rolling(x64[c], cfg, m_lo=a, m_hi=a + K, filters=filters[c])
    want = onet.forward(onet.parse_blob(blob), wins)
    assert len(picks) >= 20 and rel_err(inc[0, picks, 0], want) <= 2e-2 and rel_err(ful[0, picks, 0], want) <= 2e-2


def test_incremental_network_is_not_used_where_it_does_not_apply(af):
    fc, tc = full_config(), tiny_config()
    ctx = af.Context(precision=af.F16, stride=512)               # more than 48 rows per layer and update
    w = ctx.load_weights(make_weight_blob(**fc))
    st = ctx.stream_create(w)
    assert st.incremental == 0
    st.close()
    ctx = af.Context(n_design=4096, kernel_len=tc["kernel_len"], precision=af.FP32)   # fp32 CUDA-core path
    w = ctx.load_weights(make_weight_blob(**tc))
    st = ctx.stream_create(w)
    assert st.incremental == 0
    st.close()
