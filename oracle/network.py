"""O-5  1D ResNet forward pass in float64.  (Oracle: test infrastructure only.)

Paper: "Our neural-network architecture modifies a standard ResNet54 [...] maps fixed
length time-series of gravitational wave strain from two interferometers [...] to a scalar
detection statistic [...] we replace 2D with 1D convolutions [...] replace standard Batch
Normalization layers with Group Normalization" (Sec. II); "the architecture implements
global pooling layers, the convolution layers use a kernel length of 3 samples".
The paper states no widths/strides; BASELINE.json configs[0]/[1] fix them and readings B1-B8
 fix the rest.  The architecture is data: a layer table in the weight blob
(format: synthdata/weights.py; this file has its own parser).

  conv1d : out[co][t] = sum_ci sum_{d<k} W[co][ci][d] in[ci][t*stride + d - pad], zero outside [0, T_in)
           T_out = floor((T_in + 2 pad - k)/stride) + 1                                   (B3)
  norm   : frozen statistics, y = (z - mu_g)/sqrt(v_g + eps) gamma_c + beta_c             (B6)
           folded form  W' = a_c W, b' = beta_c - mu_g a_c, a_c = gamma_c / sqrt(v_g + eps)
  layer  : y = norm(conv(in)); y += out[residual_from] (if any); y = relu(y) (if relu)     (B4)
  maxpool: max over the k taps, padding never wins                                       (B3)
  head   : mean over T, dot with w, + b  -> raw logit (no sigmoid)                        (B8)
"""
from __future__ import annotations

import struct

import numpy as np

KIND_CONV, KIND_MAXPOOL, KIND_HEAD = 0, 1, 2


def parse_blob(blob: bytes):
    magic, version, n_layers, norm_kind, n_groups, eps_bits, in_ch, _ = struct.unpack_from("<8I", blob, 0)
    if magic != 0x57524641 or version != 1:
        raise ValueError("bad weight blob")
    eps = struct.unpack("<f", struct.pack("<I", eps_bits))[0]
    tab = np.frombuffer(blob, dtype="<i4", count=n_layers * 12, offset=32).reshape(n_layers, 12)
    data = np.frombuffer(blob, dtype="<f4", offset=32 + n_layers * 48).astype(np.float64)
    pos = 0
    layers = []
    for row in tab:
        kind, c_in, c_out, k, stride, pad, relu, inp, res = (int(v) for v in row[:9])
        l = dict(kind=kind, c_in=c_in, c_out=c_out, k=k, stride=stride, pad=pad, relu=relu,
                 input_from=inp, residual_from=res)
        if kind == KIND_CONV:
            n_stat = c_out if norm_kind == 0 else (n_groups if norm_kind == 1 else 0)
            l["W"] = data[pos: pos + c_out * c_in * k].reshape(c_out, c_in, k); pos += c_out * c_in * k
            l["gamma"] = data[pos: pos + c_out]; pos += c_out
            l["beta"] = data[pos: pos + c_out]; pos += c_out
            l["mean"] = data[pos: pos + n_stat]; pos += n_stat
            l["var"] = data[pos: pos + n_stat]; pos += n_stat
        elif kind == KIND_HEAD:
            l["w"] = data[pos: pos + c_in]; pos += c_in
            l["b"] = float(data[pos]); pos += 1
        layers.append(l)
    if pos != data.size:
        raise ValueError("weight blob payload size mismatch")
    return dict(layers=layers, norm_kind=norm_kind, n_groups=n_groups, eps=float(eps), in_channels=in_ch)


def stat_index(c_out, norm_kind, n_groups):
    """Channel -> index of its statistics: c (per-channel) or c // (C / n_groups) (reading B6)."""
    c = np.arange(c_out)
    return c if norm_kind == 0 else c // (c_out // n_groups)


def group_norm_live(z, gamma, beta, n_groups, eps):
    """True GroupNorm ("replace standard Batch Normalization layers with Group Normalization"; NEXT-2): per window
    and per group of C / n_groups consecutive channels, mean and (biased) variance over the group's channels and all
    time steps; y = (z - mu) / sqrt(var + eps) * gamma_c + beta_c.   z [B][C][T]."""
    b, c, t = z.shape
    zg = z.reshape(b, n_groups, (c // n_groups) * t)
    mu = zg.mean(axis=2, keepdims=True)
    var = ((zg - mu) ** 2).mean(axis=2, keepdims=True)
    y = ((zg - mu) / np.sqrt(var + eps)).reshape(b, c, t)
    return y * gamma[None, :, None] + beta[None, :, None]


def fold_norm(layer, norm_kind, n_groups, eps):
    """(W', b') with W' = a_c W, b' = beta_c - mu_g a_c."""
    g = stat_index(layer["c_out"], norm_kind, n_groups)
    a = layer["gamma"] / np.sqrt(layer["var"][g] + eps)
    return layer["W"] * a[:, None, None], layer["beta"] - layer["mean"][g] * a


def conv1d_direct(x, w, stride, pad):
    """The definition, summed tap by tap.  x [C_in][T], w [C_out][C_in][k] -> [C_out][T_out]."""
    c_in, t_in = x.shape
    c_out, _, k = w.shape
    t_out = (t_in + 2 * pad - k) // stride + 1
    out = np.zeros((c_out, t_out), dtype=np.float64)
    for co in range(c_out):
        for ci in range(c_in):
            for d in range(k):
                for t in range(t_out):
                    s = t * stride + d - pad
                    if 0 <= s < t_in:
                        out[co, t] += w[co, ci, d] * x[ci, s]
    return out


def conv1d(x, w, stride, pad):
    """Same sums as ``conv1d_direct`` with the (ci, d) loops done by one matrix product per window
    (zero-padded im2col).  x [B][C_in][T] -> [B][C_out][T_out].  Tests prove it equals the definition."""
    b, c_in, t_in = x.shape
    c_out, _, k = w.shape
    t_out = (t_in + 2 * pad - k) // stride + 1
    xp = np.zeros((b, c_in, t_in + 2 * pad), dtype=np.float64)
    xp[:, :, pad: pad + t_in] = x
    cols = np.empty((b, c_in, k, t_out), dtype=np.float64)
    for d in range(k):
        cols[:, :, d, :] = xp[:, :, d: d + stride * (t_out - 1) + 1: stride]
    return np.matmul(w.reshape(c_out, c_in * k), cols.reshape(b, c_in * k, t_out))


def maxpool1d(x, k, stride, pad):
    b, c, t_in = x.shape
    t_out = (t_in + 2 * pad - k) // stride + 1
    xp = np.full((b, c, t_in + 2 * pad), -np.inf, dtype=np.float64)
    xp[:, :, pad: pad + t_in] = x
    out = np.full((b, c, t_out), -np.inf, dtype=np.float64)
    for d in range(k):
        out = np.maximum(out, xp[:, :, d: d + stride * (t_out - 1) + 1: stride])
    return out


def round_bf16(x):
    """float64 -> float32 (RNE) -> bfloat16 (RNE) -> float64; emulates the CUDA path's storage rounding."""
    f = np.asarray(x, dtype=np.float64).astype(np.float32)
    u = f.view(np.uint32).astype(np.uint64)
    r = ((u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000).astype(np.uint32)
    return r.view(np.float32).astype(np.float64)


def round_f16(x):
    """float64 -> float32 (RNE) -> IEEE half (RNE, finite values beyond +-65504 saturate, NaN stays NaN) -> float64;
    emulates the activation storage of the CUDA tensor-core path (reading B10)."""
    f = np.clip(np.asarray(x, dtype=np.float64).astype(np.float32), np.float32(-65504.0), np.float32(65504.0))
    return f.astype(np.float16).astype(np.float64)


def forward(net, windows, folded=True, act_round=None, weight_round=None, keep=False):
    """windows [B][C][K] float -> scores [B] float64.

    folded=False evaluates conv -> explicit norm (the unfolded form of reading B6); tests prove both
    agree.  act_round / weight_round (optional callables) emulate the 16-bit storage points of the CUDA
    path (reading B10: weight_round = round_bf16; act_round = round_f16, or round_bf16 for the "bf16-ideal
    ceiling" that motivated fp16 activations); the parity oracle leaves them None.
    """
    x0 = np.asarray(windows, dtype=np.float64)
    outs = []
    nk, ng, eps = net["norm_kind"], net["n_groups"], net["eps"]
    for li, l in enumerate(net["layers"]):
        src = x0 if l["input_from"] < 0 else outs[l["input_from"]]
        if l["kind"] == KIND_CONV:
            if nk == 2:                            # true GroupNorm: nothing to fold
                w = l["W"]
                if weight_round is not None and l["input_from"] >= 0:
                    w = weight_round(w)
                y = group_norm_live(conv1d(src, w, l["stride"], l["pad"]), l["gamma"], l["beta"], ng, eps)
            elif folded:
                w, bias = fold_norm(l, nk, ng, eps)
                if weight_round is not None and l["input_from"] >= 0:
                    w = weight_round(w)
                y = conv1d(src, w, l["stride"], l["pad"]) + bias[None, :, None]
            else:
                z = conv1d(src, l["W"], l["stride"], l["pad"])
                g = stat_index(l["c_out"], nk, ng)
                y = ((z - l["mean"][g][None, :, None]) / np.sqrt(l["var"][g] + eps)[None, :, None]
                     * l["gamma"][None, :, None] + l["beta"][None, :, None])
            if l["residual_from"] >= 0:
                y = y + outs[l["residual_from"]]
            if l["relu"]:
                y = np.maximum(y, 0.0)
            nxt = net["layers"][li + 1] if li + 1 < len(net["layers"]) else None
            fused_pool = nxt is not None and nxt["kind"] == KIND_MAXPOOL and nxt["input_from"] == li
            if act_round is not None and not fused_pool:
                y = act_round(y)
        elif l["kind"] == KIND_MAXPOOL:
            y = maxpool1d(src, l["k"], l["stride"], l["pad"])
            if act_round is not None:
                y = act_round(y)
        elif l["kind"] == KIND_HEAD:
            y = src.mean(axis=2) @ l["w"] + l["b"]
        else:
            raise ValueError("unknown layer kind")
        outs.append(y)
    return (outs[-1], outs) if keep else outs[-1]


def output_length(net, kernel_len):
    """Time length after every layer (shape arithmetic of B2: 3072 -> 1536 -> 768 -> ... -> 96)."""
    lens = []
    for l in net["layers"]:
        t_in = kernel_len if l["input_from"] < 0 else lens[l["input_from"]]
        if l["kind"] == KIND_HEAD:
            lens.append(1)
        else:
            lens.append((t_in + 2 * l["pad"] - l["k"]) // l["stride"] + 1)
    return lens
