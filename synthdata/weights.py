"""Seeded network parameters and the weight-blob writer.

The paper's trained weights are not available (PAPER.md:39 describes the network:
"standard ResNet54" with 1D convolutions and GroupNorm; conv kernel
length 3, global pooling).  BASELINE.json fixes the shapes (configs[0], configs[1]);
readings B1-B7 of SURVEY.md 8(c) fix the rest.  The architecture is DATA: a layer
table in the blob.  The blob stores UNFOLDED parameters (W, gamma, beta, mean, var);
the oracle and the CUDA library each fold the norm themselves.

Blob format (little endian), version 1
--------------------------------------
header, 32 bytes : u32 magic 'AFRW' (0x57524641), u32 version=1, u32 n_layers,
                   u32 norm_kind (0 = frozen per-channel statistics, 1 = frozen per-group statistics,
                                  2 = true GroupNorm: statistics computed per window at inference, NEXT-2),
                   u32 n_groups (norm_kind 1 only), f32 eps, u32 in_channels, u32 reserved
layer table      : n_layers x 12 x i32:
                   kind (0 conv+norm, 1 maxpool, 2 head = global-avg-pool + linear),
                   c_in, c_out, k, stride, pad, relu,
                   input_from (-1 = network input, else index of an earlier layer),
                   residual_from (-1 = none; added after the norm, before the ReLU),
                   3 reserved
payload (f32)    : per conv layer, in table order: W[c_out][c_in][k], gamma[c_out], beta[c_out],
                   mean[n_stat], var[n_stat]   (n_stat = c_out or n_groups; norm_kind 2: n_stat = 0, no statistics stored)
                   per head layer: w[c_in], b[1]
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List

import numpy as np

MAGIC = 0x57524641
KIND_CONV, KIND_MAXPOOL, KIND_HEAD = 0, 1, 2
NORM_CHANNEL, NORM_GROUP, NORM_GROUP_LIVE = 0, 1, 2


@dataclass
class LayerSpec:
    kind: int
    c_in: int
    c_out: int
    k: int = 1
    stride: int = 1
    pad: int = 0
    relu: int = 0
    input_from: int = -1
    residual_from: int = -1


def resnet_layer_table(in_channels, stem_width, stem_k, blocks, widths) -> List[LayerSpec]:
    """Standard-ResNet reading B2: stem conv s2 + ReLU, maxpool k3 s2 p1, basic-block stages with
    stride 2 on the first conv of stages 2.. and a conv(k1, s2)+norm projection shortcut there."""
    t: List[LayerSpec] = []
    t.append(LayerSpec(KIND_CONV, in_channels, stem_width, stem_k, 2, stem_k // 2, 1, -1, -1))
    t.append(LayerSpec(KIND_MAXPOOL, stem_width, stem_width, 3, 2, 1, 0, 0, -1))
    x, c = 1, stem_width
    for si, (nb, w) in enumerate(zip(blocks, widths)):
        for bi in range(nb):
            stride = 2 if (si > 0 and bi == 0) else 1
            t.append(LayerSpec(KIND_CONV, c, w, 3, stride, 1, 1, x, -1))
            a = len(t) - 1
            if stride != 1 or c != w:
                t.append(LayerSpec(KIND_CONV, c, w, 1, stride, 0, 0, x, -1))
                res = len(t) - 1
            else:
                res = x
            t.append(LayerSpec(KIND_CONV, w, w, 3, 1, 1, 1, a, res))
            x, c = len(t) - 1, w
    t.append(LayerSpec(KIND_HEAD, c, 1, 1, 1, 0, 0, x, -1))
    return t


def tiny_config():
    """BASELINE.json configs[0]: stem k7 width 8, stages [1,1,1,1] widths 8/16/32/64, BN-style stats."""
    return dict(table=resnet_layer_table(2, 8, 7, [1, 1, 1, 1], [8, 16, 32, 64]),
                norm_kind=NORM_CHANNEL, n_groups=0, seed=0, kernel_len=2048)


def full_config():
    """BASELINE.json configs[1]: stem k7 width 64, stages [3,4,6,3] widths 64/128/256/512, GN(8)."""
    return dict(table=resnet_layer_table(2, 64, 7, [3, 4, 6, 3], [64, 128, 256, 512]),
                norm_kind=NORM_GROUP, n_groups=8, seed=1, kernel_len=3072)


def tiny_config_live_gn():
    """NEXT-2: the tiny network with true GroupNorm (8 groups, statistics per window at inference)."""
    return dict(table=resnet_layer_table(2, 8, 7, [1, 1, 1, 1], [8, 16, 32, 64]),
                norm_kind=NORM_GROUP_LIVE, n_groups=8, seed=2, kernel_len=2048)


def full_config_live_gn():
    """NEXT-2 at full size: the configs[1] network with true GroupNorm (8 groups, statistics per window)."""
    return dict(table=resnet_layer_table(2, 64, 7, [3, 4, 6, 3], [64, 128, 256, 512]),
                norm_kind=NORM_GROUP_LIVE, n_groups=8, seed=3, kernel_len=3072)


def make_weight_blob(table, norm_kind, n_groups, seed, eps=1e-5, in_channels=2, **_unused) -> bytes:
    """He-normal (fan-in) conv weights, frozen norm statistics (reading B6/B7), head w ~ N(0, 1/C)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    head = np.zeros(8, dtype=np.uint32)
    head[0], head[1], head[2], head[3], head[4] = MAGIC, 1, len(table), norm_kind, n_groups
    head[5] = np.float32(eps).view(np.uint32)
    head[6] = in_channels
    tab = np.zeros((len(table), 12), dtype=np.int32)
    payload = []
    for i, l in enumerate(table):
        tab[i, :9] = [l.kind, l.c_in, l.c_out, l.k, l.stride, l.pad, l.relu, l.input_from, l.residual_from]
        if l.kind == KIND_CONV:
            n_stat = l.c_out if norm_kind == NORM_CHANNEL else (n_groups if norm_kind == NORM_GROUP else 0)
            w = rng.standard_normal((l.c_out, l.c_in, l.k)) * np.sqrt(2.0 / (l.c_in * l.k))
            gamma = 1.0 + 0.1 * rng.standard_normal(l.c_out)
            beta = 0.1 * rng.standard_normal(l.c_out)
            mean = 0.1 * rng.standard_normal(n_stat)
            var = np.exp(0.2 * rng.standard_normal(n_stat))
            payload += [w.ravel(), gamma, beta, mean, var]
        elif l.kind == KIND_HEAD:
            w = rng.standard_normal(l.c_in) * np.sqrt(1.0 / l.c_in)
            payload += [w, np.zeros(1)]
    data = np.concatenate(payload).astype(np.float32) if payload else np.zeros(0, np.float32)
    return head.tobytes() + tab.tobytes() + data.tobytes()
