"""Host arithmetic of the incremental streaming network (aframe_describe_stream_plan; no GPU): the rows per layer that lie
within reach of a window's own zero padding, against the oracle-side pin of the same identity
(tests/test_oracle_network.py: reach 8/7, 12/11, 18/17, 15/14 at the stage ends) and against a brute-force
dependency walk written here from the conv definition."""
import numpy as np
import pytest

from synthdata import make_weight_blob, full_config, tiny_config


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


def brute_force_edges(table, kernel_len):
    """For every layer: which output rows depend, directly or through earlier layers, on a padded position.  A row set per
    layer, propagated row by row from the definition out[t] <- in[P t - pad + d], d < k (a residual adds the same row)."""
    dirty, T = [], []
    for l in table:
        kind, k, P, pad, src, res = l.kind, l.k, l.stride, l.pad, l.input_from, l.residual_from
        if kind == 2:
            break
        t_in = kernel_len if src < 0 else T[src]
        d_in = np.zeros(t_in, bool) if src < 0 else dirty[src]
        t_out = (t_in + 2 * pad - k) // P + 1
        d = np.zeros(t_out, bool)
        for t in range(t_out):
            for j in range(k):
                r = P * t - pad + j
                if r < 0 or r >= t_in or d_in[r]:
                    d[t] = True
        if res >= 0:
            d |= dirty[res]
        dirty.append(d)
        T.append(t_out)
    return dirty


@pytest.mark.parametrize("stride", [32, 64, 128])
def test_stream_plan_rows_equal_the_brute_force_reach_of_the_padding(af, stride):
    fc = full_config()
    plan = af.describe_stream_plan(make_weight_blob(**fc), kernel_len=fc["kernel_len"], stride=stride)
    dirty = brute_force_edges(fc["table"], fc["kernel_len"])
    assert len(plan) == len(dirty) == 37
    for i, (p, d) in enumerate(zip(plan, dirty)):
        assert p["t_out"] == len(d)
        head = int(np.argmin(d))                                 # first clean row = number of head rows
        tail = int(np.argmin(d[::-1]))
        assert d[:head].all() and d[len(d) - tail:].all() and not d[head:len(d) - tail].any()
        assert (p["head"], p["tail"]) == (head, tail), i
        samples_per_row = fc["kernel_len"] // p["t_out"]
        assert p["new"] * samples_per_row == stride
        if i >= 1:
            assert p["new"] + p["head"] + p["tail"] <= 48
    ends = [(plan[i]["head"], plan[i]["tail"]) for i in (7, 16, 29, 36)]
    assert ends == [(8, 7), (12, 11), (18, 17), (15, 14)]        # the values pinned on the oracle


def test_stream_plan_refuses_what_it_cannot_run(af):
    fc, tc = full_config(), tiny_config()
    blob = make_weight_blob(**fc)
    assert af.describe_stream_plan(blob, stride=512) == []       # 128 + 15 rows per update in the first stage
    assert af.describe_stream_plan(blob, stride=1) == [] and af.describe_stream_plan(blob, stride=48) == []
    assert af.describe_stream_plan(make_weight_blob(**tc), kernel_len=tc["kernel_len"], stride=128) == []   # widths 8/16/32/64
