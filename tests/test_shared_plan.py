"""CPU-only tests of the shared-stage planner (aframe_describe_shared_plan: host arithmetic of csrc/conv_tc.cu, no device).

The packed edge batch deliberately computes boxes whose trailing tile rows are stale shared memory and whose last box of
a half overhangs into spare slots, so its slot / overhang arithmetic is checked here for every window length and spacing
the library accepts, without a GPU; the edge reach itself is pinned on the float64 oracle in test_oracle_network.py
(8/7, 12/11, 18/17, 15/14 rows at the stage ends for BASELINE.json configs[1])."""
import numpy as np
import pytest

from synthdata import full_config, make_weight_blob


@pytest.fixture(scope="module")
def af():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    return af


@pytest.fixture(scope="module")
def blob():
    return make_weight_blob(**full_config())


def test_config1_plan_is_the_documented_one(af, blob):
    s1, st = af.describe_shared_plan(blob, 3072, 2, 128, 4096)
    assert s1 == 3                                               # three fused 64-channel blocks: edge 2k+2 / 2k+1 = 8 / 7 rows
    assert [(d["T"], d["C"], d["head"], d["tail"], d["packed"]) for d in st] == [
        (384, 128, 12, 11, True), (192, 256, 18, 17, True), (96, 512, 15, 14, True)]
    # a box holds the edge rows only (at least 4); a slot also holds the two stream rows next to them, except in the last layer
    # (a packed stage that feeds a packed stage holds, in its slots, the rows the next stage's first two layers reach: 2 x
    #  their second box, read in place)
    assert st[0]["tbox"] == [5, 6, 7, 8, 9, 10, 11, 12] and st[0]["P"] == 16
    assert st[0]["e_head"] == list(range(5, 13)) and st[0]["e_tail"] == list(range(4, 12))
    assert st[1]["tbox"] == [7, 8, 9, 10, 11, 12, 13, 14, 15, 16, 17, 18] and st[1]["P"] == 22
    assert st[2]["tbox"] == [10, 11, 12, 13, 14, 15] and st[2]["P"] == 16
    assert st[1]["e_head"] == list(range(7, 19)) and st[1]["e_tail"] == list(range(6, 18))
    assert st[2]["e_head"] == list(range(10, 16)) and st[2]["e_tail"] == list(range(9, 15))
    assert all(d["spare_slots"] == 32 for d in st)


@pytest.mark.parametrize("spacing", [4, 8, 16, 32, 64, 100, 128, 256, 384, 512, 1024, 3072, 4096])
def test_packed_edge_invariants_for_every_window_length(af, blob, spacing):
    """For every window length the tensor-core path accepts (every stage's length needs a power-of-two factor >= 8, so the
    window is a multiple of 256 samples; 512 .. 8192) and many it refuses, at this spacing: whatever the planner decides to
    share or pack obeys the row and slot arithmetic the kernels rely on."""
    n_planned = 0
    for kernel_len in range(512, 8192 + 1, 32):
        for n_windows in (2, 37, 4096):
            s1, st = af.describe_shared_plan(blob, kernel_len, 2, spacing, n_windows)
            if spacing >= kernel_len or spacing % 4:
                assert s1 == 0 and st == []                      # windows do not overlap / the stem's rows do not line up
                continue
            assert 0 <= s1 <= 5
            prev_T = kernel_len // 4
            for si, d in enumerate(st):
                # rows taken from one end of a window must be out of reach of the padding at the other end
                assert d["T"] * 2 == prev_T and d["head"] >= 1 and d["tail"] >= 1 and d["head"] + d["tail"] <= d["T"]
                prev_T = d["T"]
                if not d["packed"]:
                    assert d["P"] >= max(d["head"], d["tail"]) and 2 * d["P"] <= 2 * d["T"]
                    continue
                n_planned += 1
                nl = d["n_layers"]
                eh, et, tb = d["e_head"], d["e_tail"], d["tbox"]
                assert eh == list(range(eh[0], eh[0] + nl)) and et == list(range(et[0], et[0] + nl))   # one more row per conv
                assert eh[-1] == d["head"] and et[-1] == d["tail"]
                slot_rows = []
                for q in range(nl):
                    assert tb[q] == max(eh[q], et[q], 4)
                    assert 1 <= tb[q] <= 32
                    # the slot: the box, and (all layers but the last) the two stream rows past the edge rows
                    slot_rows.append(max(tb[q], max(eh[q], et[q]) + 2) if q + 1 < nl else tb[q])
                    boxes_per_tile = 128 // tb[q]
                    assert boxes_per_tile >= 4
                    # the last box of a half starts inside the windows and covers boxes_per_tile slots: overhang < spare slots
                    assert boxes_per_tile <= d["spare_slots"]
                    n_boxes = -(-n_windows // boxes_per_tile)
                    assert n_boxes * boxes_per_tile - n_windows < d["spare_slots"] + 1
                # ... or, if a packed stage follows, the rows its entry conv and folded projection reach (an even number)
                nxt = st[si + 1] if si + 1 < len(st) and st[si + 1]["packed"] else None
                p_in = 2 * (nxt["tbox"][1] if nxt["n_layers"] > 1 else nxt["tbox"][0] + 1) if nxt else 0
                want = max(max(slot_rows), p_in)
                assert d["P"] in (max(slot_rows), want + (want & 1)) and d["T"] >= 2 * d["P"]  # a window's two slots never overlap
    if spacing in (32, 64, 128, 512):
        assert n_planned > 100


def test_plan_refuses_bad_input(af, blob):
    with pytest.raises(af.AframeError) as e:
        af.describe_shared_plan(blob[:100], 3072, 2, 128, 4096)
    assert e.value.status == af.ESHAPE
    with pytest.raises(af.AframeError) as e:
        af.describe_shared_plan(blob, 3072, 3, 128, 4096)        # wrong channel count for this table
    assert e.value.status == af.ESHAPE
    with pytest.raises(af.AframeError) as e:
        af.describe_shared_plan(blob, 3072, 2, 0, 4096)
    assert e.value.status == af.EINVAL
