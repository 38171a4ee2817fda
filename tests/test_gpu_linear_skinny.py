"""GPU parity: grouped Linear on SKINNY members (huge M, K in {4,8,16}, N in {2,..,16}) -- the run-time residue of
decompose_mm_pass, SURVEY.md 8(f) rank 4 -- vs the CPU oracle, through the C ABI.  The same
opt_linear_plan_create entry point routes such a group to the streaming row kernel."""
import numpy as np
import pytest
import torch

import oracle
from oracle import graphs
import workloads as wl
from util import BF16, bf16_ulp_distance, empty_dev, row_l2_rel_err, to_dev, to_host

from test_gpu_linear import int_member, mk

pytestmark = pytest.mark.gpu

COMBOS = [(4, 2), (4, 4), (4, 8), (4, 16), (8, 2), (8, 4), (8, 8), (8, 16), (16, 2), (16, 4), (16, 8)]     # (K, N)


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def run(ob, members, pad_x=0, pad_y=0):
    """dense tensors (ld = K / N: the paper's [M, 4] x [4, 2] layout) unless a pad is given."""
    dev, descs = [], []
    for m in members:
        x = to_dev(np.pad(m["x"], ((0, 0), (0, pad_x))), BF16)[:, :m["K"]]
        w = to_dev(m["w"], BF16)
        b = None if m["b"] is None else to_dev(np.pad(m["b"], (0, (-m["N"]) % 8)), BF16)[:m["N"]]
        y = empty_dev((m["M"], m["N"] + pad_y), BF16, fill=float("nan"))
        dev.append((x, w, b, y))
        descs.append(ob.linear_member(x, w, b, y[:, :m["N"]], m["act"]))
    plan = ob.opt_linear_plan_create(descs, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1 and plan.info()["launches"] == 1
    return [to_host(d[3]) for d in dev], plan


def test_small_integers_bit_exact_every_shape(ob):
    rng = np.random.default_rng(31)
    members = [int_member(rng, 3000 + 37 * i, N, K, 3, act=i % 2) for i, (K, N) in enumerate(COMBOS)]
    outs, _ = run(ob, members)
    _, ref = graphs.linear_group(members, BF16)
    for got, r, m in zip(outs, ref, members):
        assert got[:, :m["N"]].tobytes() == r.tobytes(), (m["K"], m["N"])


def test_random_all_shapes_activations_ragged_rows(ob):
    """every (K, N), every activation, with / without bias, M not a multiple of the 1024-row block, strided rows with
    untouched padding; row-L2 <= 1e-2 (north_star) and <= 2 bf16 ulp per element (K <= 16: fp32 sums are near exact)."""
    members = [mk(81, i, 5000 + 211 * i, N, K, act=i % 4, bias=i % 3 != 0) for i, (K, N) in enumerate(COMBOS)]
    members += [mk(81, 20, 1, 8, 8, 1), mk(81, 21, 1023, 2, 4, 0), mk(81, 22, 1025, 16, 8, 2), mk(81, 23, 8193, 8, 8, 0), mk(81, 24, 20000, 4, 16, 1)]
    for pad_x, pad_y in ((0, 0), (8, 16), (2, 6)):
        outs, plan = run(ob, members, pad_x, pad_y)
        z64, _ = graphs.linear_group(members, BF16)
        for got, z, m in zip(outs, z64, members):
            assert row_l2_rel_err(got[:, :m["N"]], z, BF16) <= 1e-2
            assert bf16_ulp_distance(got[:, :m["N"]], oracle.round_to_storage(z, BF16)).max() <= 2
            if pad_y:
                assert np.all((got[:, m["N"]:] & 0x7FFF) > 0x7F80)                # padding columns still NaN


def test_paper_shapes_scaled_and_equal_to_tensor_core_path(ob):
    """the paper's model-type-B group ([M,8]x[8,8], [M,4]x[4,2], twice; M scaled down 64x) in one launch; the 8x8
    members also through the tensor-core kernel (forced by adding a non-skinny member to the group): same result
    to within 1 bf16 ulp (both accumulate in fp32; the summation order differs)."""
    shapes = [(290372, 8, 8), (394499, 2, 4), (351595, 8, 8), (280939, 2, 4)]
    members = [mk(82, i, M, N, K, 0, bias=False) for i, (M, N, K) in enumerate(shapes)]
    outs, plan = run(ob, members)
    z64, _ = graphs.linear_group(members, BF16)
    for got, z in zip(outs, z64):
        assert row_l2_rel_err(got, z, BF16) <= 1e-2
    big = [m for m in members if m["K"] == 8] + [mk(82, 9, 256, 64, 64, 0)]
    dev, descs = [], []
    for m in big:
        x, w = to_dev(m["x"], BF16), to_dev(m["w"], BF16)
        y = empty_dev((m["M"], m["N"]), BF16)
        dev.append(y)
        descs.append(ob.linear_member(x, w, None, y, 0))
    ob.opt_linear_plan_create(descs, BF16).launch()
    torch.cuda.synchronize()
    for y, got in zip(dev[:2], [outs[0], outs[2]]):
        assert bf16_ulp_distance(to_host(y), got).max() <= 1


def test_alignment_rules(ob):
    x = empty_dev((64, 12), BF16, fill=1.0)
    w = empty_dev((2, 4), BF16, fill=1.0)
    y = empty_dev((64, 2), BF16)
    ob.opt_linear_plan_create([ob.linear_member(x[:, :4], w, None, y, 0)], BF16)          # ldx = 12: even
    ob.opt_linear_plan_create([ob.linear_member(empty_dev((64, 10), BF16)[:, :4], w, None, y, 0)], BF16)
    with pytest.raises(ob.OptError) as e:
        ob.opt_linear_plan_create([ob.linear_member(empty_dev((64, 11), BF16)[:, :4], w, None, y, 0)], BF16)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
    with pytest.raises(ob.OptError) as e:          # mixed with a non-skinny member the tensor-core rules apply (ld % 8)
        big = ob.linear_member(empty_dev((64, 64), BF16), empty_dev((64, 64), BF16), None, empty_dev((64, 64), BF16), 0)
        ob.opt_linear_plan_create([ob.linear_member(x[:, :4], w, None, y, 0), big], BF16)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
