"""GPU parity: batch_linear_lhs (Table 1) -- members that share ONE input X.  When every member of the
LHS group has N % 64 == 0 the planner logically concatenates the weights: the group is tiled as one [M, sum N]
problem whose tiles may span several members (composite tiles: the W tile is assembled from 64-row boxes of the
members' W, each 64-column chunk keeps its own bias / activation / output / FP8 copy).  The K order of every output
element is unchanged, so the result must equal the per-member schedule (opt_linear_options.no_lhs_order) BIT FOR BIT;
both are gated against the oracle."""
import numpy as np
import pytest
import torch

from oracle import graphs
import workloads as wl
from util import BF16, empty_dev, row_l2_rel_err, to_dev, to_host

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def lhs_group(seed, M, K, Ns, acts, bias_mask):
    x = wl.tensor_normal(seed, 1, (M, K), 0, 1, BF16)
    ms = []
    for i, (N, act, hb) in enumerate(zip(Ns, acts, bias_mask)):
        ms.append(dict(M=M, N=N, K=K, act=act, x=x, w=wl.tensor_normal(seed, 10 + 2 * i, (N, K), 0, K ** -0.5, BF16),
                       b=wl.tensor_normal(seed, 11 + 2 * i, (N,), 0, 0.2, BF16) if hb else None))
    return x, ms


def run(ob, x_dev, ms, options, concat, fp8_scale=None):
    dw = [to_dev(m["w"], BF16) for m in ms]
    db = [to_dev(m["b"], BF16) if m["b"] is not None else None for m in ms]
    M = ms[0]["M"]
    width = sum(m["N"] for m in ms)
    if concat:
        ycat = empty_dev((M, width), BF16, fill=float("nan"))
        off = np.concatenate(([0], np.cumsum([m["N"] for m in ms])))
        ys = [ycat[:, off[i]:off[i + 1]] for i in range(len(ms))]
    else:
        ys = [empty_dev((M, m["N"]), BF16, fill=float("nan")) for m in ms]
    y8s = [torch.full((M, m["N"]), 0xAA, dtype=torch.uint8, device="cuda") if fp8_scale and i % 2 == 0 else None for i, m in enumerate(ms)]
    descs = [ob.linear_member(x_dev, w, b, y, m["act"], 0, y8, fp8_scale or 0.0) for w, b, y, y8, m in zip(dw, db, ys, y8s, ms)]
    plan = ob.opt_linear_plan_create_ex(descs, BF16, 0, options)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    return [to_host(y) for y in ys], [None if q is None else q.cpu().numpy() for q in y8s], plan


@pytest.mark.parametrize("cta_pair", [0, 1])
@pytest.mark.parametrize("case", [
    dict(M=1000, K=512, Ns=[64] * 8, concat=True),                       # the side workload's shape class: 8 x N=64
    dict(M=300, K=72, Ns=[64, 128, 192, 64, 320], concat=False),         # chunks of several members in one tile, ragged M and K
    dict(M=513, K=256, Ns=[64, 64, 64], concat=True),                    # 3 chunks: one 192-wide tile (96 W rows per CTA of a pair)
    dict(M=257, K=128, Ns=[1024, 64], concat=False),                     # a wide member followed by a narrow one
])
def test_concatenated_weights_equal_the_per_member_schedule_bitwise(ob, case, cta_pair):
    n = len(case["Ns"])
    x, ms = lhs_group(91, case["M"], case["K"], case["Ns"], [i % 4 for i in range(n)], [i % 3 != 2 for i in range(n)])
    xd = to_dev(x, BF16)
    fused, q_fused, pf = run(ob, xd, ms, ob.opt_linear_options(cta_pair=cta_pair), case["concat"], fp8_scale=4.0)
    plain, q_plain, pp = run(ob, xd, ms, ob.opt_linear_options(cta_pair=cta_pair, no_lhs_order=1), case["concat"], fp8_scale=4.0)
    assert pf.info()["tiles"] <= pp.info()["tiles"]                   # fewer, wider tiles
    assert pf.info()["bytes"] == pp.info()["bytes"] and pf.info()["flops"] == pp.info()["flops"]
    for a, b, qa, qb, m in zip(fused, plain, q_fused, q_plain, ms):
        assert a.tobytes() == b.tobytes()
        assert (qa is None and qb is None) or np.array_equal(qa, qb)
        assert row_l2_rel_err(a, graphs.linear_member(m, BF16), BF16) <= 1e-2


def test_lhs_group_with_an_unaligned_member_falls_back_to_lhs_order(ob):
    """N % 64 != 0 somewhere in the group: no concatenation (per-member tiles, m-block-major order), same results."""
    x, ms = lhs_group(92, 400, 96, [64, 72, 128], [1, 0, 2], [True, True, False])
    xd = to_dev(x, BF16)
    a, _, pa = run(ob, xd, ms, ob.opt_linear_options(), False)
    b, _, pb = run(ob, xd, ms, ob.opt_linear_options(no_lhs_order=1), False)
    assert pa.info()["tiles"] == pb.info()["tiles"]
    for u, v, m in zip(a, b, ms):
        assert u.tobytes() == v.tobytes()
        assert row_l2_rel_err(u, graphs.linear_member(m, BF16), BF16) <= 1e-2


def test_two_lhs_groups_and_loose_members_in_one_launch(ob):
    """a group with two different shared inputs plus members with their own input: one launch, integers bit-exact."""
    rng = np.random.default_rng(17)
    conv = lambda a: wl.bf16_bits_from_f32(a.astype(np.float32))
    xa, xb = conv(rng.integers(-2, 3, (300, 48))), conv(rng.integers(-2, 3, (200, 16)))
    ms = []
    for x, Ns in ((xa, [64, 64, 128]), (xb, [128, 64])):
        for N in Ns:
            ms.append(dict(M=x.shape[0], N=N, K=x.shape[1], act=len(ms) % 2, x=x, w=conv(rng.integers(-1, 2, (N, x.shape[1]))),
                           b=conv(rng.integers(-2, 3, (N,)))))
    xl = conv(rng.integers(-2, 3, (130, 24)))
    ms.append(dict(M=130, N=40, K=24, act=1, x=xl, w=conv(rng.integers(-1, 2, (40, 24))), b=None))
    xs = {id(xa): to_dev(xa, BF16), id(xb): to_dev(xb, BF16), id(xl): to_dev(xl, BF16)}
    keep, descs, ys = [], [], []
    for m in ms:
        w = to_dev(m["w"], BF16)
        b = to_dev(m["b"], BF16) if m["b"] is not None else None
        y = empty_dev((m["M"], m["N"]), BF16, fill=float("nan"))
        keep.append((w, b)); ys.append(y)
        descs.append(ob.linear_member(xs[id(m["x"])], w, b, y, m["act"]))
    n0 = ob.opt_launch_count()
    ob.opt_linear_plan_create(descs, BF16).launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    _, ref = graphs.linear_group(ms, BF16)
    for y, r in zip(ys, ref):
        assert to_host(y).tobytes() == r.tobytes()


def test_relaunch_and_cuda_graph_replay_of_a_composite_fp8_plan(ob):
    """the plan re-arms its scheduler counters at the end of every launch: relaunches and CUDA-graph replays of a plan
    with composite tiles and FP8 copies give the same bits."""
    x, ms = lhs_group(93, 700, 200, [64, 128, 64, 256, 64], [0, 1, 2, 3, 1], [True] * 5)
    xd = to_dev(x, BF16)
    outs, q8, plan = run(ob, xd, ms, ob.opt_linear_options(), True, fp8_scale=2.0)
    first = b"".join(o.tobytes() for o in outs) + b"".join(q.tobytes() for q in q8 if q is not None)
    # `run` keeps no handle on its device buffers, so rebuild a plan whose buffers we own
    dw = [to_dev(m["w"], BF16) for m in ms]
    db = [to_dev(m["b"], BF16) for m in ms]
    ycat = empty_dev((700, sum(m["N"] for m in ms)), BF16, fill=float("nan"))
    off = np.concatenate(([0], np.cumsum([m["N"] for m in ms])))
    y8 = [torch.full((700, m["N"]), 0xAA, dtype=torch.uint8, device="cuda") if i % 2 == 0 else None for i, m in enumerate(ms)]
    plan = ob.opt_linear_plan_create([ob.linear_member(xd, w, b, ycat[:, off[i]:off[i + 1]], m["act"], 0, y8[i], 2.0)
                                      for i, (w, b, m) in enumerate(zip(dw, db, ms))], BF16)
    snap = lambda: b"".join(to_host(ycat[:, off[i]:off[i + 1]]).tobytes() for i in range(len(ms))) + \
        b"".join(q.cpu().numpy().tobytes() for q in y8 if q is not None)
    for _ in range(3):
        ycat.fill_(float("nan"))
        plan.launch()
        torch.cuda.synchronize()
        assert snap() == first
    g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.graph(g, stream=s):
        plan.launch(s.cuda_stream)
    for _ in range(2):
        ycat.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        assert snap() == first


def test_stress_many_lhs_groups_random_shapes_against_single_member_plans(ob):
    """60 members over 6 shared inputs (+ loose ones), random N (aligned and unaligned to 64), activations, bias on / off,
    FP8 copies on / off, ragged M and K: ONE launch must equal, bit for bit, the same members run as single-member plans."""
    rng = np.random.default_rng(23)
    conv = lambda a: wl.bf16_bits_from_f32(a.astype(np.float32))
    members, xs = [], []
    for gidx in range(6):
        M, K = int(rng.integers(1, 700)), int(rng.choice([8, 24, 64, 72, 128, 200, 320]))
        aligned = gidx % 2 == 0
        xs.append(to_dev(wl.tensor_normal(300 + gidx, 1, (M, K), 0, 1, BF16), BF16))
        for j in range(int(rng.integers(2, 12))):
            N = int(rng.choice([64, 128, 192, 256, 320])) if aligned else int(rng.choice([16, 40, 64, 104, 128, 264]))
            members.append(dict(xi=gidx, M=M, K=K, N=N, act=int(rng.integers(0, 4)), bias=bool(rng.integers(0, 2)),
                                fp8=bool(rng.integers(0, 2)) and N % 16 == 0))
    rng.shuffle(members)                                       # members of a group need not be adjacent in the descriptor array
    dev, fused, singles = [], [], []
    for i, m in enumerate(members):
        w = to_dev(wl.tensor_normal(400, 2 * i, (m["N"], m["K"]), 0, m["K"] ** -0.5, BF16), BF16)
        b = to_dev(wl.tensor_normal(400, 2 * i + 1, (m["N"],), 0, 0.2, BF16), BF16) if m["bias"] else None
        ya, yb = (empty_dev((m["M"], m["N"]), BF16, fill=float("nan")) for _ in range(2))
        qa, qb = ((torch.full((m["M"], m["N"]), 0xAA, dtype=torch.uint8, device="cuda") if m["fp8"] else None) for _ in range(2))
        dev.append((w, b, ya, yb, qa, qb))
        fused.append(ob.linear_member(xs[m["xi"]], w, b, ya, m["act"], 0, qa, 3.0))
        singles.append(ob.linear_member(xs[m["xi"]], w, b, yb, m["act"], 0, qb, 3.0))
    n0 = ob.opt_launch_count()
    ob.opt_linear_plan_create(fused, BF16).launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    for d in singles:
        ob.opt_linear_plan_create([d], BF16).launch()
    torch.cuda.synchronize()
    for (w, b, ya, yb, qa, qb), m in zip(dev, members):
        assert torch.equal(ya.view(torch.int16), yb.view(torch.int16)), m
        assert qa is None or torch.equal(qa, qb), m
        assert not torch.isnan(ya.float()).any()
