"""GPU parity: backward of the grouped Linear through the same grouped GEMM kernel with operands read in their
stored (transposed) layout -- dgrad dX = dY W, wgrad dW = dY^T X."""
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


def run_backward(ob, members):
    """members: dicts with dy [M,N], w [N,K], x [M,K] (bf16 bits).  One launch for all dgrads, one for all wgrads."""
    dev, dg, wg = [], [], []
    for m in members:
        M, N = m["dy"].shape
        K = m["w"].shape[1]
        dy, w, x = to_dev(m["dy"], BF16), to_dev(m["w"], BF16), to_dev(m["x"], BF16)
        dx = empty_dev((M, K), BF16, fill=float("nan"))
        dw = empty_dev((N, K), BF16, fill=float("nan"))
        dev.append((dy, w, x, dx, dw))
        # dgrad: out [M,K], contraction N: "x" = dY [M,N] (K-major), "w" = W stored [N(contraction), K]: transposed
        dg.append(ob.linear_member(dy, w, None, dx, 0, ob.OPT_LAYOUT_W_TRANSPOSED))
        # wgrad: out [N,K], contraction M: "x" = dY stored [M(contraction), N], "w" = X stored [M(contraction), K]
        wg.append(ob.linear_member(dy, x, None, dw, 0, ob.OPT_LAYOUT_X_TRANSPOSED | ob.OPT_LAYOUT_W_TRANSPOSED))
    n0 = ob.opt_launch_count()
    ob.opt_linear_plan_create(dg, BF16).launch()
    ob.opt_linear_plan_create(wg, BF16).launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 2
    return [(to_host(d[3]), to_host(d[4])) for d in dev]


def test_integers_bit_exact(ob):
    rng = np.random.default_rng(33)
    conv = lambda a: wl.bf16_bits_from_f32(a.astype(np.float32))
    members = []
    for (M, N, K) in [(128, 64, 64), (64, 64, 128), (200, 48, 40), (257, 136, 72), (5, 8, 16), (1000, 256, 264), (96, 304, 24)]:
        members.append(dict(dy=conv(rng.integers(-1, 2, (M, N))), w=conv(rng.integers(-1, 2, (N, K))), x=conv(rng.integers(-1, 2, (M, K)))))
    outs = run_backward(ob, members)
    for (dx, dw), m in zip(outs, members):
        rdx = graphs.linear_dgrad(m["dy"], m["w"])
        rdw = graphs.linear_wgrad(m["dy"], m["x"])
        assert np.abs(rdx).max() < 256 and np.abs(rdw).max() <= 1000          # dgrad exact in bf16; wgrad may round
        assert np.array_equal(wl.f32_from_bf16_bits(dx).astype(np.float64), rdx), m["dy"].shape
        from oracle import round_to_storage
        assert dw.tobytes() == round_to_storage(rdw, BF16).tobytes(), m["dy"].shape


@pytest.mark.parametrize("seed", [5, 105])
def test_random_towers(ob, seed):
    rng = np.random.default_rng(seed)
    members = []
    for i in range(12):
        M, N, K = int(rng.choice([300, 512, 1000])), int(rng.choice([64, 128, 256, 520])), int(rng.choice([32, 128, 256, 1024]))
        members.append(dict(dy=wl.tensor_normal(seed, 4 * i + 1, (M, N), 0, 1, BF16), w=wl.tensor_normal(seed, 4 * i + 2, (N, K), 0, K ** -0.5, BF16),
                            x=wl.tensor_normal(seed, 4 * i + 3, (M, K), 0, 1, BF16)))
    outs = run_backward(ob, members)
    for (dx, dw), m in zip(outs, members):
        assert row_l2_rel_err(dx, graphs.linear_dgrad(m["dy"], m["w"]), BF16) <= 1e-2
        assert row_l2_rel_err(dw, graphs.linear_wgrad(m["dy"], m["x"]), BF16) <= 1e-2


def test_relu_backward_group_bit_exact(ob):
    """OPT_PW_RELU_BWD: the gradient masks of N ReLU epilogues in ONE launch -- dense members, column slices of a
    concat buffer, fp32, both zeros in the mask: bit-exact against the oracle (no arithmetic, only a select)."""
    import oracle
    from util import F32
    rng = np.random.default_rng(91)
    shapes = [(300, 512), (77, 200), (1000, 64), (129, 1032), (64, 8), (5, 4096)]
    W = sum(w for _, w in shapes)
    chunks, host, keep = [], [], []
    for i, (r, w) in enumerate(shapes):
        g = wl.tensor_normal(91, 2 * i + 1, (r, w), 0.0, 2.0, BF16)
        y = wl.tensor_normal(91, 2 * i + 2, (r, w), 0.0, 1.0, BF16).copy()
        y[(y & 0x8000) != 0] = 0x8000 if i % 2 else 0x0000        # what a ReLU leaves: 0 (or -0) where x <= 0
        y.reshape(-1)[::53] = 0x8000
        pad = 24 if i % 2 else 0                                  # odd members: slices of wider buffers
        dg = to_dev(np.pad(g, ((0, 0), (0, pad))), BF16)[:, :w]
        dy = to_dev(np.pad(y, ((0, 0), (8, pad))), BF16)[:, 8:8 + w]
        dd = empty_dev((r, w + pad), BF16, fill=float("nan"))[:, :w]
        chunks.append(ob.chunk(dg, dd, ob.OPT_PW_RELU_BWD, dy))
        host.append((g, y)); keep.append((dg, dy, dd))
    plan = ob.opt_pointwise_plan_create(chunks, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    for (g, y), (_, _, dd) in zip(host, keep):
        ref = oracle.round_to_storage(oracle.pointwise_ext(g, y, oracle.PW_RELU_BWD, [], BF16), BF16)
        assert to_host(dd).tobytes() == ref.tobytes()
    # fp32, in place on the gradient
    g = wl.tensor_normal(92, 1, (100, 36), 0, 2, F32); y = np.maximum(wl.tensor_normal(92, 2, (100, 36), 0, 1, F32), np.float32(0))
    dg, dy = to_dev(g, F32), to_dev(y, F32)
    ob.opt_pointwise_plan_create([ob.chunk(dg, dg, ob.OPT_PW_RELU_BWD, dy)], F32).launch()
    torch.cuda.synchronize()
    assert np.array_equal(to_host(dg), oracle.round_to_storage(oracle.pointwise_ext(g, y, oracle.PW_RELU_BWD, [], F32), F32))


def test_full_backward_of_a_linear_relu_group(ob):
    """Forward Y_i = relu(X_i W_i^T + b_i) (one launch), then the whole backward in three launches: the ReLU masks
    of all members, all dgrads, all wgrads -- against the oracle run one op at a time on the same forward output."""
    import oracle
    members = []
    for i, (M, N, K) in enumerate([(300, 128, 64), (512, 64, 256), (1000, 256, 128), (257, 136, 72)]):
        members.append(dict(x=wl.tensor_normal(7, 4 * i + 1, (M, K), 0, 1, BF16), w=wl.tensor_normal(7, 4 * i + 2, (N, K), 0, K ** -0.5, BF16),
                            b=wl.tensor_normal(7, 4 * i + 3, (N,), 0, 0.1, BF16), g=wl.tensor_normal(7, 4 * i + 4, (M, N), 0, 1, BF16)))
    dev, fwd, msk, dg, wg = [], [], [], [], []
    for m in members:
        (M, K), N = m["x"].shape, m["w"].shape[0]
        x, w, b, g = (to_dev(m[k], BF16) for k in ("x", "w", "b", "g"))
        y, dz = empty_dev((M, N), BF16), empty_dev((M, N), BF16, fill=float("nan"))
        dx, dw = empty_dev((M, K), BF16, fill=float("nan")), empty_dev((N, K), BF16, fill=float("nan"))
        dev.append((x, w, b, g, y, dz, dx, dw))
        fwd.append(ob.linear_member(x, w, b, y, ob.OPT_ACT_RELU))
        msk.append(ob.chunk(g, dz, ob.OPT_PW_RELU_BWD, y))
        dg.append(ob.linear_member(dz, w, None, dx, 0, ob.OPT_LAYOUT_W_TRANSPOSED))
        wg.append(ob.linear_member(dz, x, None, dw, 0, ob.OPT_LAYOUT_X_TRANSPOSED | ob.OPT_LAYOUT_W_TRANSPOSED))
    n0 = ob.opt_launch_count()
    ob.opt_linear_plan_create(fwd, BF16).launch()
    ob.opt_pointwise_plan_create(msk, BF16).launch()
    ob.opt_linear_plan_create(dg, BF16).launch()
    ob.opt_linear_plan_create(wg, BF16).launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 4
    for m, d in zip(members, dev):
        y = to_host(d[4])                                          # the mask source both sides use: the stored forward output
        dz = oracle.round_to_storage(oracle.pointwise_ext(m["g"], y, oracle.PW_RELU_BWD, [], BF16), BF16)
        assert to_host(d[5]).tobytes() == dz.tobytes()
        assert 0.2 < np.mean(dz == 0) < 0.8                        # the mask really cuts about half
        assert row_l2_rel_err(to_host(d[6]), graphs.linear_dgrad(dz, m["w"]), BF16) <= 1e-2
        assert row_l2_rel_err(to_host(d[7]), graphs.linear_wgrad(dz, m["x"]), BF16) <= 1e-2


def test_tanh_sigmoid_relu_backward_mixed_group(ob):
    """OPT_PW_TANH_BWD / OPT_PW_SIGMOID_BWD / OPT_PW_RELU_BWD members in ONE launch, the stored output y taken from the
    ORACLE's forward (rounded to bf16, so saturated +-1 / 0 / 1 occur): <= 2 bf16 ulp of the oracle (fp32 arithmetic,
    one rounding: 1 - y^2 and (1 - y) y are exact or 2^-24-accurate for a bf16 y); dense members and column slices."""
    import oracle
    from util import bf16_ulp_distance
    ops = [(ob.OPT_PW_TANH_BWD, oracle.PW_TANH_BWD, 2), (ob.OPT_PW_SIGMOID_BWD, oracle.PW_SIGMOID_BWD, 3), (ob.OPT_PW_RELU_BWD, oracle.PW_RELU_BWD, 1)]
    shapes = [(300, 512), (77, 200), (1000, 64), (129, 1032), (64, 8), (5, 4096)]
    chunks, host, keep = [], [], []
    for i, (r, w) in enumerate(shapes):
        op, oop, act = ops[i % 3]
        g = wl.tensor_normal(93, 2 * i + 1, (r, w), 0.0, 2.0, BF16)
        z = wl.tensor_normal(93, 2 * i + 2, (r, w), 0.0, 3.0, BF16)
        y = oracle.round_to_storage(oracle.pointwise(z, act, BF16), BF16)
        pad = 24 if i % 2 else 0
        dg = to_dev(np.pad(g, ((0, 0), (0, pad))), BF16)[:, :w]
        dy = to_dev(np.pad(y, ((0, 0), (8, pad))), BF16)[:, 8:8 + w]
        dd = empty_dev((r, w + pad), BF16, fill=float("nan"))[:, :w]
        chunks.append(ob.chunk(dg, dd, op, dy))
        host.append((g, y, oop)); keep.append((dg, dy, dd))
    plan = ob.opt_pointwise_plan_create(chunks, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    for (g, y, oop), (_, _, dd) in zip(host, keep):
        ref = oracle.round_to_storage(oracle.pointwise_ext(g, y, oop, [], BF16), BF16)
        d = bf16_ulp_distance(to_host(dd), ref)
        assert d.max() <= 2, (oop, int(d.max()))
    # fp32 storage: relative to the gradient, a few fp32 roundings
    from util import F32
    for op, oop, act in ops[:2]:
        g = wl.tensor_normal(94, 1, (100, 36), 0, 2, F32)
        y = oracle.round_to_storage(oracle.pointwise(wl.tensor_normal(94, 2, (100, 36), 0, 2, F32), act, F32), F32)
        dg, dy, dd = to_dev(g, F32), to_dev(y, F32), empty_dev((100, 36), F32, fill=float("nan"))
        ob.opt_pointwise_plan_create([ob.chunk(dg, dd, op, dy)], F32).launch()
        torch.cuda.synchronize()
        ref = oracle.pointwise_ext(g, y, oop, [], F32)
        assert np.all(np.abs(to_host(dd).astype(np.float64) - ref) <= 4e-7 * np.abs(g.astype(np.float64)))


@pytest.mark.parametrize("act", [2, 3])
def test_whole_backward_of_a_linear_tanh_sigmoid_group(ob, act):
    """Forward Y_i = act(X_i W_i^T + b_i) (one launch), then the backward in four launches -- activation derivative
    from the stored output, bias gradients, dgrads, wgrads -- against graphs.linear_act_backward, which runs its own
    fp64 forward.  The derivative is smooth in y, so the 2-ulp difference of the two forwards stays inside the GEMM
    tolerance: dz rows, dX rows, dW rows <= 1e-2 row-L2; db within 1e-2 of the column's sum |dz|."""
    from util import F32, values64
    members = []
    for i, (M, N, K) in enumerate([(300, 128, 64), (512, 64, 256), (1000, 256, 128), (257, 136, 72)]):
        members.append(dict(x=wl.tensor_normal(9, 4 * i + 1, (M, K), 0, 1, BF16), w=wl.tensor_normal(9, 4 * i + 2, (N, K), 0, K ** -0.5, BF16),
                            b=wl.tensor_normal(9, 4 * i + 3, (N,), 0, 0.1, BF16), g=wl.tensor_normal(9, 4 * i + 4, (M, N), 0, 1, BF16)))
    dev, fwd, der, bg, dg, wg = [], [], [], [], [], []
    for m in members:
        (M, K), N = m["x"].shape, m["w"].shape[0]
        x, w, b, g = (to_dev(m[k], BF16) for k in ("x", "w", "b", "g"))
        y, dz = empty_dev((M, N), BF16), empty_dev((M, N), BF16, fill=float("nan"))
        dx, dw, db = empty_dev((M, K), BF16, fill=float("nan")), empty_dev((N, K), BF16, fill=float("nan")), empty_dev((N,), F32, fill=float("nan"))
        dev.append((dz, dx, dw, db))
        fwd.append(ob.linear_member(x, w, b, y, ob.OPT_ACT_TANH if act == 2 else ob.OPT_ACT_SIGMOID))
        der.append(ob.chunk(g, dz, ob.OPT_PW_TANH_BWD if act == 2 else ob.OPT_PW_SIGMOID_BWD, y))
        bg.append(ob.bias_grad_member(dz, db))
        dg.append(ob.linear_member(dz, w, None, dx, 0, ob.OPT_LAYOUT_W_TRANSPOSED))
        wg.append(ob.linear_member(dz, x, None, dw, 0, ob.OPT_LAYOUT_X_TRANSPOSED | ob.OPT_LAYOUT_W_TRANSPOSED))
        dev[-1] += (x, w, b, g, y)
    n0 = ob.opt_launch_count()
    ob.opt_linear_plan_create(fwd, BF16).launch()
    ob.opt_pointwise_plan_create(der, BF16).launch()
    ob.opt_bias_grad_plan_create(bg, BF16, F32).launch()
    ob.opt_linear_plan_create(dg, BF16).launch()
    ob.opt_linear_plan_create(wg, BF16).launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 5
    for m, d in zip(members, dev):
        r = graphs.linear_act_backward(m, m["g"], act, BF16)
        assert row_l2_rel_err(to_host(d[0]), values64(r["dz"], BF16), BF16) <= 1e-2
        l1 = np.abs(values64(r["dz"], BF16)).sum(axis=0)
        assert np.all(np.abs(to_host(d[3]).astype(np.float64) - r["db64"]) <= 1e-2 * l1)
        assert row_l2_rel_err(to_host(d[1]), r["dx64"], BF16) <= 1e-2
        assert row_l2_rel_err(to_host(d[2]), r["dw64"], BF16) <= 1e-2
