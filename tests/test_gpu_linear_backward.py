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
