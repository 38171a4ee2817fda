"""GPU parity under many small, randomly shaped members: hundreds of members per launch, every shape class the
planners distinguish (tile tails, lane mappings, staged / direct / extended pointwise groups), one launch each,
every member compared with the CPU oracle."""
import numpy as np
import pytest
import torch

import oracle
from oracle import graphs
import workloads as wl
from util import BF16, bf16_ulp_distance, empty_dev, row_l2_rel_err, to_dev, to_host

from test_gpu_layernorm import check_ln, run_ln
from test_gpu_linear import mk, run_linear

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def test_linear_400_random_members(ob):
    rng = np.random.default_rng(2024)
    members = []
    for i in range(400):
        M, N, K = int(rng.integers(1, 300)), int(rng.integers(1, 300)), int(rng.integers(1, 200))
        m = mk(71, i, M, N, K, int(rng.integers(0, 4)), bias=bool(rng.integers(0, 2)))
        members.append(m)
    # unaligned K / N need padded (16-byte aligned) row strides: run_linear allocates dense tensors, so pad here
    dev, descs = [], []
    for m in members:
        ldk, ldn = (m["K"] + 7) // 8 * 8, (m["N"] + 7) // 8 * 8
        x = empty_dev((m["M"], ldk), BF16, fill=0.0); x[:, :m["K"]] = to_dev(m["x"], BF16)
        w = empty_dev((m["N"], ldk), BF16, fill=0.0); w[:, :m["K"]] = to_dev(m["w"], BF16)
        b = None
        if m["b"] is not None:
            b = empty_dev((1, ldn), BF16, fill=0.0); b[0, :m["N"]] = to_dev(m["b"], BF16)
        y = empty_dev((m["M"], ldn), BF16, fill=float("nan"))
        dev.append((x, w, b, y))
        descs.append(ob.linear_member(x[:, :m["K"]], w[:, :m["K"]], None if b is None else b[0, :m["N"]], y[:, :m["N"]], m["act"]))
    plan = ob.opt_linear_plan_create(descs, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    z64, _ = graphs.linear_group(members, BF16)
    worst = 0.0
    for (x, w, b, y), m, z in zip(dev, members, z64):
        worst = max(worst, row_l2_rel_err(to_host(y)[:, :m["N"]], z, BF16))
    assert worst <= 1e-2, worst


def test_layernorm_500_random_members(ob):
    rng = np.random.default_rng(2025)
    members = []
    for i in range(500):
        rows, D = int(rng.integers(1, 200)), 8 * int(rng.integers(1, 257))
        members.append(dict(x=wl.tensor_normal(72, 3 * i + 1, (rows, D), float(rng.uniform(-2, 2)), float(rng.uniform(0.5, 4)), BF16),
                            gamma=wl.tensor_normal(72, 3 * i + 2, (D,), 1.0, 0.3, BF16) if rng.integers(0, 4) else None,
                            beta=wl.tensor_normal(72, 3 * i + 3, (D,), 0.0, 0.3, BF16) if rng.integers(0, 4) else None, eps=1e-5))
    outs = run_ln(ob, members, pad=8 * int(rng.integers(0, 2)))
    esc = tot = 0
    for got, m in zip(outs, members):
        e, t = check_ln(got, m)
        esc += e
        tot += t
    assert esc < 1e-3 * tot


def test_pointwise_300_random_chunks_all_ops(ob):
    rng = np.random.default_rng(2026)
    chunks, host, keep = [], [], []
    for i in range(300):
        rows, w = int(rng.integers(1, 400)), 8 * int(rng.integers(1, 130))
        op = int(rng.integers(0, 9))
        a = wl.tensor_normal(73, 2 * i + 1, (rows, w), 0.0, 2.0, BF16)
        b = wl.tensor_normal(73, 2 * i + 2, (rows, w), 1.0, 1.0, BF16) if op >= 6 else None
        prm = [-1.0, 0.75] if op == 4 else [0.0, 5.0, -5.0] if op == 5 else []
        pad = 8 * int(rng.integers(0, 3))
        da = to_dev(np.pad(a, ((0, 0), (0, pad))), BF16)[:, :w]
        db = None if b is None else to_dev(np.pad(b, ((0, 0), (0, pad))), BF16)[:, :w]
        dd = empty_dev((rows, w + pad), BF16, fill=float("nan"))[:, :w]
        chunks.append(ob.chunk(da, dd, op, db, prm))
        host.append((a, b, op, prm))
        keep.append((da, db, dd))
    plan = ob.opt_pointwise_plan_create(chunks, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    for (a, b, op, prm), (_, _, dd) in zip(host, keep):
        ref64 = oracle.pointwise(a, op, BF16) if op < 4 else oracle.pointwise_ext(a, b, op, prm, BF16)
        d = bf16_ulp_distance(to_host(dd), oracle.round_to_storage(ref64, BF16))
        assert d.max() <= 2, (op, int(d.max()))
        if op == 0:
            assert to_host(dd).tobytes() == a.tobytes()


def test_ln_linear2_300_random_towers(ob):
    """300 towers with random (M, K, H, N), activations, optional affine / biases, in ONE launch: every fold flag,
    tile tail and chunk width the LayerNorm-folded chain distinguishes; relaunched three times (epoch flags)."""
    from test_gpu_ln_linear2 import KEYS, mk as mk_tower
    rng = np.random.default_rng(2027)
    members, descs, keep = [], [], []
    for i in range(300):
        M, K, H, N = int(rng.integers(1, 400)), 8 * int(rng.integers(1, 33)), 16 * int(rng.integers(1, 33)), 16 * int(rng.integers(1, 5))
        m = mk_tower(74, i, M, K, H, N, act1=int(rng.integers(0, 4)), act2=int(rng.integers(0, 4)), bias=bool(rng.integers(0, 2)),
                     affine=bool(rng.integers(0, 4)), mean=float(rng.uniform(-2, 2)), std=float(rng.uniform(0.5, 3)))
        d = {k: (to_dev(m[k], BF16) if m.get(k) is not None else None) for k in KEYS}
        y = empty_dev((M, N), BF16, fill=float("nan"))
        members.append(m)
        keep.append((d, y))
        descs.append(ob.ln_linear2_member(d["x"], d["gamma"], d["beta"], m["eps"], d["w1"], d["b1"], d["w2"], d["b2"], y, m["act1"], m["act2"]))
    plan = ob.opt_ln_linear2_plan_create(descs, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    first = [to_host(y) for _, y in keep]
    # Reading Q26: the chain has three bf16 rounding stages (folded weight, hidden tensor, output)
    # instead of the single GEMM's one, and rows of 16 outputs behind a ReLU can keep only a few small elements, so
    # the row-L2 metric has a heavier tail than on a GEMM row: gate 2e-2 on the worst of ~60 000 rows, and the
    # typical row (median over members of the worst row) must sit at the bf16 rounding floor.
    per_member = [row_l2_rel_err(got, graphs.ln_linear2(m, BF16)["y64"], BF16) for got, m in zip(first, members)]
    assert max(per_member) <= 2e-2, max(per_member)
    assert float(np.median(per_member)) <= 5e-3, float(np.median(per_member))
    for _ in range(3):
        plan.launch()
    torch.cuda.synchronize()
    assert all(to_host(y).tobytes() == f.tobytes() for (_, y), f in zip(keep, first))
