"""GPU parity: batched_layernorm vs the CPU oracle (through the C ABI)."""
import numpy as np
import pytest
import torch

import oracle
import workloads as wl
from util import BF16, F32, bf16_ulp_distance, empty_dev, to_dev, to_host, values64

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def check_ln(got_bits, m, dt=BF16, param_dt=None):
    """DESIGN.md tolerance (Q11 + Q12 + Q12b): <= 2 bf16 ulp of the oracle rounded to bf16, OR within
    2^-16 * (|xhat*gamma| + |beta|) where the result is a cancellation of larger terms, OR within the fp32
    accuracy floor of x - mu; the escapes must be used by < 1e-3 of the elements."""
    param_dt = dt if param_dt is None else param_dt
    y64, xh = oracle.layernorm(m["x"], m.get("gamma"), m.get("beta"), m["eps"], dt, param_dt, return_xhat=True)
    ref = oracle.round_to_storage(y64, dt)
    d = bf16_ulp_distance(got_bits, ref)
    g = values64(m["gamma"], param_dt) if m.get("gamma") is not None else 1.0
    b = values64(m["beta"], param_dt) if m.get("beta") is not None else 0.0
    slack = 2.0 ** -16 * (np.abs(xh * g) + np.abs(b))
    # Q12b: x - mu cancels too.  fp32 statistics carry mu with relative error ~ log2(D) 2^-24, so the normalised value
    # has an ABSOLUTE error floor of ~ 2^-20 (1 + |mu| / sqrt(v + eps)) whatever the kernel; where |y| is that small,
    # bf16 ulps of y are meaningless.  Allowed: 2^-19 |gamma| (1 + |mu| rstd), i.e. < 2^-11 of a bf16 ulp of xhat ~ 1.
    x64 = values64(m["x"], dt)
    mu = x64.mean(axis=1, keepdims=True)
    rstd = 1.0 / np.sqrt(x64.var(axis=1, keepdims=True) + float(np.float32(m["eps"])))
    slack = np.maximum(slack, 2.0 ** -19 * np.abs(g) * (1.0 + np.abs(mu) * rstd))
    bad = (d > 2) & ~(np.abs(values64(got_bits, dt) - y64) <= slack)
    assert not bad.any(), "LN mismatch: max ulp %d at %s" % (d.max(), np.argwhere(bad)[:4])
    return int((d > 2).sum()), d.size


def run_ln(ob, members, dt=BF16, param_dt=None, pad=0):
    dev = []
    for m in members:
        rows, D = m["x"].shape
        xfull = empty_dev((rows, D + pad), dt, fill=0.0)
        xfull[:, :D] = to_dev(m["x"], dt)
        yfull = empty_dev((rows, D + pad), dt, fill=float("nan"))
        pdt = dt if param_dt is None else param_dt
        g = to_dev(m["gamma"], pdt) if m.get("gamma") is not None else None
        b = to_dev(m["beta"], pdt) if m.get("beta") is not None else None
        dev.append((xfull, yfull, g, b))
    descs = [ob.layernorm_member(x[:, :m["x"].shape[1]], y[:, :m["x"].shape[1]], g, b, m["eps"])
             for (x, y, g, b), m in zip(dev, members)]
    plan = ob.opt_layernorm_plan_create(descs, dt, param_dt)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    outs = []
    for (x, y, g, b), m in zip(dev, members):
        yh = to_host(y)
        D = m["x"].shape[1]
        if pad:
            assert np.all((yh[:, D:] & 0x7FFF) > 0x7F80), "wrote outside the member's columns"
        outs.append(yh[:, :D])
    return outs


@pytest.mark.parametrize("seed", [1, 101, 201])
def test_config1_small(ob, seed):
    cfg = wl.config1(seed=seed, rows=333, n=24)          # all D classes, ragged row count
    outs = run_ln(ob, cfg["members"])
    esc = tot = 0
    for got, m in zip(outs, cfg["members"]):
        e, t = check_ln(got, m)
        esc += e
        tot += t
    assert esc < 1e-3 * tot


def test_dims_edges_and_strides(ob):
    members = []
    for i, D in enumerate([8, 16, 24, 32, 40, 64, 72, 128, 192, 200, 256, 384, 512, 1000, 1024, 1536, 2040, 2048]):
        rows = [1, 2, 5, 17, 64, 100][i % 6]
        members.append(dict(x=wl.tensor_normal(21, 3 * i + 1, (rows, D), 0.5, 2.0, BF16),
                            gamma=wl.tensor_normal(21, 3 * i + 2, (D,), 1.0, 0.3, BF16),
                            beta=wl.tensor_normal(21, 3 * i + 3, (D,), 0.0, 0.3, BF16), eps=1e-5))
    outs = run_ln(ob, members, pad=8)                    # ld > D on both sides
    for got, m in zip(outs, members):
        check_ln(got, m)


def test_null_affine_fp32_params_and_constant_rows(ob):
    x = wl.tensor_normal(22, 1, (50, 96), -1.0, 3.0, BF16)
    x[7, :] = x[7, 0]                                    # constant row -> beta exactly
    m0 = dict(x=x, gamma=None, beta=None, eps=1e-5)
    got = run_ln(ob, [m0])[0]
    check_ln(got, m0)
    assert np.all(bf16_ulp_distance(got[7], np.zeros(96, np.uint16)) == 0)
    m1 = dict(x=x, gamma=wl.tensor_normal(22, 2, (96,), 1.0, 0.3, F32), beta=wl.tensor_normal(22, 3, (96,), 0, 0.3, F32),
              eps=1e-3)
    got = run_ln(ob, [m1], param_dt=F32)[0]
    check_ln(got, m1, param_dt=F32)


def test_unsupported_and_alias(ob):
    x = empty_dev((4, 4096), BF16, fill=0.0)
    y = empty_dev((4, 4096), BF16, fill=0.0)
    with pytest.raises(ob.OptError) as e:
        ob.opt_layernorm_plan_create([ob.layernorm_member(x, y, None, None, 1e-5)], BF16)
    assert e.value.status == ob.OPT_ERR_UNSUPPORTED
    with pytest.raises(ob.OptError) as e:
        ob.opt_layernorm_plan_create([ob.layernorm_member(x[:, :64], x[:, :64], None, None, 1e-5)], BF16)
    assert e.value.status == ob.OPT_ERR_ALIAS
    with pytest.raises(ob.OptError) as e:
        ob.opt_layernorm_plan_create([ob.layernorm_member(x[:, :60], y[:, :60], None, None, 1e-5)], BF16)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT


def test_relaunch_rearms_the_scheduler_and_is_bitwise_reproducible(ob):
    cfg = wl.config1(seed=301, rows=777, n=40)
    dev = []
    for m in cfg["members"]:
        dev.append((to_dev(m["x"], BF16), empty_dev(m["x"].shape, BF16, fill=float("nan")), to_dev(m["gamma"], BF16),
                    to_dev(m["beta"], BF16)))
    plan = ob.opt_layernorm_plan_create([ob.layernorm_member(x, y, g, b, m["eps"]) for (x, y, g, b), m in zip(dev, cfg["members"])], BF16)
    ref = None
    for it in range(4):
        for d in dev:
            d[1].fill_(float("nan"))
        plan.launch()
        torch.cuda.synchronize()
        got = b"".join(to_host(d[1]).tobytes() for d in dev)
        if ref is None:
            ref = got
            for d, m in zip(dev, cfg["members"]):
                check_ln(to_host(d[1]), m)
        assert got == ref
