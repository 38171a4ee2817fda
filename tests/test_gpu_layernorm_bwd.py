"""GPU parity: batched LayerNorm BACKWARD vs the CPU oracle (through the C ABI).  SURVEY.md 8(f) rank 3.
Tolerance (backward): dx rows and the dgamma / dbeta vectors are sums with cancellation, so the
bound is the GEMM's -- L2 error relative to the L2 norm of the reference row / vector <= 1e-2 (bf16 output rounding
alone is 2^-9)."""
import numpy as np
import pytest
import torch

import oracle
import workloads as wl
from util import BF16, F32, empty_dev, row_l2_rel_err, to_dev, to_host, values64

pytestmark = pytest.mark.gpu
TOL = 1e-2


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def vec_rel_err(got64, ref64):
    return float(np.linalg.norm(got64 - ref64) / max(np.linalg.norm(ref64), 1e-30))


def run_bwd(ob, members, param_dt=BF16, pad=0, want_params=True):
    dev = []
    for m in members:
        rows, D = m["x"].shape
        x = empty_dev((rows, D + pad), BF16, fill=0.0); x[:, :D] = to_dev(m["x"], BF16)
        dy = empty_dev((rows, D + pad), BF16, fill=0.0); dy[:, :D] = to_dev(m["dy"], BF16)
        dx = empty_dev((rows, D + pad), BF16, fill=float("nan"))
        g = to_dev(m["gamma"], param_dt) if m.get("gamma") is not None else None
        dg = empty_dev((1, D), param_dt, fill=float("nan")) if want_params else None
        db = empty_dev((1, D), param_dt, fill=float("nan")) if want_params else None
        dev.append((x, dy, dx, g, dg, db))
    descs = [ob.layernorm_bwd_member(x[:, :m["x"].shape[1]], dy[:, :m["x"].shape[1]], g, dx[:, :m["x"].shape[1]],
                                     None if dg is None else dg[0], None if db is None else db[0], m["eps"])
             for (x, dy, dx, g, dg, db), m in zip(dev, members)]
    plan = ob.opt_layernorm_bwd_plan_create(descs, BF16, param_dt)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    return dev, plan


def check(dev, members, param_dt=BF16, pad=0, want_params=True):
    for (x, dy, dx, g, dg, db), m in zip(dev, members):
        D = m["x"].shape[1]
        rdx, rdg, rdb = oracle.layernorm_backward(m["x"], m["dy"], m.get("gamma"), m["eps"], BF16, param_dt)
        got = to_host(dx)
        assert row_l2_rel_err(got[:, :D], rdx, BF16) <= TOL
        if pad:
            assert np.all((got[:, D:] & 0x7FFF) > 0x7F80), "wrote outside the member's columns"
        if want_params:
            assert vec_rel_err(values64(to_host(dg)[0], param_dt), rdg) <= TOL
            assert vec_rel_err(values64(to_host(db)[0], param_dt), rdb) <= TOL


def mk(seed, i, rows, D, gamma=True):
    return dict(x=wl.tensor_normal(seed, 4 * i + 1, (rows, D), 0.5, 2.0, BF16), dy=wl.tensor_normal(seed, 4 * i + 2, (rows, D), 0.0, 1.0, BF16),
                gamma=wl.tensor_normal(seed, 4 * i + 3, (D,), 1.0, 0.3, BF16) if gamma else None, eps=1e-5)


@pytest.mark.parametrize("seed", [1, 101])
def test_config1_shapes_small(ob, seed):
    rng = np.random.default_rng(seed)
    members = [mk(seed, i, 333, int(rng.choice([64, 128, 192, 256, 384, 512]))) for i in range(24)]
    dev, _ = run_bwd(ob, members)
    check(dev, members)


def test_dims_edges_strides_null_gamma_fp32_params(ob):
    dims = [8, 16, 24, 32, 40, 64, 72, 128, 200, 256, 384, 504, 512]
    members = [mk(7, i, [1, 2, 5, 17, 64, 100, 700][i % 7], D, gamma=(i % 3 != 0)) for i, D in enumerate(dims)]
    dev, _ = run_bwd(ob, members, pad=8)
    check(dev, members, pad=8)
    mf = [dict(m, gamma=None if m["gamma"] is None else wl.f32_from_bf16_bits(m["gamma"])) for m in members]
    dev, _ = run_bwd(ob, mf, param_dt=F32)
    check(dev, mf, param_dt=F32)
    dev, _ = run_bwd(ob, members, want_params=False)           # dx only
    check(dev, members, want_params=False)


def test_relaunch_is_bitwise_reproducible_many_parts(ob):
    members = [mk(9, i, 5000, 64 * (1 + i % 4)) for i in range(6)]          # dozens of partial-sum parts per member
    dev, plan = run_bwd(ob, members)
    check(dev, members)
    snap = lambda: b"".join(to_host(t).tobytes() for d in dev for t in (d[2], d[4], d[5]))
    first = snap()
    for _ in range(3):
        for d in dev:
            d[4].fill_(float("nan")); d[5].fill_(float("nan"))
        plan.launch()
        torch.cuda.synchronize()
        assert snap() == first


def test_wide_rows_up_to_the_forward_limit(ob):
    """512 < D <= 2048 (a warp per row, column sums in shared memory): every D the forward takes has a backward;
    wide and narrow members mixed in one launch, ragged row counts, several partial-sum parts, NULL gamma, fp32
    parameters, dx-only; relaunches give the same bits."""
    dims = [520, 768, 1024, 1032, 1536, 2040, 2048, 256, 64]
    rows = [300, 17, 1000, 5, 129, 64, 700, 333, 2000]
    members = [mk(13, i, r, D, gamma=(i % 4 != 1)) for i, (r, D) in enumerate(zip(rows, dims))]
    dev, plan = run_bwd(ob, members, pad=8)
    check(dev, members, pad=8)
    snap = lambda: b"".join(to_host(t).tobytes() for d in dev for t in (d[2], d[4], d[5]))
    first = snap()
    for d in dev:
        d[4].fill_(float("nan")); d[5].fill_(float("nan"))
    plan.launch()
    torch.cuda.synchronize()
    assert snap() == first
    mf = [dict(m, gamma=None if m["gamma"] is None else wl.f32_from_bf16_bits(m["gamma"])) for m in members]
    dev, _ = run_bwd(ob, mf, param_dt=F32)
    check(dev, mf, param_dt=F32)
    dev, _ = run_bwd(ob, members, want_params=False)
    check(dev, members, want_params=False)


def test_errors(ob):
    x = empty_dev((4, 4096), BF16, fill=0.0)
    y = empty_dev((4, 4096), BF16, fill=0.0)
    z = empty_dev((4, 4096), BF16, fill=0.0)
    with pytest.raises(ob.OptError) as e:              # D = 4096 exceeds the limit (2048, as in the forward)
        ob.opt_layernorm_bwd_plan_create([ob.layernorm_bwd_member(x, y, None, z, None, None, 1e-5)], BF16)
    assert e.value.status == ob.OPT_ERR_UNSUPPORTED
    with pytest.raises(ob.OptError) as e:              # dx overlaps x
        ob.opt_layernorm_bwd_plan_create([ob.layernorm_bwd_member(x[:, :64], y[:, :64], None, x[:, :64], None, None, 1e-5)], BF16)
    assert e.value.status == ob.OPT_ERR_ALIAS
