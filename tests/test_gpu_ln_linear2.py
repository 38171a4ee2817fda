"""GPU parity: grouped LayerNorm + CHAINED Linear (the whole tower of configs[4] in one launch, the normalised tensor
never materialised) vs the CPU oracle `graphs.ln_linear2` (reading Q25), through the C ABI.  SURVEY.md 8(f) rank 1."""
import numpy as np
import pytest
import torch

from oracle import graphs
import workloads as wl
from util import BF16, empty_dev, row_l2_rel_err, to_dev, to_host

pytestmark = pytest.mark.gpu

TOL = 1e-2          # north_star: bf16 GEMM, max relative error normalised by the row's L2 norm


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def mk(seed, i, M, K, H, N, act1=1, act2=0, bias=True, affine=True, mean=0.0, std=1.0, eps=1e-5):
    t = lambda r, shape, mu, sd: wl.tensor_normal(seed, 10 * i + r, shape, mu, sd, BF16)
    return dict(M=M, K=K, H=H, N=N, act1=act1, act2=act2, eps=eps, x=t(1, (M, K), mean, std),
                gamma=t(6, (K,), 1.0, 0.1) if affine else None, beta=t(7, (K,), 0.0, 0.1) if affine else None,
                w1=t(2, (H, K), 0, K ** -0.5), b1=t(3, (H,), 0, 0.1) if bias else None,
                w2=t(4, (N, H), 0, H ** -0.5), b2=t(5, (N,), 0, 0.1) if bias else None)


KEYS = ("x", "gamma", "beta", "w1", "b1", "w2", "b2")


def run_fused(ob, members, concat=True):
    M = members[0]["M"]
    width = sum(m["N"] for m in members)
    ycat = empty_dev((M, width), BF16, fill=float("nan")) if concat else None
    off, descs, ys, dev = 0, [], [], []
    for m in members:
        d = {k: (to_dev(m[k], BF16) if m.get(k) is not None else None) for k in KEYS}
        y = ycat[:, off:off + m["N"]] if concat else empty_dev((m["M"], m["N"]), BF16, fill=float("nan"))
        off += m["N"]
        dev.append(d)
        ys.append(y)
        descs.append(ob.ln_linear2_member(d["x"], d["gamma"], d["beta"], m["eps"], d["w1"], d["b1"], d["w2"], d["b2"], y,
                                          m["act1"], m["act2"]))
    plan = ob.opt_ln_linear2_plan_create(descs, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1 and plan.info()["launches"] == 1
    return ys, plan, dev


def check(ob, members, concat=True, tol=TOL):
    ys, plan, dev = run_fused(ob, members, concat)
    worst = 0.0
    for y, m in zip(ys, members):
        r = graphs.ln_linear2(m, BF16)
        worst = max(worst, row_l2_rel_err(to_host(y), r["y64"], BF16))
    assert worst <= tol, worst
    return ys, plan, dev


def test_sign_rows_small_integers_bit_exact(ob):
    """rows of equally many -1 / +1 (mean 0, variance 1, eps = 0) with integer gamma, beta and weights: the whole
    tower is integer arithmetic, every fp32 step exact -> the output must equal the oracle's bits."""
    rng = np.random.default_rng(21)
    conv = lambda a: wl.bf16_bits_from_f32(np.asarray(a).astype(np.float32))
    members = []
    for (M, K, H, N) in [(128, 64, 128, 64), (200, 32, 48, 16), (257, 136, 272, 64), (5, 8, 16, 16)]:
        x = np.stack([rng.permutation(np.repeat([-1, 1], K // 2)) for _ in range(M)])
        members.append(dict(M=M, K=K, H=H, N=N, act1=1, act2=0, eps=0.0, x=conv(x),
                            gamma=conv(rng.integers(-2, 3, (K,))), beta=conv(rng.integers(-1, 2, (K,))),
                            w1=conv(rng.integers(-1, 2, (H, K))), b1=conv(rng.integers(-2, 3, (H,))),
                            w2=conv(rng.integers(-1, 2, (N, H)) * (rng.random((N, H)) < 0.1)), b2=conv(rng.integers(-2, 3, (N,)))))
    ys, _, _ = run_fused(ob, members, concat=False)
    for y, m in zip(ys, members):
        r = graphs.ln_linear2(m, BF16)
        assert np.abs(r["h64"]).max() <= 256 and np.abs(r["y64"]).max() <= 256      # everything exact in bf16
        assert to_host(y).tobytes() == r["y"].tobytes()


def test_towers_random_all_shape_classes(ob):
    """configs[4]-like towers plus every tail class: K in {32..256} incl. K % 64 != 0 and K % 16 == 8, H with partial
    128-chunks, N in {16..64}, M with a ragged last tile, all activations, with / without affine and biases."""
    shapes = [(300, 32, 128, 64), (300, 64, 256, 64), (300, 128, 512, 64), (300, 256, 512, 64), (300, 256, 128, 64),
              (300, 72, 144, 48), (300, 200, 336, 32), (300, 8, 16, 16), (300, 24, 48, 64), (300, 248, 496, 16)]
    members = [mk(61, i, *s, act1=(1, 2, 3, 0)[i % 4], act2=(0, 0, 2, 3)[i % 4], bias=i % 3 != 1, affine=i % 4 != 2)
               for i, s in enumerate(shapes)]
    check(ob, members)


def test_shifted_and_scaled_rows(ob):
    """rows far from zero mean / unit variance (the statistics are shifted-single-pass fp32; the mean term cancels
    against s = row sums of the FOLDED weight): mean 8 std 0.5, mean -3 std 4, tiny std, constant rows (var = 0)."""
    members = [mk(62, 0, 256, 128, 256, 64, mean=8.0, std=0.5), mk(62, 1, 256, 256, 384, 64, mean=-3.0, std=4.0),
               mk(62, 2, 256, 64, 128, 32, mean=0.25, std=0.01, eps=1e-5)]
    const = mk(62, 3, 256, 64, 128, 32)
    const["x"] = wl.bf16_bits_from_f32(np.full((256, 64), 3.0, dtype=np.float32))     # xn = beta exactly
    members.append(const)
    check(ob, members, concat=False)


def test_config4_small_matches_oracle_and_three_group_path(ob):
    """the configs[4] tower recipe at reduced batch: against the oracle, and against this library's own three-group
    path (LN -> bf16 -> Linear+ReLU -> bf16 -> Linear), from which it differs by one rounding of the LN output."""
    cfg = wl.config4(seed=4, B=384, n=24)
    members = [dict(M=t["B"], K=t["D"], H=t["H"], N=t["out"], act1=1, act2=0, eps=t["eps"], x=t["x"], gamma=t["gamma"],
                    beta=t["beta"], w1=t["w1"], b1=t["b1"], w2=t["w2"], b2=t["b2"]) for t in cfg["towers"]]
    ys, plan, dev = check(ob, members)
    xn = [empty_dev((m["M"], m["K"]), BF16) for m in members]
    hs = [empty_dev((m["M"], m["H"]), BF16) for m in members]
    y3 = [empty_dev((m["M"], m["N"]), BF16) for m in members]
    ob.opt_layernorm_plan_create([ob.layernorm_member(d["x"], a, d["gamma"], d["beta"], m["eps"]) for d, a, m in zip(dev, xn, members)], BF16).launch()
    ob.opt_linear_plan_create([ob.linear_member(a, d["w1"], d["b1"], h, 1) for d, a, h in zip(dev, xn, hs)], BF16).launch()
    ob.opt_linear_plan_create([ob.linear_member(h, d["w2"], d["b2"], y, 0) for d, h, y in zip(dev, hs, y3)], BF16).launch()
    torch.cuda.synchronize()
    for y, yy, m in zip(ys, y3, members):
        ref = wl.f32_from_bf16_bits(to_host(yy)).astype(np.float64)
        assert row_l2_rel_err(to_host(y), ref, BF16) <= TOL


def test_relaunch_refolds_current_weights_and_graph_replay(ob):
    """the fold (W1 diag(gamma), s, c) is redone from the CURRENT parameters inside every launch: change gamma / W1 /
    b1 in place, relaunch the same plan -> new result; launches are bitwise reproducible, also replayed from a graph."""
    members = [mk(63, i, 400, 128, 256, 64) for i in range(6)]
    ys, plan, dev = check(ob, members)
    first = [to_host(y).copy() for y in ys]
    for _ in range(3):
        plan.launch()
    torch.cuda.synchronize()
    assert all(to_host(y).tobytes() == f.tobytes() for y, f in zip(ys, first))
    new = [mk(64, i, 400, 128, 256, 64) for i in range(6)]
    for d, m, n in zip(dev, members, new):
        for k in ("gamma", "w1", "b1"):
            d[k].copy_(to_dev(n[k], BF16))
            m[k] = n[k]
    plan.launch()
    torch.cuda.synchronize()
    for y, m, f in zip(ys, members, first):
        assert row_l2_rel_err(to_host(y), graphs.ln_linear2(m, BF16)["y64"], BF16) <= TOL
        assert to_host(y).tobytes() != f.tobytes()
    second = [to_host(y).copy() for y in ys]
    g = torch.cuda.CUDAGraph()
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        plan.launch(stream.cuda_stream)
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=stream):
            plan.launch(stream.cuda_stream)
            plan.launch(stream.cuda_stream)
    for y in ys:
        y.fill_(float("nan"))
    g.replay(); g.replay()
    torch.cuda.synchronize()
    assert all(to_host(y).tobytes() == f.tobytes() for y, f in zip(ys, second))


def test_errors_launch_nothing(ob):
    m = mk(65, 0, 64, 64, 128, 64)
    d = {k: to_dev(m[k], BF16) for k in KEYS}
    y = empty_dev((64, 64), BF16)
    n0 = ob.opt_launch_count()
    with pytest.raises(ob.OptError) as e:          # K beyond the on-chip limit
        big = mk(65, 1, 64, 512, 128, 64)
        db = {k: to_dev(big[k], BF16) for k in KEYS}
        ob.opt_ln_linear2_plan_create([ob.ln_linear2_member(db["x"], db["gamma"], db["beta"], 1e-5, db["w1"], db["b1"], db["w2"], db["b2"], y)], BF16)
    assert e.value.status == ob.OPT_ERR_UNSUPPORTED
    with pytest.raises(ob.OptError) as e:          # output aliases gamma's owner tensor
        ob.opt_ln_linear2_plan_create([ob.ln_linear2_member(d["x"], d["gamma"], d["beta"], 1e-5, d["w1"], d["b1"], d["w2"], d["b2"], d["x"][:, :64])], BF16)
    assert e.value.status == ob.OPT_ERR_ALIAS
    with pytest.raises(ob.OptError) as e:
        ob.opt_ln_linear2_plan_create([ob.ln_linear2_member(d["x"], d["gamma"], d["beta"], -1.0, d["w1"], d["b1"], d["w2"], d["b2"], y)], BF16)
    assert e.value.status == ob.OPT_ERR_INVALID_ARG
    assert ob.opt_launch_count() == n0
