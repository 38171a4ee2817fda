"""GPU parity: batched bias gradient db[n] = sum_m dZ[m, n] of N Linear layers in ONE launch vs the CPU oracle
(through the C ABI).  SURVEY.md 8(f) rank 3; PAPER.md:292 batch_linear_post_grad, PAPER.md:437 training.

Tolerance (reading Q27): the kernel adds in fp32 along a fixed tree of depth
d <= rows per thread + row groups + row parts <= 200 for every shape below, so per column
|db - ref| <= d 2^-24 sum_m |dZ[m, n]| <= 2e-5 sum_m |dZ[m, n]|; a bf16 result adds its own rounding 2^-8 |ref|.
Sums of small integers are exact: bit for bit."""
import numpy as np
import pytest
import torch

import oracle
from oracle import graphs
import workloads as wl
from util import BF16, F32, empty_dev, row_l2_rel_err, to_dev, to_host, values64

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def run(ob, dzs, param_dt, pad=0, launches=1):
    """dzs: host bf16-bit arrays [M,N]; pad > 0: each is a column slice of a wider device buffer."""
    dev = []
    for z in dzs:
        M, N = z.shape
        buf = empty_dev((M, N + 2 * pad), BF16, fill=float("nan"))
        buf[:, pad:pad + N] = to_dev(z, BF16)
        db = empty_dev((N,), param_dt, fill=float("nan"))
        dev.append((buf, db))
    plan = ob.opt_bias_grad_plan_create([ob.bias_grad_member(buf[:, pad:pad + z.shape[1]], db) for (buf, db), z in zip(dev, dzs)],
                                        BF16, param_dt)
    outs = []
    for _ in range(launches):
        for _, db in dev:
            db.fill_(float("nan"))
        n0 = ob.opt_launch_count()
        plan.launch()
        torch.cuda.synchronize()
        assert ob.opt_launch_count() - n0 == 1
        outs.append([to_host(db) for _, db in dev])
    return outs, plan


def check(got, z, param_dt):
    ref = graphs.linear_bias_grad(z, BF16)
    l1 = np.abs(values64(z, BF16)).sum(axis=0)
    g64 = values64(got, param_dt)
    bound = 2e-5 * l1 + (2.0 ** -8 * np.abs(ref) if param_dt == BF16 else 0.0)
    assert np.all(np.abs(g64 - ref) <= bound), float(np.max(np.abs(g64 - ref) - bound))


SHAPES = [(300, 512), (77, 200), (1000, 64), (129, 1032), (64, 8), (5, 4096), (1, 24), (100000, 16), (8192, 264), (4097, 40)]


@pytest.mark.parametrize("param_dt", [F32, BF16])
def test_integers_bit_exact(ob, param_dt):
    rng = np.random.default_rng(61)
    dzs = [wl.bf16_bits_from_f32(rng.integers(-2, 3, s).astype(np.float32)) for s in SHAPES]
    (outs,), _ = run(ob, dzs, param_dt)
    for got, z in zip(outs, dzs):
        ref = graphs.linear_bias_grad(z, BF16)                 # |sums| <= 2e5 < 2^24: every fp32 partial is exact
        assert got.tobytes() == oracle.round_to_storage(ref, param_dt).tobytes(), z.shape


@pytest.mark.parametrize("param_dt,pad", [(F32, 0), (BF16, 0), (F32, 24)])
def test_random_group(ob, param_dt, pad):
    dzs = [wl.tensor_normal(62, i + 1, s, 0.1 * (i % 3), 1.0 + i, BF16) for i, s in enumerate(SHAPES)]
    outs, _ = run(ob, dzs, param_dt, pad=pad, launches=3)
    for got, z in zip(outs[0], dzs):
        check(got, z, param_dt)
    # fixed summation order + re-armed tickets: every relaunch gives the same bits
    for again in outs[1:]:
        for a, b in zip(outs[0], again):
            assert a.tobytes() == b.tobytes()


def test_many_small_members(ob):
    """300 members of random shape in one launch (ragged tails, 1-row members, several column tiles)."""
    rng = np.random.default_rng(63)
    shapes = [(int(rng.integers(1, 700)), 8 * int(rng.integers(1, 80))) for _ in range(300)]
    dzs = [wl.tensor_normal(63, i + 1, s, 0.0, 1.0, BF16) for i, s in enumerate(shapes)]
    (outs,), plan = run(ob, dzs, F32)
    for got, z in zip(outs, dzs):
        check(got, z, F32)
    assert plan.info()["bytes"] == sum(z.size * 2 + z.shape[1] * 4 for z in dzs)


def test_fused_relu_mask(ob):
    """y given: dZ = dY where y > 0 (torch threshold_backward: a NaN y keeps the gradient, -0 and +0 cut it) formed,
    written and summed in one pass.  dz_out bit-exact against the oracle's pointwise op 11; db within the summation
    bound of the oracle's column sums of that dZ.  Members: separate dz_out, slices of wider buffers, in place,
    and no dz_out at all."""
    devs, descs, host = [], [], []
    for i, (M, N) in enumerate(SHAPES):
        g = wl.tensor_normal(65, 2 * i + 1, (M, N), 0.0, 2.0, BF16)
        y = wl.tensor_normal(65, 2 * i + 2, (M, N), 0.0, 1.0, BF16).copy()
        y[(y & 0x8000) != 0] = 0x8000 if i % 2 else 0x0000        # what a ReLU leaves: 0 (or -0) where x <= 0
        y.reshape(-1)[::53] = 0x8000
        y.reshape(-1)[7::211] = 0x7FC0                            # NaN forward value
        pad = 24 if i % 2 else 0
        dg = to_dev(np.pad(g, ((0, 0), (0, pad))), BF16)[:, :N]
        dy = to_dev(np.pad(y, ((0, 0), (8, pad))), BF16)[:, 8:8 + N]
        mode = i % 3                                              # 0: separate output, 1: in place, 2: no output
        out = empty_dev((M, N + pad), BF16, fill=float("nan"))[:, :N] if mode == 0 else (dg if mode == 1 else None)
        db = empty_dev((N,), F32, fill=float("nan"))
        descs.append(ob.bias_grad_member(dg, db, dy, out))
        devs.append((dg, dy, out, db)); host.append((g, y, mode))
    plan = ob.opt_bias_grad_plan_create(descs, BF16, F32)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    for (dg, dy, out, db), (g, y, mode) in zip(devs, host):
        ref = oracle.round_to_storage(oracle.pointwise_ext(g, y, oracle.PW_RELU_BWD, [], BF16), BF16)
        if out is not None:
            assert to_host(out).tobytes() == ref.tobytes(), (g.shape, mode)
        else:
            assert to_host(dg).tobytes() == g.tobytes()            # inputs untouched
        check(to_host(db), ref, F32)
    assert plan.info()["bytes"] == sum(g.size * 2 * (3 if mode < 2 else 2) + g.shape[1] * 4 for g, _, mode in host)


@pytest.mark.parametrize("act", [2, 3])
def test_fused_tanh_sigmoid_derivative(ob, act):
    """act = tanh / sigmoid with y given: dZ = dY (1 - y^2) / dY (1 - y) y formed, rounded to bf16, written and summed in
    one pass.  (1) Exact case -- y from {0.5, -0.5 | 0.25, 0, 1}, gradients multiples of 16: every product is exact, so
    dz_out AND db are bit for bit the oracle's.  (2) Random case: dz_out <= 2 bf16 ulp of the oracle's op 12 / 13 and
    bitwise equal to what the pointwise kernel writes for the same op; db within the summation bound plus the two
    ulp (2^-7 relative) each summed element may differ by."""
    from util import bf16_ulp_distance
    oop = oracle.PW_TANH_BWD if act == 2 else oracle.PW_SIGMOID_BWD
    pop = ob.OPT_PW_TANH_BWD if act == 2 else ob.OPT_PW_SIGMOID_BWD
    rng = np.random.default_rng(66 + act)
    yset = np.array([0.5, -0.5 if act == 2 else 0.25, 0.0, 1.0], dtype=np.float32)
    exact, rand = [], []
    for i, (M, N) in enumerate(SHAPES):
        exact.append((wl.bf16_bits_from_f32((16 * rng.integers(-3, 4, (M, N))).astype(np.float32)), wl.bf16_bits_from_f32(yset[rng.integers(0, 4, (M, N))])))
        z = wl.tensor_normal(67, 2 * i + 2, (M, N), 0.0, 2.0, BF16)
        rand.append((wl.tensor_normal(67, 2 * i + 1, (M, N), 0.0, 2.0, BF16), oracle.round_to_storage(oracle.pointwise(z, act, BF16), BF16)))
    for case, members in (("exact", exact), ("random", rand)):
        devs, descs, chunks = [], [], []
        for i, (g, y) in enumerate(members):
            M, N = g.shape
            pad = 24 if i % 2 else 0
            dg = to_dev(np.pad(g, ((0, 0), (0, pad))), BF16)[:, :N]
            dy = to_dev(np.pad(y, ((0, 0), (8, pad))), BF16)[:, 8:8 + N]
            out = empty_dev((M, N + pad), BF16, fill=float("nan"))[:, :N]
            out2 = empty_dev((M, N), BF16, fill=float("nan"))
            db = empty_dev((N,), F32, fill=float("nan"))
            descs.append(ob.bias_grad_member(dg, db, dy, out, act))
            chunks.append(ob.chunk(dg, out2, pop, dy))
            devs.append((out, out2, db, dg, dy))              # keep the inputs alive until the launches are done
        n0 = ob.opt_launch_count()
        ob.opt_bias_grad_plan_create(descs, BF16, F32).launch()
        torch.cuda.synchronize()
        assert ob.opt_launch_count() - n0 == 1
        ob.opt_pointwise_plan_create(chunks, BF16).launch()
        torch.cuda.synchronize()
        for (g, y), (out, out2, db, _, _) in zip(members, devs):
            ref64 = oracle.pointwise_ext(g, y, oop, [], BF16)
            ref = oracle.round_to_storage(ref64, BF16)
            got = to_host(out)
            assert got.tobytes() == to_host(out2).tobytes(), (case, g.shape)
            rdb = graphs.linear_bias_grad(ref, BF16)
            if case == "exact":
                assert np.array_equal(values64(got, BF16), ref64), g.shape
                assert to_host(db).tobytes() == oracle.round_to_storage(rdb, F32).tobytes(), g.shape
            else:
                assert bf16_ulp_distance(got, ref).max() <= 2
                l1 = np.abs(values64(ref, BF16)).sum(axis=0)
                assert np.all(np.abs(to_host(db).astype(np.float64) - rdb) <= (2e-5 + 2.0 ** -7) * l1)


@pytest.mark.parametrize("fused", [False, True])
def test_whole_backward_of_a_linear_relu_group(ob, fused):
    """Forward Y_i = relu(X_i W_i^T + b_i) (one launch) and the whole backward in four launches -- ReLU masks, bias
    gradients, dgrads, wgrads (three with the mask fused into the bias-gradient launch) -- against graphs.linear_relu_backward, which runs its OWN forward in fp64 (no oracle
    input comes from the CUDA path).  The two forwards may disagree in the sign of a pre-activation that is zero to
    rounding, so the masks are compared as sets: <= 1e-4 of the elements may differ."""
    members = []
    for i, (M, N, K) in enumerate([(300, 128, 64), (512, 64, 256), (1000, 256, 128), (257, 136, 72)]):
        members.append(dict(x=wl.tensor_normal(8, 4 * i + 1, (M, K), 0, 1, BF16), w=wl.tensor_normal(8, 4 * i + 2, (N, K), 0, K ** -0.5, BF16),
                            b=wl.tensor_normal(8, 4 * i + 3, (N,), 0, 0.1, BF16), g=wl.tensor_normal(8, 4 * i + 4, (M, N), 0, 1, BF16)))
    dev, fwd, msk, bg, dg, wg = [], [], [], [], [], []
    for m in members:
        (M, K), N = m["x"].shape, m["w"].shape[0]
        x, w, b, g = (to_dev(m[k], BF16) for k in ("x", "w", "b", "g"))
        y, dz = empty_dev((M, N), BF16), empty_dev((M, N), BF16, fill=float("nan"))
        dx, dw, db = empty_dev((M, K), BF16, fill=float("nan")), empty_dev((N, K), BF16, fill=float("nan")), empty_dev((N,), F32, fill=float("nan"))
        dev.append((x, w, b, g, y, dz, dx, dw, db))
        fwd.append(ob.linear_member(x, w, b, y, ob.OPT_ACT_RELU))
        msk.append(ob.chunk(g, dz, ob.OPT_PW_RELU_BWD, y))
        bg.append(ob.bias_grad_member(g, db, y, dz) if fused else ob.bias_grad_member(dz, db))
        dg.append(ob.linear_member(dz, w, None, dx, 0, ob.OPT_LAYOUT_W_TRANSPOSED))
        wg.append(ob.linear_member(dz, x, None, dw, 0, ob.OPT_LAYOUT_X_TRANSPOSED | ob.OPT_LAYOUT_W_TRANSPOSED))
    n0 = ob.opt_launch_count()
    ob.opt_linear_plan_create(fwd, BF16).launch()
    if not fused:
        ob.opt_pointwise_plan_create(msk, BF16).launch()
    ob.opt_bias_grad_plan_create(bg, BF16, F32).launch()       # fused: the mask is formed, written and summed here
    ob.opt_linear_plan_create(dg, BF16).launch()
    ob.opt_linear_plan_create(wg, BF16).launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == (4 if fused else 5)
    for m, d in zip(members, dev):
        r = graphs.linear_relu_backward(m, m["g"], BF16)
        dz = to_host(d[5])
        assert np.mean(dz != r["dz"]) <= 1e-4
        assert 0.2 < np.mean(dz == 0) < 0.8
        l1 = np.abs(values64(r["dz"], BF16)).sum(axis=0)
        gmax = np.abs(values64(m["g"], BF16)).max()
        nflip = int((dz != r["dz"]).sum())
        assert np.all(np.abs(to_host(d[8]).astype(np.float64) - r["db64"]) <= 2e-5 * l1 + nflip * gmax)
        if nflip == 0:
            assert row_l2_rel_err(to_host(d[6]), r["dx64"], BF16) <= 1e-2
            assert row_l2_rel_err(to_host(d[7]), r["dw64"], BF16) <= 1e-2


def test_full_size_c2_bias_grads(ob):
    """configs[2] at full size, the launch bench.py times: the 128 members' gradients are column slices of ONE
    [4096, sum N] concat buffer.  Oracle on every column of 16 sampled members."""
    M, Ns = 4096, [int(n) for n in np.random.default_rng(64).choice([128, 256, 512, 1024], size=128)]      # configs[2]'s recipe
    off = np.concatenate([[0], np.cumsum(Ns)])
    gen = torch.Generator(device="cuda").manual_seed(64)
    dy_cat = torch.empty((M, int(off[-1])), dtype=torch.bfloat16, device="cuda").normal_(0.0, 1.0, generator=gen)
    dbs = [torch.full((n,), float("nan"), dtype=torch.float32, device="cuda") for n in Ns]
    plan = ob.opt_bias_grad_plan_create([ob.bias_grad_member(dy_cat[:, off[i]:off[i + 1]], dbs[i]) for i in range(len(Ns))], BF16, F32)
    plan.launch()
    torch.cuda.synchronize()
    for i in list(range(0, len(Ns), 9)) + [len(Ns) - 1]:
        z = to_host(dy_cat[:, off[i]:off[i + 1]])
        check(to_host(dbs[i]), z, F32)


def test_stress_many_members_mixed_modes_relaunched(ob):
    """4000 members in one plan -- tiny (1..3 rows, one block, one part), ragged, multi-part, plain / ReLU mask /
    tanh / sigmoid derivative mixed, with and without dz_out -- launched 10 times back to back without a sync:
    the self re-arming tickets must leave every relaunch bitwise identical, and every member within its bound."""
    rng = np.random.default_rng(68)
    host, descs, keep = [], [], []
    big = torch.empty(64 << 20, dtype=torch.bfloat16, device="cuda")         # one arena: members are slices of it
    big_y = torch.empty_like(big)
    big.normal_(0.0, 1.0, generator=torch.Generator(device="cuda").manual_seed(68))
    big_y.uniform_(-1.0, 1.0, generator=torch.Generator(device="cuda").manual_seed(69))
    off = 0
    for i in range(4000):
        kind = i % 5
        M = int(rng.integers(1, 4)) if kind == 0 else int(rng.integers(1, 3000)) if kind < 4 else int(rng.integers(9000, 20000))
        N = 8 * int(rng.integers(1, 9 if kind == 4 else 40))
        if off + M * N > big.numel():
            break
        z = big[off:off + M * N].view(M, N); y = big_y[off:off + M * N].view(M, N)
        off += (M * N + 7) // 8 * 8
        mode = int(rng.integers(0, 4))                                       # 0 plain, 1 relu, 2 tanh, 3 sigmoid
        db = torch.full((N,), float("nan"), dtype=torch.float32, device="cuda")
        out = torch.empty((M, N), dtype=torch.bfloat16, device="cuda") if mode and i % 2 else None
        descs.append(ob.bias_grad_member(z, db) if mode == 0 else ob.bias_grad_member(z, db, y, out, mode))
        keep.append((z, y, db, out, mode))
    plan = ob.opt_bias_grad_plan_create(descs, BF16, F32)
    plan.launch()
    torch.cuda.synchronize()
    first = torch.cat([k[2] for k in keep]).clone()
    for k in keep:
        k[2].fill_(float("nan"))
    for _ in range(10):
        plan.launch()
    torch.cuda.synchronize()
    assert torch.equal(torch.cat([k[2] for k in keep]).view(torch.int32), first.view(torch.int32))
    ops = {1: oracle.PW_RELU_BWD, 2: oracle.PW_TANH_BWD, 3: oracle.PW_SIGMOID_BWD}
    for j in list(range(0, len(keep), 37)) + [len(keep) - 1]:              # oracle on a sample of the members
        z, y, db, out, mode = keep[j]
        zh = to_host(z)
        if mode:
            zh = oracle.round_to_storage(oracle.pointwise_ext(zh, to_host(y), ops[mode], [], BF16), BF16)
        l1 = np.abs(values64(zh, BF16)).sum(axis=0)
        slack = (2e-5 if mode < 2 else 2e-5 + 2.0 ** -7) * l1
        assert np.all(np.abs(to_host(db).astype(np.float64) - graphs.linear_bias_grad(zh, BF16)) <= slack), (j, mode, z.shape)
        if out is not None and mode == 1:
            assert to_host(out).tobytes() == zh.tobytes()


def test_fp32_groups_configs0_backward(ob):
    """fp32 activations (configs[0]-like groups, "bias gradient for fp32 groups"): plain column sums,
    the fused ReLU mask (bit-exact select) and the fused tanh / sigmoid derivative, fp32 and bf16 parameter dtype.
    Sums of small integers bit for bit; random data within the fp32 summation bound (depth M/8 + 8, reading Q28)."""
    rng = np.random.default_rng(3)
    # integers: exact
    zi = [rng.integers(-3, 4, (M, N)).astype(np.float32) for M, N in [(64, 32), (64, 16), (1000, 64), (7, 48), (333, 100)]]
    dz = [torch.from_numpy(z).cuda() for z in zi]
    for pdt, tdt in ((F32, torch.float32), (BF16, torch.bfloat16)):
        db = [torch.full((z.shape[1],), float("nan"), dtype=tdt, device="cuda") for z in zi]
        n0 = ob.opt_launch_count()
        ob.opt_bias_grad_plan_create([ob.bias_grad_member(z, d) for z, d in zip(dz, db)], F32, pdt).launch()
        torch.cuda.synchronize()
        assert ob.opt_launch_count() - n0 == 1
        for z, d in zip(zi, db):
            assert np.array_equal(d.float().cpu().numpy().astype(np.float64), graphs.linear_bias_grad(z, F32))
    # configs[0]: the whole backward of the tanh group's epilogue (dZ = dY (1 - y^2), db) in one launch, and a ReLU variant
    c0 = wl.config0()
    for act, op in ((2, oracle.PW_TANH_BWD), (3, oracle.PW_SIGMOID_BWD), (1, oracle.PW_RELU_BWD)):
        keep, descs = [], []
        for i, m in enumerate(c0["members"]):
            y64 = graphs.linear_member(dict(m, act=act), F32)
            y = oracle.round_to_storage(y64, F32)
            dy = wl.tensor_normal(77, i + 1, y.shape, 0.0, 1.0, F32)
            ty, tdy = torch.from_numpy(y).cuda(), torch.from_numpy(dy).cuda()
            tdz = torch.full_like(tdy, float("nan")); tdb = torch.full((y.shape[1],), float("nan"), device="cuda")
            keep.append((y, dy, tdz, tdb, ty, tdy))
            descs.append(ob.bias_grad_member(tdy, tdb, ty, tdz, act))
        ob.opt_bias_grad_plan_create(descs, F32, F32).launch()
        torch.cuda.synchronize()
        for y, dy, tdz, tdb, _, _ in keep:
            ref = oracle.pointwise_ext(dy, y, op, [], F32)
            got = tdz.cpu().numpy()
            if act == 1:
                assert got.tobytes() == oracle.round_to_storage(ref, F32).tobytes()
            else:
                assert np.allclose(got, ref, rtol=3e-7, atol=1e-30)          # one or two fp32 roundings
            l1 = np.abs(got.astype(np.float64)).sum(axis=0)
            assert np.all(np.abs(tdb.cpu().numpy().astype(np.float64) - graphs.linear_bias_grad(got, F32)) <= 2e-5 * l1 + 1e-30)
    # errors: N % 4, act without y
    with pytest.raises(ob.OptError) as e:
        ob.opt_bias_grad_plan_create([ob.bias_grad_member(torch.zeros(8, 8, device="cuda")[:, :6], torch.zeros(6, device="cuda"))], F32, F32)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
