"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The step is built by bench.Step (same arenas, same plans, same six launches).  The oracle cannot
finish the full groups in seconds, so it computes SAMPLED rows (all members, all columns of the
sampled rows -- every op of the path is row-independent): first/last rows, rows around every
128-row tile boundary class, and seeded random rows.  C3's data movement is checked on the whole
[8192, 8192] tensor bit for bit (numpy fancy indexing of the oracle's column map).

C4 (reading Q3): every group is gated against the oracle fed with the GPU's actual bf16
input of that group.
"""
import numpy as np
import pytest
import torch

import oracle
from oracle import graphs
import workloads as wl
from util import BF16, bf16_ulp_distance, row_l2_rel_err, to_host, values64

pytestmark = pytest.mark.gpu

TOL_BF16 = 1e-2


def sample_rows(n_rows, k, seed):
    fixed = [0, 1, 127, 128, 129, n_rows // 2 - 1, n_rows // 2, n_rows - 129, n_rows - 128, n_rows - 2, n_rows - 1]
    rng = np.random.default_rng(seed)
    rows = set(r for r in fixed if 0 <= r < n_rows)
    rows.update(int(r) for r in rng.integers(0, n_rows, size=k))
    return np.array(sorted(rows))


def tile_boundary_rows(n_rows, k, seed):
    """>= k rows: both sides of EVERY 128-row boundary (each CTA's half of every 256-row pair tile, hence every
    pair-tile boundary too), the first and last rows, and seeded random rows up to k."""
    rows = {0, 1, n_rows - 2, n_rows - 1}
    for b in range(128, n_rows, 128):
        rows.update((b - 1, b))
    rng = np.random.default_rng(seed)
    while len(rows) < k:
        rows.update(int(r) for r in rng.integers(0, n_rows, size=k - len(rows)))
    return np.array(sorted(r for r in rows if 0 <= r < n_rows))


@pytest.fixture(scope="module")
def step():
    import bench
    s = bench.Step("cuda:0", bench.FULL, pinned_host=False)
    import paper_2607_02945_b200 as ob
    n0 = ob.opt_launch_count()
    s.launch_all()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 6, "one launch per group"
    return {g.name: g for g in s.groups}


def ln_check(got, x, gamma, beta, eps):
    y64, xh = oracle.layernorm(x, gamma, beta, eps, BF16, BF16, return_xhat=True)
    ref = oracle.round_to_storage(y64, BF16)
    d = bf16_ulp_distance(got, ref)
    g64 = values64(gamma, BF16)
    slack = 2.0 ** -16 * (np.abs(xh * g64) + np.abs(values64(beta, BF16)))                 # Q12
    x64 = values64(x, BF16)                                                                   # Q12b
    mu = x64.mean(axis=1, keepdims=True)
    rstd = 1.0 / np.sqrt(x64.var(axis=1, keepdims=True) + float(np.float32(eps)))
    slack = np.maximum(slack, 2.0 ** -19 * np.abs(g64) * (1.0 + np.abs(mu) * rstd))
    bad = (d > 2) & ~(np.abs(values64(got, BF16) - y64) <= slack)
    assert not bad.any(), "LN mismatch: max ulp %d" % d.max()
    return int((d > 2).sum()), d.size


def test_c1_full_layernorm(step):
    g = step["C1_batched_layernorm"]
    esc = tot = 0
    for i, ((ix, ig, ib, iy), m) in enumerate(zip(g.idx, g.cfg["members"])):
        rows = sample_rows(m["rows"], 24, 1000 + i)
        got = to_host(g.aout.tensor(iy)[torch.from_numpy(rows).cuda()])
        e, t = ln_check(got, np.ascontiguousarray(m["x"][rows]), m["gamma"], m["beta"], m["eps"])
        esc, tot = esc + e, tot + t
    assert esc < 1e-3 * tot


def test_c2_full_grouped_linear(step):
    g = step["C2_grouped_linear_tower"]
    ycat = g.aout.tensor(g.iy)
    worst = 0.0
    for i, m in enumerate(g.cfg["members"]):
        rows = tile_boundary_rows(m["M"], 256, 2000 + i)
        assert len(rows) >= 256
        got = to_host(ycat[torch.from_numpy(rows).cuda(), m["col_off"]:m["col_off"] + m["N"]])
        sub = dict(m, x=np.ascontiguousarray(m["x"][rows]))
        z64 = graphs.linear_member(sub, BF16)
        worst = max(worst, row_l2_rel_err(got, z64, BF16))
        assert np.percentile(bf16_ulp_distance(got, oracle.round_to_storage(z64, BF16)), 99) <= 1
    assert worst <= TOL_BF16, worst


def test_c3_full_split_pointwise_cat(step):
    g = step["C3_split_pointwise_cat"]
    cfg = g.cfg
    out = to_host(g.aout.tensor(g.iy))
    x, widths, ops, perm = cfg["x"], cfg["widths"], cfg["ops"], cfg["perm"]
    rows = sample_rows(cfg["rows"], 200, 3000)
    _, ref = graphs.split_pointwise_cat(np.ascontiguousarray(x[rows]), widths, ops, perm, BF16)
    d = bf16_ulp_distance(out[rows], ref)
    assert d.max() <= 2, "max ulp %d" % d.max()
    # whole tensor: ReLU chunks are pure movement for positive inputs -> bit-exact everywhere;
    # every other column must at least be finite and in the op's range
    starts = np.concatenate(([0], np.cumsum(widths)))
    dpos = 0
    for p in perm:
        w = widths[p]
        src = x[:, starts[p]:starts[p] + w]
        dst = out[:, dpos:dpos + w]
        if ops[p] == wl.gen.PW_RELU:
            pos = (src & 0x8000) == 0
            assert np.array_equal(dst[pos], src[pos])
            assert np.all(dst[~pos & ((src & 0x7FFF) <= 0x7F80)] == 0)
        else:
            v = values64(dst, BF16)
            lo = -1.0 if ops[p] == wl.gen.PW_TANH else 0.0
            assert np.all((v >= lo) & (v <= 1.0))
        dpos += w


def test_c3_full_all_rows_against_the_oracle(step):
    """Every one of the 8192 x 8192 outputs against the oracle (reading Q16 (iii)), in row blocks: <= 2 bf16 ulp of
    f(source element at the mapped index); the oracle's pointwise is row-parallel, 67 M elements take seconds."""
    g = step["C3_split_pointwise_cat"]
    cfg = g.cfg
    out = to_host(g.aout.tensor(g.iy))
    x, widths, ops, perm = cfg["x"], cfg["widths"], cfg["ops"], cfg["perm"]
    worst = 0
    for r0 in range(0, cfg["rows"], 1024):
        _, ref = graphs.split_pointwise_cat(np.ascontiguousarray(x[r0:r0 + 1024]), widths, ops, perm, BF16)
        worst = max(worst, int(bf16_ulp_distance(out[r0:r0 + 1024], ref).max()))
    assert worst <= 2, "max ulp %d" % worst


def test_c3_full_movement_bit_exact_on_the_whole_tensor(step):
    """`north_star`: "movement checked bit-exact" (reading Q16 (i) and (ii)) at configs[3]'s
    FULL size, same widths / permutation / launch shape as the timed plan, every op = COPY:
    (i) the whole output equals the oracle's split -> cat in permuted order, byte for byte;
    (ii) with the identity permutation the output IS the input (split followed by cat of the same chunks)."""
    import paper_2607_02945_b200 as ob
    g = step["C3_split_pointwise_cat"]
    cfg = g.cfg
    x_dev = g.ain.tensor(g.ix)
    widths, perm = cfg["widths"], cfg["perm"]
    n = len(widths)
    out = torch.empty_like(x_dev)
    out.fill_(float("nan"))
    plan = ob.opt_pointwise_plan_create(ob.split_cat_chunks(x_dev, out, widths, [wl.gen.PW_COPY] * n, perm), BF16)
    assert plan.info()["tiles"] == g.plan.info()["tiles"], "same launch shape as the timed plan"
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    assert to_host(out).tobytes() == graphs.split_copy_cat(cfg["x"], widths, perm).tobytes()
    out.fill_(float("nan"))
    ident = ob.opt_pointwise_plan_create(ob.split_cat_chunks(x_dev, out, widths, [wl.gen.PW_COPY] * n, list(range(n))), BF16)
    ident.launch()
    torch.cuda.synchronize()
    assert to_host(out).tobytes() == np.ascontiguousarray(cfg["x"]).tobytes()
    assert graphs.split_copy_cat(cfg["x"], widths, list(range(n))).tobytes() == np.ascontiguousarray(cfg["x"]).tobytes()


def _single_member_outputs(ob, descs_of, out_like):
    """Run every member as its OWN one-member plan into a fresh buffer shaped like the group's output."""
    alt = torch.empty_like(out_like)
    alt.fill_(float("nan"))
    plans = [ob.opt_linear_plan_create([d], BF16) for d in descs_of(alt)]
    for p in plans:
        p.launch()
    torch.cuda.synchronize()
    return alt


def test_c2_full_fused_equals_single_member_plans_bitwise(step):
    """All 4096 rows of all 128 members: the ONE fused launch against 128 single-member launches of the same library
    (same tile shapes and K order => the same bits).  Catches any scheduler / queue / concat-slot fault in rows the
    oracle sample does not visit; the single-member plans are themselves gated against the oracle on small shapes."""
    import paper_2607_02945_b200 as ob
    g = step["C2_grouped_linear_tower"]
    ycat = g.aout.tensor(g.iy)
    T = g.ain.tensor
    alt = _single_member_outputs(ob, lambda buf: [ob.linear_member(T(ix), T(iw), T(ib), buf[:, m["col_off"]:m["col_off"] + m["N"]], m["act"])
                                                  for (ix, iw, ib), m in zip(g.idx, g.cfg["members"])], ycat)
    assert torch.equal(alt.view(torch.int16), ycat.view(torch.int16))


def test_c4_full_fused_equals_single_member_plans_bitwise(step):
    """Same cross-check for configs[4]'s two GEMM groups (all 8192 rows of all 512 towers)."""
    import paper_2607_02945_b200 as ob
    ga, gc = step["C4a_batched_layernorm"], step["C4c_grouped_linear_concat"]
    T, A = ga.ain.tensor, ga.amid.tensor
    towers = ga.cfg["towers"]
    for k, (i, t) in enumerate(zip(ga.idx, towers)):          # group 2: per-tower hidden tensors
        h = A(i["h"])
        alt = torch.empty_like(h)
        ob.opt_linear_plan_create([ob.linear_member(A(i["xn"]), T(i["w1"]), T(i["b1"]), alt, 1)], BF16).launch()
        torch.cuda.synchronize()
        assert torch.equal(alt.view(torch.int16), h.view(torch.int16)), k
    out = gc.aout.tensor(gc.iy)
    alt = _single_member_outputs(ob, lambda buf: [ob.linear_member(A(i["h"]), T(i["w2"]), T(i["b2"]), buf[:, k * t["out"]:(k + 1) * t["out"]], 0)
                                                  for k, (i, t) in enumerate(zip(ga.idx, towers))], out)
    assert torch.equal(alt.view(torch.int16), out.view(torch.int16))


def test_c4_full_three_groups(step):
    ga, gb, gc = step["C4a_batched_layernorm"], step["C4b_grouped_linear_relu"], step["C4c_grouped_linear_concat"]
    towers = ga.cfg["towers"]
    out = gc.aout.tensor(gc.iy)
    amid = ga.amid
    esc = tot = 0
    worst_b = worst_c = worst_e2e = 0.0
    for k in range(0, len(towers), 2):                 # every 2nd tower: all (D, H) classes, 256 towers
        t, i = towers[k], ga.idx[k]
        rows = tile_boundary_rows(t["B"], 256, 4000 + k)   # both sides of every 128-row boundary + random rows
        rsel = torch.from_numpy(rows).cuda()
        xn = to_host(amid.tensor(i["xn"])[rsel])
        h = to_host(amid.tensor(i["h"])[rsel])
        o = to_host(out[rsel, k * t["out"]:(k + 1) * t["out"]])
        e, n = ln_check(xn, np.ascontiguousarray(t["x"][rows]), t["gamma"], t["beta"], t["eps"])
        esc, tot = esc + e, tot + n
        # group 2 from the GPU's own bf16 LN output, group 3 from the GPU's own bf16 H
        h64 = oracle.activation(oracle.linear(xn, t["w1"], t["b1"], BF16), 1)
        worst_b = max(worst_b, row_l2_rel_err(h, h64, BF16))
        o64 = oracle.linear(h, t["w2"], t["b2"], BF16)
        worst_c = max(worst_c, row_l2_rel_err(o, o64, BF16))
        # informational end-to-end chain (oracle rounds at each group boundary), 3x looser
        chain = graphs.recsys_tower(dict(t, x=np.ascontiguousarray(t["x"][rows])))
        worst_e2e = max(worst_e2e, row_l2_rel_err(o, chain["out64"], BF16))
    assert esc < 1e-3 * tot
    assert worst_b <= TOL_BF16 and worst_c <= TOL_BF16, (worst_b, worst_c)
    assert worst_e2e <= 3 * TOL_BF16, worst_e2e


def test_c4_full_one_launch_towers(step):
    """SURVEY 8(f) rank 1 at configs[4]'s full size, on the step's own tensors: the 512 towers as ONE chained-Linear
    launch (from the step's bf16 LN output: bitwise equal to the two-group path) and as ONE LayerNorm-folded launch
    (from the raw inputs: sampled rows against graphs.ln_linear2, reading Q25)."""
    import paper_2607_02945_b200 as ob
    ga, gb, gc = step["C4a_batched_layernorm"], step["C4b_grouped_linear_relu"], step["C4c_grouped_linear_concat"]
    towers = ga.cfg["towers"]
    T, A = ga.ain.tensor, ga.amid.tensor
    ref_out = gc.aout.tensor(gc.iy)
    out2, out3 = torch.empty_like(ref_out), torch.empty_like(ref_out)
    p2 = ob.opt_linear2_plan_create([ob.linear2_member(A(i["xn"]), T(i["w1"]), T(i["b1"]), T(i["w2"]), T(i["b2"]),
                                                       out2[:, k * t["out"]:(k + 1) * t["out"]], 1, 0)
                                     for k, (i, t) in enumerate(zip(ga.idx, towers))], BF16)
    p3 = ob.opt_ln_linear2_plan_create([ob.ln_linear2_member(T(i["x"]), T(i["gamma"]), T(i["beta"]), t["eps"], T(i["w1"]), T(i["b1"]),
                                                             T(i["w2"]), T(i["b2"]), out3[:, k * t["out"]:(k + 1) * t["out"]], 1, 0)
                                        for k, (i, t) in enumerate(zip(ga.idx, towers))], BF16)
    n0 = ob.opt_launch_count()
    p2.launch(); p3.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 2
    assert torch.equal(out2.view(torch.int16), ref_out.view(torch.int16))
    worst = 0.0
    for k in range(0, len(towers), 4):                 # every 4th tower: all (D, H) classes, 128 towers
        t = towers[k]
        rows = sample_rows(t["B"], 6, 5000 + k)
        rsel = torch.from_numpy(rows).cuda()
        o = to_host(out3[rsel, k * t["out"]:(k + 1) * t["out"]])
        r = graphs.ln_linear2(dict(t, x=np.ascontiguousarray(t["x"][rows]), act1=1, act2=0), BF16)
        worst = max(worst, row_l2_rel_err(o, r["y64"], BF16))
    assert worst <= TOL_BF16, worst
    # and the two one-launch results differ only by the LN output's rounding (Q25)
    d = (out3.float() - out2.float()).norm(dim=1) / out2.float().norm(dim=1).clamp_min(1e-30)
    assert float(d.max()) <= TOL_BF16
