"""Pins for the CPU oracle (oracle/), none of which re-use the oracle's own
formulas: the paper's worked example (tests/golden), closed forms, hand-computed
brute-force cases, identities, library routines on special cases, exhaustive
rounding enumeration.  SURVEY.md 8(c) P1-P12, Q5, Q13.  CPU only.
"""
import math
import os

import numpy as np
import pytest

import oracle
from oracle import BF16, F32, graphs
import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def bf16(a):
    """float array exactly representable in bf16 -> bits (asserts exactness)."""
    a = np.asarray(a, dtype=np.float32)
    u = wl.bf16_bits_from_f32(a)
    assert np.array_equal(wl.f32_from_bf16_bits(u), a), "test value not exact in bf16"
    return u


def st(a, dt):
    return np.asarray(a, dtype=np.float32) if dt == F32 else bf16(a)


# ------------------------------------------------------------------ P12 -----
def _bf16_value(u):
    """value of a finite non-negative bf16 pattern from the format definition."""
    e, f = u >> 7, u & 0x7F
    return math.ldexp(f, -133) if e == 0 else math.ldexp(128 + f, e - 134)


def test_p12_bf16_rounding_exhaustive():
    us = np.arange(0, 0x7F80, dtype=np.int64)               # all finite non-negative patterns
    vals = np.array([_bf16_value(int(u)) for u in us], dtype=np.float64)
    # exact values round to themselves, both signs; widen is the inverse
    assert np.array_equal(oracle.round_to_storage(vals, BF16), us.astype(np.uint16))
    neg = oracle.round_to_storage(-vals, BF16)
    assert np.array_equal(neg, (us | 0x8000).astype(np.uint16))
    assert np.array_equal(oracle.widen(us.astype(np.uint16), BF16), vals)
    # midpoints between consecutive patterns: ties to even; one double ulp either side decides
    lo, hi = vals[:-1], vals[1:]
    mid = (lo + hi) / 2.0
    assert np.all((mid > lo) & (mid < hi))
    even = (us[:-1] % 2 == 0)
    exp_tie = np.where(even, us[:-1], us[1:]).astype(np.uint16)
    assert np.array_equal(oracle.round_to_storage(mid, BF16), exp_tie)
    assert np.array_equal(oracle.round_to_storage(np.nextafter(mid, np.inf), BF16), us[1:].astype(np.uint16))
    assert np.array_equal(oracle.round_to_storage(np.nextafter(mid, -np.inf), BF16), us[:-1].astype(np.uint16))
    assert np.array_equal(oracle.round_to_storage(-mid, BF16), exp_tie | np.uint16(0x8000))
    # overflow: max finite is 0x7F7F; the midpoint to 2^128 ties to even = inf
    vmax = _bf16_value(0x7F7F)
    top = (vmax + math.ldexp(1.0, 128)) / 2.0
    r = oracle.round_to_storage(np.array([top, np.nextafter(top, 0.0), 1e300, -1e300, np.inf]), BF16)
    assert list(r) == [0x7F80, 0x7F7F, 0x7F80, 0xFF80, 0x7F80]
    # underflow: half the min subnormal ties to even (0); just above -> min subnormal
    tiny = math.ldexp(1.0, -134)
    r = oracle.round_to_storage(np.array([tiny, np.nextafter(tiny, 1.0), tiny / 4, 0.0, -0.0]), BF16)
    assert list(r) == [0, 1, 0, 0, 0x8000]
    assert oracle.round_to_storage(np.array([np.nan]), BF16)[0] & 0x7FFF > 0x7F80


def test_p12_double_rounding_trap():
    # 1 + 2^-8 + 2^-40 lies just above the bf16 midpoint between 1 and 1+2^-7; rounding through fp32
    # first lands exactly on the midpoint and then ties to even (1.0): the oracle must round directly.
    d = 1.0 + 2.0 ** -8 + 2.0 ** -40
    assert oracle.round_to_storage(np.array([d]), BF16)[0] == 0x3F81
    assert wl.bf16_bits_from_f32(np.array([np.float32(d)]))[0] == 0x3F80   # the via-fp32 answer differs


def test_f32_rounding_matches_ieee_cast():
    rng = np.random.default_rng(0)
    z = rng.standard_normal(10000) * np.exp(rng.uniform(-30, 30, 10000))
    assert np.array_equal(oracle.round_to_storage(z, F32), z.astype(np.float32))


# ------------------------------------------------------------------- P1 -----
def _read_golden():
    d = {}
    for line in open(os.path.join(GOLD, "listing2_split_cat.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, rest = line.split(None, 1)
        if ";" in rest:
            d[k] = np.array([[int(t) for t in row.split()] for row in rest.split(";")])
        else:
            d[k] = [int(t) for t in rest.split()]
    return d


@pytest.mark.parametrize("dt", [F32, BF16])
def test_p1_paper_listing2_is_identity(dt):
    g = _read_golden()
    assert g["input_shape"] == [2, 6] and g["cat_dim"] == [1]
    # (a) explicit integer instance, pieces written by hand in the fixture
    x = st(g["x"], dt)
    fs = oracle.split(x, g["first_split"])
    assert np.array_equal(fs[0], st(g["item0"], dt)) and np.array_equal(fs[1], st(g["item1"], dt))
    it = oracle.split(fs[1], g["second_split"])
    assert np.array_equal(it[0], st(g["item2"], dt)) and np.array_equal(it[1], st(g["item3"], dt))
    out = oracle.cat([fs[0]] + it)
    assert np.array_equal(out, st(g["cat"], dt)) and np.array_equal(out, x)
    # (b) the paper's own instance: random [2,6] input, result == input bit for bit (Listing 1)
    ex = wl.listing2_example(dtype=dt)
    fs = oracle.split(ex["x"], ex["first_split"])
    out = oracle.cat([fs[0]] + oracle.split(fs[1], ex["second_split"]))
    assert out.tobytes() == ex["x"].tobytes()


# ------------------------------------------------------------------- P2 -----
def test_p2_split_cat_identities_and_permutation():
    rng = np.random.default_rng(5)
    for trial in range(20):
        rows, n = int(rng.integers(1, 9)), int(rng.integers(1, 12))
        widths = [int(w) for w in rng.integers(1, 7, size=n)]
        W = sum(widths)
        x = rng.integers(0, 65536, size=(rows, W)).astype(np.uint16)
        pieces = oracle.split(x, widths)
        s = 0
        for p, w in zip(pieces, widths):                    # split against numpy slicing (library)
            assert np.array_equal(p, x[:, s:s + w])
            s += w
        assert np.array_equal(oracle.cat(pieces), x)        # split then cat = identity
        back = oracle.split(oracle.cat(pieces), widths)     # cat then split = identity
        assert all(np.array_equal(a, b) for a, b in zip(back, pieces))
        perm = rng.permutation(n)
        y = graphs.split_copy_cat(x, widths, perm)
        assert np.array_equal(y, np.concatenate([x[:, sum(widths[:p]):sum(widths[:p + 1])] for p in perm], axis=1))
        inv = np.argsort(perm)
        z = graphs.split_copy_cat(y, [widths[p] for p in perm], inv)
        assert np.array_equal(z, x)                         # permutation then inverse = identity
    with pytest.raises(ValueError):
        oracle.split(np.zeros((2, 6), np.uint16), [2, 3])
    # strided (non-dense) source
    big = rng.integers(0, 65536, size=(4, 20)).astype(np.uint16)
    v = big[:, 3:15]
    assert np.array_equal(oracle.cat(oracle.split(v, [5, 7])), v)


# ------------------------------------------------------------------- P3 -----
@pytest.mark.parametrize("dt", [F32, BF16])
def test_p3_linear_hand_computed(dt):
    # X:[2,2], W:[3,2] ([N,K], torch layout), b:[3].  By hand:
    # row0: [1*1+2*0, 1*0+2*1, 1*1+2*1] + b = [1,2,3]+[10,20,30]; row1: [3,4,7]+b
    X = st([[1, 2], [3, 4]], dt)
    W = st([[1, 0], [0, 1], [1, 1]], dt)
    b = st([10, 20, 30], dt)
    Z = oracle.linear(X, W, b, dt)
    assert np.array_equal(Z, np.array([[11, 22, 33], [13, 24, 37]], dtype=np.float64))
    # asymmetric 2x3 . (2x3)^T : catches a transposed operand or swapped index
    X = st([[1, 2, 3], [4, 5, 6]], dt)
    W = st([[1, -1, 2], [0, 3, -2]], dt)
    Z = oracle.linear(X, W, None, dt)
    assert np.array_equal(Z, np.array([[1 - 2 + 6, 6 - 6], [4 - 5 + 12, 15 - 12]], dtype=np.float64))


@pytest.mark.parametrize("dt", [F32, BF16])
def test_p3_layernorm_hand_computed(dt):
    x = st([[1, 2, 3, 4]], dt)
    y, xh = oracle.layernorm(x, None, None, 0.0, dt, return_xhat=True)
    # mu = 2.5, v = 1.25 : xhat = (x-2.5)/sqrt(1.25)
    exp = np.array([-1.5, -0.5, 0.5, 1.5]) / math.sqrt(1.25)
    assert np.allclose(y[0], exp, rtol=0, atol=1e-15) and np.array_equal(y, xh)
    eps = float(np.float32(1e-5))
    y = oracle.layernorm(x, st([2, 2, 2, 2], dt), st([1, 0, -1, 0.5], dt), 1e-5, dt)
    exp = np.array([-1.5, -0.5, 0.5, 1.5]) / math.sqrt(1.25 + eps) * 2 + np.array([1, 0, -1, 0.5])
    assert np.allclose(y[0], exp, rtol=0, atol=1e-15)
    # constant row -> beta exactly; D = 1 -> beta
    beta = st([0.5, -0.25, 2, 1], dt)
    y = oracle.layernorm(st([[3, 3, 3, 3]], dt), st([1, 2, 3, 4], dt), beta, 1e-5, dt)
    assert np.array_equal(y[0], np.array([0.5, -0.25, 2, 1]))
    y = oracle.layernorm(st([[7], [-2]], dt), st([3], dt), st([0.75], dt), 1e-5, dt)
    assert np.array_equal(y, np.array([[0.75], [0.75]]))


# ------------------------------------------------------------ P4, P5, P6 ----
def _rand_linear(rng, M, N, K, dt):
    x = wl.tensor_normal(int(rng.integers(1 << 30)), 1, (M, K), 0, 1, dt)
    w = wl.tensor_normal(int(rng.integers(1 << 30)), 2, (N, K), 0, K ** -0.5, dt)
    b = wl.tensor_normal(int(rng.integers(1 << 30)), 3, (N,), 0, 0.1, dt)
    return x, w, b


@pytest.mark.parametrize("dt", [F32, BF16])
def test_p4_zero_padding_invariance(dt):
    """pad_aten_mm_pass: pad -> mm -> slice leaves the result unchanged."""
    rng = np.random.default_rng(11)
    M, N, K = 5, 13, 11
    x, w, b = _rand_linear(rng, M, N, K, dt)
    z = oracle.linear(x, w, b, dt)
    xp = np.zeros((M, 16), x.dtype); xp[:, :K] = x
    wp = np.zeros((16, 16), w.dtype); wp[:N, :K] = w
    bp = np.zeros((16,), b.dtype); bp[:N] = b
    zp = oracle.linear(xp, wp, bp, dt)
    assert np.array_equal(zp[:, :N], z)
    assert np.array_equal(zp[:, N:], np.zeros((M, 3)))


@pytest.mark.parametrize("dt", [F32, BF16])
def test_p5_linear_equals_mul_then_reduce_and_library(dt):
    """decompose_mm_pass: mm == pointwise mul + reduce over K; and == the library matmul."""
    rng = np.random.default_rng(12)
    for (M, N, K) in [(7, 9, 33), (3, 64, 128), (16, 5, 1)]:
        x, w, b = _rand_linear(rng, M, N, K, dt)
        z = oracle.linear(x, w, b, dt)
        z2 = oracle.linear(x, w, b, dt, mulreduce=True)
        xd, wd, bd = (wl.f32_from_bf16_bits(a).astype(np.float64) if dt == BF16 else a.astype(np.float64)
                      for a in (x, w, b))
        z3 = xd @ wd.T + bd                                   # library routine
        scale = np.abs(xd) @ np.abs(wd).T + np.abs(bd)
        assert np.all(np.abs(z - z2) <= 1e-13 * scale)
        assert np.all(np.abs(z - z3) <= 1e-13 * scale)
        # strided x (ldx > K)
        xb = np.zeros((M, K + 5), x.dtype); xb[:, :K] = x
        assert np.array_equal(oracle.linear(xb[:, :K], w, b, dt), z)


def test_p6_equal_shape_group_equals_batched_matmul():
    """batch fusion: stack -> one batched multiply -> unbind (Fig. 4)."""
    rng = np.random.default_rng(13)
    n, M, N, K = 5, 6, 8, 16
    members = []
    for i in range(n):
        x, w, b = _rand_linear(rng, M, N, K, BF16)
        members.append(dict(x=x, w=w, b=b, act=0))
    z64, ys = graphs.linear_group(members, BF16)
    X = np.stack([wl.f32_from_bf16_bits(m["x"]).astype(np.float64) for m in members])
    W = np.stack([wl.f32_from_bf16_bits(m["w"]).astype(np.float64) for m in members])
    B = np.stack([wl.f32_from_bf16_bits(m["b"]).astype(np.float64) for m in members])
    Z = np.matmul(X, W.transpose(0, 2, 1)) + B[:, None, :]
    for i in range(n):
        assert np.allclose(z64[i], Z[i], rtol=1e-13, atol=1e-13)
    # the concat slotting: member i occupies columns [i*N, (i+1)*N)
    _, ycat = graphs.linear_group_concat(members, BF16)
    for i in range(n):
        assert np.array_equal(ycat[:, i * N:(i + 1) * N], ys[i])


# ------------------------------------------------------------------- P7 -----
def test_p7_layernorm_closed_forms():
    cfg = wl.config1(seed=1, rows=32, n=8)
    for m in cfg["members"]:
        x = m["x"]
        eps = float(np.float32(m["eps"]))
        y, xh = oracle.layernorm(x, m["gamma"], m["beta"], m["eps"], BF16, return_xhat=True)
        xd = wl.f32_from_bf16_bits(x).astype(np.float64)
        v = xd.var(axis=1)                                     # biased variance (library)
        assert np.all(np.abs(xh.mean(axis=1)) <= 1e-6)         # north_star invariant: mean 0
        assert np.all(np.abs(xh.var(axis=1) - v / (v + eps)) <= 1e-6)      # Q5 closed form
        _, xh0 = oracle.layernorm(x, None, None, 0.0, BF16, return_xhat=True)
        assert np.all(np.abs(xh0.var(axis=1) - 1.0) <= 1e-6)   # north_star invariant, literally, at eps=0
        assert np.all(np.abs(xh0.mean(axis=1)) <= 1e-6)
        # affine: y = xhat*gamma + beta
        g = wl.f32_from_bf16_bits(m["gamma"]).astype(np.float64)
        b = wl.f32_from_bf16_bits(m["beta"]).astype(np.float64)
        assert np.allclose(y, xh * g + b, rtol=0, atol=1e-14)
        # against the textbook formula through numpy
        ref = (xd - xd.mean(axis=1, keepdims=True)) / np.sqrt(v + eps)[:, None] * g + b
        assert np.allclose(y, ref, rtol=1e-12, atol=1e-12)


def test_p7_layernorm_shift_and_scale_invariance():
    rng = np.random.default_rng(3)
    x = rng.integers(-20, 20, size=(6, 24)).astype(np.float32)     # exact in fp32 after shift/scale
    y = oracle.layernorm(x, None, None, 1e-5, F32)
    y_shift = oracle.layernorm(x + np.float32(64.0), None, None, 1e-5, F32)
    assert np.allclose(y, y_shift, rtol=0, atol=1e-12)             # LN(x+c) = LN(x)
    eps = float(np.float32(1e-5))
    a = 4.0
    y_scale = oracle.layernorm(x * np.float32(a), None, None, np.float32(a * a * eps), F32)
    assert np.allclose(y, y_scale, rtol=0, atol=1e-9)               # LN_{a^2 eps}(a x) = LN_eps(x)
    # a wrong sign of the normalisation or un-biased variance would fail:
    xd = x.astype(np.float64)
    unbiased = (xd - xd.mean(1, keepdims=True)) / np.sqrt(xd.var(1, ddof=1) + eps)[:, None]
    assert not np.allclose(y, unbiased, rtol=0, atol=1e-4)


# ------------------------------------------------------------- P8, Q13 ------
def test_p8_pointwise_identities_and_values():
    xs = np.linspace(-12, 12, 4801)
    t = oracle.activation(xs, 2)
    s = oracle.activation(xs, 3)
    r = oracle.activation(xs, 1)
    assert np.allclose(oracle.activation(-xs, 2), -t, rtol=0, atol=0)           # odd
    assert np.allclose(s + oracle.activation(-xs, 3), 1.0, rtol=0, atol=4e-16)
    assert np.allclose(t, 2 * oracle.activation(2 * xs, 3) - 1, rtol=0, atol=1e-15)
    assert np.array_equal(oracle.activation(r, 1), r) and np.array_equal(r, np.maximum(xs, 0))
    assert np.array_equal(oracle.activation(xs, 0), xs)
    # textbook values
    v = oracle.activation(np.array([0.0, 1.0, -1.0, 0.5]), 2)
    assert v[0] == 0.0 and abs(v[1] - 0.7615941559557649) < 1e-15 and abs(v[3] - 0.46211715726000974) < 1e-15
    v = oracle.activation(np.array([0.0, 1.0, -1.0, 40.0, -40.0]), 3)
    assert v[0] == 0.5 and abs(v[1] - 0.7310585786300049) < 1e-15 and abs(v[2] - 0.2689414213699951) < 1e-15
    assert abs(v[4] - math.exp(-40.0)) < 1e-30 and v[3] == 1.0
    # against the C library through python's math module
    for x in (-3.3, -0.1, 1e-9, 0.7, 5.0):
        assert abs(oracle.activation(np.array([x]), 2)[0] - math.tanh(x)) <= 2e-16
        assert abs(oracle.activation(np.array([x]), 3)[0] - 1 / (1 + math.exp(-x))) <= 2e-16


def test_q13_special_values():
    sp = np.array([np.nan, np.inf, -np.inf, -0.0, 0.0])
    r = oracle.activation(sp, 1)
    assert np.isnan(r[0]) and r[1] == np.inf and r[2] == 0 and r[3] == 0 and r[4] == 0
    t = oracle.activation(sp, 2)
    assert np.isnan(t[0]) and t[1] == 1 and t[2] == -1 and t[3] == 0 and np.signbit(t[3])
    s = oracle.activation(sp, 3)
    assert np.isnan(s[0]) and s[1] == 1 and s[2] == 0 and s[3] == 0.5
    # pointwise on storage applies the same function to the widened value
    x = bf16([[-2.0, -0.5, 0.0, 0.5, 3.0]])
    for op in (0, 1, 2, 3):
        assert np.array_equal(oracle.pointwise(x, op, BF16)[0],
                              oracle.activation(np.array([-2.0, -0.5, 0.0, 0.5, 3.0]), op))


# ------------------------------------------------------------- P9, P11 ------
def test_p9_small_integer_case_is_exact():
    rng = np.random.default_rng(9)
    for (M, N, K, lim) in [(8, 16, 16, 3), (4, 8, 256, 1)]:
        X = rng.integers(-lim, lim + 1, size=(M, K))
        W = rng.integers(-lim, lim + 1, size=(N, K))
        b = rng.integers(-lim, lim + 1, size=(N,))
        Z = X @ W.T + b                                       # exact integer arithmetic
        assert np.abs(Z).max() < 256
        for dt in (F32, BF16):
            z = oracle.linear(st(X, dt), st(W, dt), st(b, dt), dt)
            assert np.array_equal(z, Z.astype(np.float64))
            y = oracle.round_to_storage(oracle.activation(z, 1), dt)
            assert np.array_equal(y, st(np.maximum(Z, 0), dt))


def test_p11_linearity_in_x_with_power_of_two():
    rng = np.random.default_rng(10)
    x, w, b = _rand_linear(rng, 6, 10, 24, F32)
    z = oracle.linear(x, w, b, F32)
    bd = b.astype(np.float64)
    for alpha in (2.0, 0.25, -8.0):
        za = oracle.linear(x * np.float32(alpha), w, b, F32)
        assert np.array_equal(za, alpha * (z - bd) + bd) or np.allclose(za, alpha * (z - bd) + bd, rtol=1e-15, atol=1e-15)
    # dropping the bias term would fail this:
    z0 = oracle.linear(x, w, None, F32)
    assert np.allclose(z - z0, np.broadcast_to(bd, z.shape), rtol=0, atol=1e-15)


# ------------------------------------------------- config graphs (Q2, Q14) --
def test_config0_graph_separate_equals_concat_slots():
    cfg = wl.config0()
    z64, ys = graphs.linear_group(cfg["members"], F32)
    _, ycat = graphs.linear_group_concat(cfg["members"], F32)
    assert ycat.shape == (64, 160)
    off = 0
    for m, y in zip(cfg["members"], ys):
        assert y.shape == (64, m["N"]) and np.array_equal(ycat[:, off:off + m["N"]], y)
        off += m["N"]
    assert all(np.all(np.abs(z) < 1) for z in z64)            # tanh range


def test_config3_graph_permutation_direction():
    cfg = wl.config3(seed=3, rows=4, width=256, nchunks=8)
    out64, out = graphs.split_pointwise_cat(cfg["x"], cfg["widths"], cfg["ops"], cfg["perm"], BF16)
    xd = wl.f32_from_bf16_bits(cfg["x"]).astype(np.float64)
    starts = np.concatenate(([0], np.cumsum(cfg["widths"])))
    d = 0
    for j, p in enumerate(cfg["perm"]):                       # output position j holds SOURCE chunk perm[j]
        w = cfg["widths"][p]
        src = xd[:, starts[p]:starts[p] + w]
        assert np.array_equal(out64[:, d:d + w], oracle.activation(src, cfg["ops"][p]))
        d += w
    assert d == 256 and out.shape == (4, 256)
    assert sum(cfg["widths"]) == 256 and all(w % 8 == 0 and w > 0 for w in cfg["widths"])
    assert sorted(cfg["perm"]) == list(range(8))


def test_workload_draws_are_reproducible_and_shaped():
    a, b = wl.config2(seed=2, M=8, n=16), wl.config2(seed=2, M=8, n=16)
    assert all(np.array_equal(p["x"], q["x"]) and p["K"] == q["K"] for p, q in zip(a["members"], b["members"]))
    assert {m["K"] for m in a["members"]} <= {128, 256, 512, 1024}
    c = wl.config2(seed=102, M=8, n=16)
    assert [m["K"] for m in c["members"]] != [m["K"] for m in a["members"]]
    c1 = wl.config1(seed=1, rows=4096, n=4)
    for m in c1["members"]:
        xd = wl.f32_from_bf16_bits(m["x"]).astype(np.float64)
        assert abs(xd.mean() - m["mu"]) < 0.1 * m["sigma"] and abs(xd.std() - m["sigma"]) < 0.05 * m["sigma"]
    c3 = wl.config3()
    assert len(c3["widths"]) == 256 and sum(c3["widths"]) == 8192 and c3["x"].shape == (8192, 8192)
    xd = wl.f32_from_bf16_bits(c3["x"][:64]).astype(np.float64)
    assert abs(xd.var() - 2.0) < 0.05


# ------------------------------------------------- linear2 --
def test_linear2_small_integers_exact_and_rounding_point():
    """Two chained Linear layers: with small integers every intermediate is an exactly representable
    integer, so the chain must equal numpy's integer arithmetic bit for bit -- pins operand order, bias,
    where the ReLU sits and that W2 multiplies the HIDDEN tensor (not x)."""
    rng = np.random.default_rng(5)
    M, K, H, N = 7, 16, 24, 8
    x = rng.integers(-2, 3, (M, K)); w1 = rng.integers(-2, 3, (H, K)); b1 = rng.integers(-2, 3, (H,))
    w2 = rng.integers(-1, 2, (N, H)); b2 = rng.integers(-2, 3, (N,))
    h = np.maximum(x @ w1.T + b1, 0)                       # |h| <= 16*4+2 = 66: exact in bf16
    y = h @ w2.T + b2                                      # |y| <= 24*66+2 < 2^11 but needs 8 bits: keep small
    assert np.abs(y).max() < 256 * 8
    m = dict(x=bf16(x), w1=bf16(w1), b1=bf16(b1), w2=bf16(w2), b2=bf16(b2), act1=1, act2=0)
    r = graphs.linear2(m, BF16)
    assert np.array_equal(r["h64"], h.astype(np.float64))
    assert np.array_equal(wl.f32_from_bf16_bits(r["h"]), h.astype(np.float32))
    assert np.array_equal(r["y64"], y.astype(np.float64))
    # the hidden tensor is ROUNDED to bf16 before the second layer (reading Q3): 257 is not a bf16 value
    m2 = dict(x=bf16([[1.0]]), w1=bf16([[257.0 - 1.0]]), b1=bf16([1.0]), w2=bf16([[1.0]]), b2=None, act1=0, act2=0)
    r2 = graphs.linear2(m2, BF16)
    assert r2["h64"][0, 0] == 257.0 and wl.f32_from_bf16_bits(r2["h"])[0, 0] == 256.0 and r2["y64"][0, 0] == 256.0


def test_linear2_identity_second_layer_returns_hidden():
    """W2 = I, b2 = 0, act2 = none: y equals the rounded hidden tensor bit for bit (and tanh hidden values
    equal the oracle's own single-layer group, which P5/P8 pin separately)."""
    H = 16
    m = dict(x=wl.tensor_normal(9, 1, (5, 32), 0, 1, BF16), w1=wl.tensor_normal(9, 2, (H, 32), 0, 32 ** -0.5, BF16),
             b1=wl.tensor_normal(9, 3, (H,), 0, 0.1, BF16), w2=bf16(np.eye(H)), b2=None, act1=2, act2=0)
    r = graphs.linear2(m, BF16)
    assert r["y"].tobytes() == r["h"].tobytes()
    ref = np.tanh(wl.f32_from_bf16_bits(m["x"]).astype(np.float64) @ wl.f32_from_bf16_bits(m["w1"]).astype(np.float64).T
                  + wl.f32_from_bf16_bits(m["b1"]).astype(np.float64))
    assert np.allclose(r["h64"], ref, rtol=1e-13, atol=1e-15)


def test_ln_linear2_sign_rows_reduce_to_integer_chain_and_affine_invariance():
    """LayerNorm folded into the chain (reading Q25).  Rows made of equally many -1 and +1 have mean 0 and variance
    1, so with eps = 0 the normalised row IS the row, and with small integer gamma / beta the whole chain is integer
    arithmetic: must equal numpy's integers bit for bit (pins: gamma multiplies before beta is added, LN feeds W1,
    ReLU sits after the first layer, W2 multiplies the hidden tensor).  Layer norm is invariant under x -> a x + c
    (a > 0) when eps = 0: the same rows mapped to {2, 8} give the same result to rounding.  A row that is NOT
    pre-normalised is checked against a literal numpy transcription of torch's layer_norm formula."""
    rng = np.random.default_rng(11)
    M, K, H, N = 6, 16, 24, 8
    x = np.stack([rng.permutation(np.repeat([-1, 1], K // 2)) for _ in range(M)])
    g = rng.integers(-2, 3, (K,)); be = rng.integers(-2, 3, (K,))
    w1 = rng.integers(-2, 3, (H, K)); b1 = rng.integers(-2, 3, (H,))
    w2 = rng.integers(-1, 2, (N, H)); b2 = rng.integers(-2, 3, (N,))
    xn = x * g + be
    h = np.maximum(xn @ w1.T + b1, 0)                      # |h| <= 16*4*2+2 = 130: exact in bf16
    y = h @ w2.T + b2
    m = dict(x=bf16(x), gamma=bf16(g), beta=bf16(be), eps=0.0, w1=bf16(w1), b1=bf16(b1), w2=bf16(w2), b2=bf16(b2), act1=1, act2=0)
    r = graphs.ln_linear2(m, BF16)
    assert np.array_equal(r["xn64"], xn.astype(np.float64))
    assert np.array_equal(r["h64"], h.astype(np.float64)) and np.array_equal(r["y64"], y.astype(np.float64))
    m2 = dict(m, x=bf16(3 * x + 5))                        # {-1, 1} -> {2, 8}: same normalised rows
    r2 = graphs.ln_linear2(m2, BF16)
    assert np.allclose(r2["y64"], y, rtol=0, atol=1e-9)
    # general rows, eps > 0: literal formula in numpy
    xg = wl.tensor_normal(12, 1, (5, K), 1.5, 2.0, BF16)
    m3 = dict(m, x=xg, eps=1e-5, act1=2)
    xd = wl.f32_from_bf16_bits(xg).astype(np.float64)
    mu = xd.mean(1, keepdims=True); v = ((xd - mu) ** 2).mean(1, keepdims=True)
    xn3 = (xd - mu) / np.sqrt(v + np.float64(np.float32(1e-5))) * g + be
    h3 = np.tanh(xn3 @ w1.T + b1)
    r3 = graphs.ln_linear2(m3, BF16)
    assert np.allclose(r3["h64"], h3, rtol=1e-12, atol=1e-13)
    # the fused op skips exactly one rounding of the unfused graph (Q3 vs Q25): results agree to bf16 resolution
    t = graphs.recsys_tower(dict(x=xg, gamma=m["gamma"], beta=m["beta"], eps=1e-5, w1=m["w1"], b1=m["b1"], w2=m["w2"], b2=m["b2"]), BF16)
    r4 = graphs.ln_linear2(dict(m3, act1=1), BF16)
    assert np.abs(r4["y64"] - t["out64"]).max() <= 2.0 ** -6 * np.abs(t["out64"]).max()


def test_linear_f64x_and_colsum_hand_values_and_agreement_with_linear():
    """oracle_linear_f64x (first layer of the LayerNorm-folded chain, reading Q25) and oracle_colsum (bias gradient):
    the plain C++ loops, no BLAS.  Pins: an asymmetric hand-computed 2x3x2 case whose activations are NOT storage
    values (a swapped operand, a dropped bias or a transposed index fails it); on activations that ARE storage
    values it equals `linear` bit for bit (same summation order); against numpy's matmul to 1e-13; colsum on a
    strided slice by hand and against numpy."""
    x64 = np.array([[1.5, -2.0, 0.25], [3.0, 0.5, -1.0]])
    w = np.array([[1, 2, 3], [4, 5, 6]], dtype=np.float32)
    b = np.array([10, 20], dtype=np.float32)
    assert np.array_equal(oracle.linear_f64x(x64, w, b, F32), [[8.25, 17.5], [11.0, 28.5]])
    assert np.array_equal(oracle.linear_f64x(x64, w, None, F32), [[-1.75, -2.5], [1.0, 8.5]])
    third = np.array([[1.0 / 3.0, 0.0, 0.0]])                       # not representable in fp32 / bf16: stays fp64
    assert oracle.linear_f64x(third, w, None, F32)[0, 1] == 4.0 * (1.0 / 3.0)
    xs = wl.tensor_normal(31, 1, (7, 19), 0.0, 1.0, BF16); ws = wl.tensor_normal(31, 2, (5, 19), 0.0, 0.3, BF16)
    bs = wl.tensor_normal(31, 3, (5,), 0.0, 0.3, BF16)
    assert oracle.linear_f64x(oracle.widen(xs, BF16), ws, bs, BF16).tobytes() == oracle.linear(xs, ws, bs, BF16).tobytes()
    xr = np.random.default_rng(5).standard_normal((6, 19))
    ref = xr @ oracle.widen(ws, BF16).T + oracle.widen(bs, BF16)
    assert np.allclose(oracle.linear_f64x(xr, ws, bs, BF16), ref, rtol=1e-13, atol=1e-14)
    wide = np.arange(24, dtype=np.float32).reshape(4, 6)            # column slice [1:4] of a [4, 6] buffer
    assert np.array_equal(oracle.colsum(wide[:, 1:4], F32), [1 + 7 + 13 + 19, 2 + 8 + 14 + 20, 3 + 9 + 15 + 21])
    g = wl.tensor_normal(31, 4, (53, 12), 0.0, 1.0, BF16)
    assert np.allclose(oracle.colsum(g, BF16), oracle.widen(g, BF16).sum(axis=0), rtol=0, atol=1e-12)


def test_saved_activation_fp8_is_quantisation_of_the_rounded_output():
    """Reading Q29: the FP8 copy a fused epilogue emits is the quantisation of the ROUNDED storage-dtype output (what
    the unfused graph's separate quantise op reads), not of the fp64 / fp32 pre-rounding value.  Hand case where the
    two differ: z = 1.0625 + 2^-9 (bf16 keeps 8 significand bits: rounds DOWN to 1.0625 = 17/16, a tie between the
    E4M3 neighbours 1.0 and 1.125 -> ties-to-even gives 1.0 = code 0x38; quantising z itself rounds UP to 1.125 =
    0x39).  Also: the composition equals the two ops applied by hand, codes of integer outputs are exact."""
    zval = 1.0625 + 2.0 ** -9          # built as a K = 2 dot product (zval itself is not a bf16 value)
    m = dict(x=bf16(np.array([[1.0, 1.0]])), w=bf16(np.array([[1.0625, 2.0 ** -9]])), b=None, act=0)
    y64, y, codes = graphs.linear_member_fp8(m, 1.0, BF16)
    assert y64[0, 0] == zval and wl.f32_from_bf16_bits(y)[0, 0] == 1.0625
    assert codes[0, 0] == 0x38 and oracle.quant_e4m3(np.array([[zval]], dtype=np.float32), 1.0, F32)[0, 0] == 0x39
    rng = np.random.default_rng(3)
    mi = dict(x=bf16(rng.integers(-1, 2, (5, 8))), w=bf16(rng.integers(-1, 2, (6, 8))), b=bf16(rng.integers(-2, 3, (6,))), act=1)
    y64, y, codes = graphs.linear_member_fp8(mi, 0.5, BF16)
    assert y64.max() <= 10 and np.array_equal(oracle.dequant_e4m3(codes, 2.0), y64)       # n / 2, n <= 15: 4 significant bits, exact codes
    ln = dict(x=wl.tensor_normal(41, 1, (7, 24), 0.5, 2.0, BF16), gamma=wl.tensor_normal(41, 2, (24,), 1.0, 0.3, BF16),
              beta=wl.tensor_normal(41, 3, (24,), 0.0, 0.3, BF16), eps=1e-5)
    y64, y, codes = graphs.layernorm_fp8(ln, 16.0, BF16)
    assert y.tobytes() == oracle.round_to_storage(oracle.layernorm(ln["x"], ln["gamma"], ln["beta"], 1e-5, BF16), BF16).tobytes()
    assert codes.tobytes() == oracle.quant_e4m3(y, 16.0, BF16).tobytes()


# --------------------------------- Table-1 pointwise patterns --
def test_pointwise_ext_hand_values_and_special_values():
    """batch_clamp / batch_nan_to_num / batch_aten_sub,div,mul against hand-computed values (torch semantics)."""
    inf, nan = float("inf"), float("nan")
    x = np.array([[-3.0, -0.5, 0.0, 0.75, 2.0, 100.0, inf, -inf]], dtype=np.float32)
    y = oracle.pointwise_ext(x, None, oracle.PW_CLAMP, [-1.0, 1.5], F32)
    assert np.array_equal(y, np.array([[-1.0, -0.5, 0.0, 0.75, 1.5, 1.5, 1.5, -1.0]]))
    xn = np.array([[nan, 1.0]], dtype=np.float32)
    yn = oracle.pointwise_ext(xn, None, oracle.PW_CLAMP, [-1.0, 1.5], F32)
    assert np.isnan(yn[0, 0]) and yn[0, 1] == 1.0                      # NaN propagates through clamp
    # lo > hi: torch.clamp returns hi everywhere (min(max(x, lo), hi))
    assert np.array_equal(oracle.pointwise_ext(x[:, :4], None, oracle.PW_CLAMP, [2.0, 1.0], F32), np.full((1, 4), 1.0))
    z = np.array([[nan, inf, -inf, 3.5, -0.0]], dtype=np.float32)
    w = oracle.pointwise_ext(z, None, oracle.PW_NAN_TO_NUM, [7.0, 9.0, -9.0], F32)
    assert np.array_equal(w[0, :4], [7.0, 9.0, -9.0, 3.5]) and w[0, 4] == 0.0 and np.signbit(w[0, 4])
    a = bf16([[6.0, -1.5, 0.25, 8.0]]); b = bf16([[2.0, 0.5, -4.0, 0.0]])
    assert np.array_equal(oracle.pointwise_ext(a, b, oracle.PW_SUB, [], BF16), [[4.0, -2.0, 4.25, 8.0]])
    assert np.array_equal(oracle.pointwise_ext(a, b, oracle.PW_MUL, [], BF16), [[12.0, -0.75, -1.0, 0.0]])
    d = oracle.pointwise_ext(a, b, oracle.PW_DIV, [], BF16)
    assert np.array_equal(d[0, :3], [3.0, -3.0, -0.0625]) and d[0, 3] == inf


def test_pointwise_ext_identities_on_random_data():
    a = wl.tensor_normal(13, 1, (6, 40), 0.0, 2.0, BF16)
    b = wl.tensor_normal(13, 2, (6, 40), 1.0, 3.0, BF16)
    a64, b64 = oracle.widen(a, BF16), oracle.widen(b, BF16)
    assert np.array_equal(oracle.pointwise_ext(a, b, oracle.PW_SUB, [], BF16), a64 - b64)          # numpy, not the oracle
    assert np.array_equal(oracle.pointwise_ext(a, b, oracle.PW_MUL, [], BF16), oracle.pointwise_ext(b, a, oracle.PW_MUL, [], BF16))
    assert np.array_equal(oracle.pointwise_ext(a, a, oracle.PW_DIV, [], BF16), np.ones((6, 40)))
    c = oracle.pointwise_ext(a, None, oracle.PW_CLAMP, [-1.0, 1.0], BF16)
    assert np.array_equal(c, np.clip(a64, -1.0, 1.0)) and np.array_equal(np.clip(c, -1.0, 1.0), c)    # idempotent
    assert np.array_equal(oracle.pointwise_ext(a, None, oracle.PW_CLAMP, [-np.inf, np.inf], BF16), a64)
    assert np.array_equal(oracle.pointwise_ext(a, None, oracle.PW_NAN_TO_NUM, [0.0, 1.0, -1.0], BF16), a64)   # finite: untouched


def test_relu_backward_hand_values_and_finite_differences():
    """ReLU backward (op 11: the ReLU epilogue of a grouped Linear in a post-grad graph, PAPER.md:292
    batch_linear_post_grad): hand values incl. both zeros, then the derivative of a numpy ReLU by central
    differences, and the two mask sources (forward output / forward input) agreeing."""
    g = np.array([[1.5, -2.0, 3.0, 4.0, -5.0, 6.0]], dtype=np.float32)
    y = np.array([[2.0, 0.0, -0.0, -1.0, 1e-30, 0.5]], dtype=np.float32)
    got = oracle.pointwise_ext(g, y, oracle.PW_RELU_BWD, [], F32)
    assert np.array_equal(got, np.array([[1.5, 0.0, 0.0, 0.0, -5.0, 6.0]]))
    # numpy forward, perturbed: d/dx sum(relu(x) * g) = g * [x > 0] away from the kink
    x = wl.tensor_normal(17, 1, (5, 24), 0.0, 1.0, F32)
    x = np.where(np.abs(x) < 1e-2, np.float32(0.5), x)
    gg = wl.tensor_normal(17, 2, (5, 24), 0.0, 1.0, F32)
    x64, g64, h = x.astype(np.float64), gg.astype(np.float64), 1e-4
    fd = ((np.maximum(x64 + h, 0.0) - np.maximum(x64 - h, 0.0)) / (2 * h)) * g64
    assert np.allclose(oracle.pointwise_ext(gg, x, oracle.PW_RELU_BWD, [], F32), fd, rtol=0, atol=1e-9)
    out = np.maximum(x, np.float32(0.0))                  # mask from the forward OUTPUT: same gradient
    assert np.array_equal(oracle.pointwise_ext(gg, out, oracle.PW_RELU_BWD, [], F32),
                          oracle.pointwise_ext(gg, x, oracle.PW_RELU_BWD, [], F32))
    # bf16 storage: the gradient passes through bit-exactly where the mask is on
    gb = wl.tensor_normal(17, 3, (4, 16), 0.0, 3.0, BF16); mb = wl.tensor_normal(17, 4, (4, 16), 0.0, 1.0, BF16)
    r = oracle.pointwise_ext(gb, mb, oracle.PW_RELU_BWD, [], BF16)
    assert np.array_equal(r, np.where(oracle.widen(mb, BF16) > 0, oracle.widen(gb, BF16), 0.0))


def test_tanh_and_sigmoid_backward_hand_values_and_finite_differences():
    """Ops 12 / 13 (backward of the tanh / sigmoid epilogues, PAPER.md:292 batch_linear_post_grad on post-grad graphs):
    hand values at outputs where the closed form is a short decimal, then central differences of numpy's own
    tanh / logistic through the forward output, and the limits y -> +-1 (tanh) and y -> 0, 1 (sigmoid): gradient 0."""
    g = np.array([[2.0, -4.0, 1.0, 8.0]], dtype=np.float32)
    y = np.array([[0.5, -0.5, 0.0, 1.0]], dtype=np.float32)
    assert np.array_equal(oracle.pointwise_ext(g, y, oracle.PW_TANH_BWD, [], F32), [[1.5, -3.0, 1.0, 0.0]])
    ys = np.array([[0.5, 0.25, 0.0, 1.0]], dtype=np.float32)
    assert np.array_equal(oracle.pointwise_ext(g, ys, oracle.PW_SIGMOID_BWD, [], F32), [[0.5, -0.75, 0.0, 0.0]])
    z = wl.tensor_normal(18, 1, (6, 20), 0.0, 1.5, F32).astype(np.float64)
    gg = wl.tensor_normal(18, 2, (6, 20), 0.0, 1.0, F32)
    h = 1e-5
    for op, f in ((oracle.PW_TANH_BWD, np.tanh), (oracle.PW_SIGMOID_BWD, lambda t: 1.0 / (1.0 + np.exp(-t)))):
        fd = (f(z + h) - f(z - h)) / (2 * h) * gg.astype(np.float64)
        out32 = f(z).astype(np.float32)                                  # the stored forward output (fp32 storage)
        got = oracle.pointwise_ext(gg, out32, op, [], F32)
        assert np.allclose(got, fd, rtol=0, atol=2e-6), np.abs(got - fd).max()      # fp32 rounding of y: 6e-8 * |dy/dy| terms
    # the two ops differ (a swapped op code fails): at y = 0.5, tanh' = 0.75, sigmoid' = 0.25
    half = np.full((1, 1), 0.5, dtype=np.float32); one = np.ones((1, 1), dtype=np.float32)
    assert oracle.pointwise_ext(one, half, oracle.PW_TANH_BWD, [], F32)[0, 0] == 0.75
    assert oracle.pointwise_ext(one, half, oracle.PW_SIGMOID_BWD, [], F32)[0, 0] == 0.25
    # bf16 storage: widened exactly, product in fp64
    gb = wl.tensor_normal(18, 3, (4, 16), 0.0, 3.0, BF16); yb = wl.tensor_uniform(18, 4, (4, 16), -1.0, 1.0, BF16)
    a, b = oracle.widen(gb, BF16), oracle.widen(yb, BF16)
    assert np.array_equal(oracle.pointwise_ext(gb, yb, oracle.PW_TANH_BWD, [], BF16), a * (1.0 - b * b))
    assert np.array_equal(oracle.pointwise_ext(gb, yb, oracle.PW_SIGMOID_BWD, [], BF16), a * ((1.0 - b) * b))


# ------------------------------------------ backward of the grouped Linear --
def test_linear_backward_integers_and_adjointness():
    """dgrad / wgrad against numpy integer arithmetic (exact), and the adjoint identities that DEFINE them:
    <dY, X W^T> = <dY W, X> = <dY^T X, W> on random bf16 data (fp64 sums agree to rounding)."""
    rng = np.random.default_rng(21)
    M, N, K = 9, 6, 11
    dy = rng.integers(-3, 4, (M, N)); w = rng.integers(-3, 4, (N, K)); x = rng.integers(-3, 4, (M, K))
    assert np.array_equal(graphs.linear_dgrad(bf16(dy), bf16(w)), (dy @ w).astype(np.float64))
    assert np.array_equal(graphs.linear_wgrad(bf16(dy), bf16(x)), (dy.T @ x).astype(np.float64))
    dyr = wl.tensor_normal(31, 1, (M, N), 0, 1, BF16); wr = wl.tensor_normal(31, 2, (N, K), 0, 1, BF16)
    xr = wl.tensor_normal(31, 3, (M, K), 0, 1, BF16)
    y64 = oracle.linear(xr, wr, None, BF16)
    lhs = float((oracle.widen(dyr, BF16) * y64).sum())
    assert abs(lhs - float((graphs.linear_dgrad(dyr, wr) * oracle.widen(xr, BF16)).sum())) <= 1e-12 * max(1.0, abs(lhs))
    assert abs(lhs - float((graphs.linear_wgrad(dyr, xr) * oracle.widen(wr, BF16)).sum())) <= 1e-12 * max(1.0, abs(lhs))


# --------------------------------------------- LayerNorm backward --
def test_bias_grad_and_full_linear_relu_backward_by_finite_differences():
    """linear_bias_grad: hand values; equals dY^T . 1 through the pinned `linear`; and the whole backward of
    relu(x W^T + b) (mask, db, dX, dW) against central differences of a NUMPY forward in fp64."""
    dz = np.array([[1.0, -2.0, 0.5], [3.0, 4.0, -0.5], [-1.0, 0.25, 8.0]], dtype=np.float32)
    assert np.array_equal(graphs.linear_bias_grad(dz, F32), [3.0, 2.25, 8.0])
    g = wl.tensor_normal(23, 1, (37, 12), 0.0, 1.0, F32)
    ones = np.ones((37, 1), dtype=np.float32)
    assert np.allclose(graphs.linear_bias_grad(g, F32), graphs.linear_wgrad(g, ones, F32)[:, 0], rtol=0, atol=1e-12)
    x = wl.tensor_normal(23, 2, (9, 6), 0.0, 1.0, F32); w = wl.tensor_normal(23, 3, (5, 6), 0.0, 0.5, F32)
    b = wl.tensor_normal(23, 4, (5,), 0.0, 0.5, F32); dy = wl.tensor_normal(23, 5, (9, 5), 0.0, 1.0, F32)
    r = graphs.linear_relu_backward(dict(x=x, w=w, b=b), dy, F32)
    x64, w64, b64, dy64 = (a.astype(np.float64) for a in (x, w, b, dy))
    loss = lambda xx, ww, bb: float((np.maximum(xx @ ww.T + bb, 0.0) * dy64).sum())
    assert np.abs(x64 @ w64.T + b64).min() > 1e-3                       # no pre-activation sits on the kink
    h = 1e-6
    def fd(a, which):
        out = np.zeros_like(a)
        for idx in np.ndindex(a.shape):
            ap, am = a.copy(), a.copy(); ap[idx] += h; am[idx] -= h
            args_p = [x64, w64, b64]; args_m = [x64, w64, b64]
            args_p[which], args_m[which] = ap, am
            out[idx] = (loss(*args_p) - loss(*args_m)) / (2 * h)
        return out
    assert np.allclose(r["db64"], fd(b64, 2), rtol=0, atol=1e-6)
    assert np.allclose(r["dx64"], fd(x64, 0), rtol=0, atol=1e-6)
    assert np.allclose(r["dw64"], fd(w64, 1), rtol=0, atol=1e-6)


@pytest.mark.parametrize("act", [2, 3])
def test_full_linear_tanh_sigmoid_backward_by_finite_differences(act):
    """graphs.linear_act_backward for the tanh / sigmoid epilogues against central differences of a NUMPY fp64 forward
    (fp32 storage: the stored output carries a 6e-8 rounding, the gate is 1e-5); act = 1 equals linear_relu_backward."""
    x = wl.tensor_normal(24, 2, (9, 6), 0.0, 1.0, F32); w = wl.tensor_normal(24, 3, (5, 6), 0.0, 0.5, F32)
    b = wl.tensor_normal(24, 4, (5,), 0.0, 0.5, F32); dy = wl.tensor_normal(24, 5, (9, 5), 0.0, 1.0, F32)
    r = graphs.linear_act_backward(dict(x=x, w=w, b=b), dy, act, F32)
    x64, w64, b64, dy64 = (a.astype(np.float64) for a in (x, w, b, dy))
    f = np.tanh if act == 2 else (lambda t: 1.0 / (1.0 + np.exp(-t)))
    loss = lambda xx, ww, bb: float((f(xx @ ww.T + bb) * dy64).sum())
    h = 1e-6
    def fd(a, which):
        out = np.zeros_like(a)
        for idx in np.ndindex(a.shape):
            ap, am = a.copy(), a.copy(); ap[idx] += h; am[idx] -= h
            args_p = [x64, w64, b64]; args_m = [x64, w64, b64]
            args_p[which], args_m[which] = ap, am
            out[idx] = (loss(*args_p) - loss(*args_m)) / (2 * h)
        return out
    assert np.allclose(r["db64"], fd(b64, 2), rtol=0, atol=1e-5)
    assert np.allclose(r["dx64"], fd(x64, 0), rtol=0, atol=1e-5)
    assert np.allclose(r["dw64"], fd(w64, 1), rtol=0, atol=1e-5)
    r1, r0 = graphs.linear_act_backward(dict(x=x, w=w, b=b), dy, 1, F32), graphs.linear_relu_backward(dict(x=x, w=w, b=b), dy, F32)
    assert all(np.array_equal(r1[k], r0[k]) for k in r0)


def test_layernorm_backward_finite_differences_and_identities():
    """dx, dgamma, dbeta against central finite differences of the oracle's OWN forward are not a pin (same code
    base), so the forward used here is numpy's: L(x, gamma, beta) = sum(dy * LN(x)) in fp64.  Plus the closed forms:
    every dx row sums to 0; with eps = 0 it is also orthogonal to xhat; dbeta = column sums of dy."""
    rng = np.random.default_rng(17)
    rows, D, eps = 5, 12, 1e-5
    x = rng.normal(0.5, 2.0, (rows, D)).astype(np.float32)
    dy = rng.normal(0.0, 1.0, (rows, D)).astype(np.float32)
    gamma = rng.normal(1.0, 0.3, (D,)).astype(np.float32)
    beta = rng.normal(0.0, 0.3, (D,)).astype(np.float32)
    e32 = float(np.float32(eps))

    def ln(xx, gg, bb):
        mu = xx.mean(axis=1, keepdims=True)
        v = ((xx - mu) ** 2).mean(axis=1, keepdims=True)
        return (xx - mu) / np.sqrt(v + e32) * gg + bb
    loss = lambda xx, gg, bb: float((dy.astype(np.float64) * ln(xx, gg, bb)).sum())
    x64, g64, b64 = x.astype(np.float64), gamma.astype(np.float64), beta.astype(np.float64)
    dx, dg, db = oracle.layernorm_backward(x, dy, gamma, eps, F32)
    h = 1e-6
    for (r, j) in [(0, 0), (2, 5), (4, 11), (1, 7)]:
        xp, xm = x64.copy(), x64.copy(); xp[r, j] += h; xm[r, j] -= h
        assert abs((loss(xp, g64, b64) - loss(xm, g64, b64)) / (2 * h) - dx[r, j]) <= 1e-7 * max(1.0, abs(dx[r, j]))
    for j in (0, 3, 11):
        gp, gm = g64.copy(), g64.copy(); gp[j] += h; gm[j] -= h
        assert abs((loss(x64, gp, b64) - loss(x64, gm, b64)) / (2 * h) - dg[j]) <= 1e-7 * max(1.0, abs(dg[j]))
    assert np.allclose(db, dy.astype(np.float64).sum(axis=0), rtol=1e-14, atol=1e-14)
    assert np.abs(dx.sum(axis=1)).max() <= 1e-12
    dx0, _, _ = oracle.layernorm_backward(x, dy, gamma, 0.0, F32)
    mu = x64.mean(axis=1, keepdims=True)
    xh = (x64 - mu) / np.sqrt(((x64 - mu) ** 2).mean(axis=1, keepdims=True))
    assert np.abs((dx0 * xh).sum(axis=1)).max() <= 1e-12
    # gamma = None means 1
    dx1, dg1, _ = oracle.layernorm_backward(x, dy, None, eps, F32)
    dx2, dg2, _ = oracle.layernorm_backward(x, dy, np.ones(D, np.float32), eps, F32)
    assert np.array_equal(dx1, dx2) and np.array_equal(dg1, dg2)


# -------------------------------- FP8 E4M3 activation quantisation --
def _e4m3_from_definition(c):
    """value of a code from the format definition (OCP FP8 E4M3: bias 7, no infinities, S.1111.111 = NaN)."""
    e, m = (c >> 3) & 0xF, c & 7
    if e == 0xF and m == 7:
        return float("nan")
    v = m * 2.0 ** -9 if e == 0 else (1 + m / 8.0) * 2.0 ** (e - 7)
    return -v if c & 0x80 else v


def test_e4m3_decode_exhaustive_and_encode_ties_saturation():
    codes = np.arange(256, dtype=np.uint8).reshape(1, 256)
    vals = oracle.dequant_e4m3(codes, 1.0)[0]
    ref = np.array([_e4m3_from_definition(int(c)) for c in range(256)])
    assert np.array_equal(np.isnan(vals), np.isnan(ref)) and np.array_equal(vals[~np.isnan(ref)], ref[~np.isnan(ref)])
    assert vals[0x7E] == 448.0 and vals[0x01] == 2.0 ** -9 and vals[0x08] == 2.0 ** -6
    # encode: every finite code maps to itself; midpoints between neighbours go to the EVEN code; just off the
    # midpoint goes to the nearer one; beyond 448 saturates; NaN stays NaN; inf saturates (satfinite)
    pos = np.array([_e4m3_from_definition(c) for c in range(0x7F)])
    enc = lambda a: oracle.quant_e4m3(np.asarray(a, dtype=np.float32).reshape(1, -1), 1.0, F32)[0]
    assert np.array_equal(enc(pos), np.arange(0x7F)) and np.array_equal(enc(-pos[1:]), np.arange(1, 0x7F) | 0x80)
    mids = (pos[:-1] + pos[1:]) / 2                       # exactly representable in fp32
    got = enc(mids)
    want = np.where(np.arange(0x7E) % 2 == 0, np.arange(0x7E), np.arange(1, 0x7F))
    assert np.array_equal(got, want)
    assert np.array_equal(enc(np.nextafter(mids.astype(np.float32), np.float32(np.inf))), np.arange(1, 0x7F))
    assert np.array_equal(enc(np.nextafter(mids.astype(np.float32), np.float32(0))), np.arange(0x7E))
    assert list(enc([448.0, 449.0, 1e9, np.inf, -np.inf, -500.0])) == [0x7E, 0x7E, 0x7E, 0x7E, 0xFE, 0xFE]
    assert enc([np.nan])[0] & 0x7F == 0x7F
    # scaling: quantise(x, s) == quantise(x * s, 1) for a power-of-two scale; dequantise multiplies back
    x = wl.tensor_normal(51, 1, (4, 64), 0, 3.0, BF16)
    q = oracle.quant_e4m3(x, 0.25, BF16)
    assert np.array_equal(q, enc(wl.f32_from_bf16_bits(x).reshape(-1) * 0.25).reshape(4, 64))
    assert np.array_equal(oracle.dequant_e4m3(q, 4.0), oracle.dequant_e4m3(q, 1.0) * 4.0)
