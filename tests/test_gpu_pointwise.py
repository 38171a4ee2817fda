"""GPU parity: multi_pointwise_splitcat vs the CPU oracle (through the C ABI)."""
import numpy as np
import pytest
import torch

import oracle
from oracle import graphs
import workloads as wl
from util import BF16, F32, bf16_ulp_distance, empty_dev, to_dev, to_host

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def run_split_cat(ob, x_host, widths, ops, perm, dt=BF16):
    x = to_dev(x_host, dt)
    out = empty_dev(x.shape, dt, fill=float("nan"))
    plan = ob.opt_pointwise_plan_create(ob.split_cat_chunks(x, out, widths, ops, perm), dt)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1 and plan.info()["launches"] == 1
    return to_host(out), plan


@pytest.mark.parametrize("dt", [BF16, F32])
def test_paper_listing2_example_bit_exact(ob, dt):
    """PAPER.md:403-416 Listing 2 == Listing 1 (return x).  Widths are in units the
    alignment rule allows (x8 for bf16, x4 for fp32): [2,4] -> [2*V, 4*V], second split (2*V, 2*V)."""
    V = 8 if dt == BF16 else 4
    x_host = wl.tensor_normal(7, 1, (2, 6 * V), 0, 1, dt)
    widths = [2 * V, 2 * V, 2 * V]          # item0, item2, item3 of the listing
    got, _ = run_split_cat(ob, x_host, widths, [0, 0, 0], [0, 1, 2], dt)
    assert got.tobytes() == x_host.tobytes()
    fs = oracle.split(x_host, [2 * V, 4 * V])
    ref = oracle.cat([fs[0]] + oracle.split(fs[1], [2 * V, 2 * V]))
    assert got.tobytes() == ref.tobytes()


@pytest.mark.parametrize("seed", [3, 103, 203])
def test_config3_small_movement_and_math(ob, seed):
    cfg = wl.config3(seed=seed, rows=200, width=2048, nchunks=64)      # ragged rows, several column blocks
    x, widths, ops, perm = cfg["x"], cfg["widths"], cfg["ops"], cfg["perm"]
    # (i) every op = COPY: bit-exact column permutation
    got, _ = run_split_cat(ob, x, widths, [0] * len(widths), perm)
    assert got.tobytes() == graphs.split_copy_cat(x, widths, perm).tobytes()
    # (ii) identity permutation + COPY: split o cat = identity
    got, _ = run_split_cat(ob, x, widths, [0] * len(widths), list(range(len(widths))))
    assert got.tobytes() == x.tobytes()
    # (iii) real ops: <= 2 bf16 ulp of the oracle; ReLU chunks bit-exact
    got, plan = run_split_cat(ob, x, widths, ops, perm)
    ref64, ref = graphs.split_pointwise_cat(x, widths, ops, perm, BF16)
    d = bf16_ulp_distance(got, ref)
    assert d.max() <= 2, "max ulp %d" % d.max()
    pos = 0
    for p in perm:
        if ops[p] == wl.gen.PW_RELU:
            assert np.array_equal(bf16_ulp_distance(got[:, pos:pos + widths[p]], ref[:, pos:pos + widths[p]]),
                                  np.zeros((200, widths[p]), dtype=np.int64))
        pos += widths[p]
    assert plan.info()["bytes"] == 2 * x.size * 2


def test_multi_tensor_standalone_all_ops(ob):
    """batch_relu / batch_sigmoid / batch_aten_tanh / batch_detach: n separate tensors, ragged sizes."""
    shapes = [(1, 8), (3, 24), (64, 64), (257, 136), (1000, 512), (5, 8 * 1031), (2, 8 * 600)]
    xs = [wl.tensor_normal(11, i + 1, s, 0, 2.0, BF16) for i, s in enumerate(shapes)]
    ops = [i % 4 for i in range(len(shapes))]
    dx = [to_dev(x, BF16) for x in xs]
    dy = [empty_dev(x.shape, BF16, fill=float("nan")) for x in xs]
    plan = ob.opt_pointwise_plan_create([ob.chunk(a, b, op) for a, b, op in zip(dx, dy, ops)], BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    for x, y, op in zip(xs, dy, ops):
        ref = oracle.round_to_storage(oracle.pointwise(x, op, BF16), BF16)
        d = bf16_ulp_distance(to_host(y), ref)
        assert d.max() <= (0 if op in (0, 1) else 2), (x.shape, op, d.max())


def test_strided_chunks_and_in_place(ob):
    base = wl.tensor_normal(12, 1, (100, 320), 0, 1.5, BF16)
    b = to_dev(base, BF16)
    # in place tanh on a column slice, relu on another, rest untouched
    chunks = [ob.chunk(b[:, 8:72], b[:, 8:72], ob.OPT_PW_TANH), ob.chunk(b[:, 200:264], b[:, 200:264], ob.OPT_PW_RELU)]
    ob.opt_pointwise_plan_create(chunks, BF16).launch()
    torch.cuda.synchronize()
    got = to_host(b)
    ref = base.copy()
    ref[:, 8:72] = oracle.round_to_storage(oracle.pointwise(base[:, 8:72], 2, BF16), BF16)
    ref[:, 200:264] = oracle.round_to_storage(oracle.pointwise(base[:, 200:264], 1, BF16), BF16)
    assert bf16_ulp_distance(got, ref).max() <= 2
    assert np.array_equal(got[:, :8], base[:, :8]) and np.array_equal(got[:, 72:200], base[:, 72:200])


def test_special_values_q13(ob):
    vals = np.array([np.nan, np.inf, -np.inf, -0.0, 0.0, 1e-30, -1e-30, 88.0, -88.0, 100.0, -100.0, 3e38, -3e38,
                     1e-3, -1e-3, 20.0], dtype=np.float32)
    x = wl.bf16_bits_from_f32(vals).reshape(1, 16)
    x[0, 0] = 0x7FC0
    for op in (1, 2, 3):
        dx = to_dev(x, BF16)
        dy = empty_dev(x.shape, BF16)
        ob.opt_pointwise_plan_create([ob.chunk(dx, dy, op)], BF16).launch()
        torch.cuda.synchronize()
        ref = oracle.round_to_storage(oracle.pointwise(x, op, BF16), BF16)
        d = bf16_ulp_distance(to_host(dy), ref)
        assert d.max() <= 2, (op, to_host(dy), ref)


def test_fp32_io(ob):
    x = wl.tensor_normal(13, 1, (77, 100), 0, 2.0, F32)
    for op in (0, 1, 2, 3):
        dx, dy = to_dev(x, F32), empty_dev(x.shape, F32)
        ob.opt_pointwise_plan_create([ob.chunk(dx, dy, op)], F32).launch()
        torch.cuda.synchronize()
        ref = oracle.pointwise(x, op, F32)
        got = to_host(dy).astype(np.float64)
        if op in (0, 1):
            assert np.array_equal(got, ref)
        else:   # fp32 libdevice tanhf/expf: a few fp32 ulp
            assert np.all(np.abs(got - ref) <= 4 * 2.0 ** -23 * np.maximum(np.abs(ref), 2.0 ** -20))


def test_errors_launch_nothing(ob):
    x = empty_dev((16, 64), BF16, fill=0.0)
    y = empty_dev((16, 64), BF16, fill=0.0)
    n0 = ob.opt_launch_count()
    with pytest.raises(ob.OptError) as e:
        ob.opt_pointwise_plan_create([ob.chunk(x[:, :36], y[:, :36])], BF16)         # width % 8
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
    with pytest.raises(ob.OptError) as e:
        ob.opt_pointwise_plan_create([ob.chunk(x[:, :32], y[:, :32]), ob.chunk(x[:, 32:], y[:, 24:56])], BF16)
    assert e.value.status == ob.OPT_ERR_ALIAS
    with pytest.raises(ob.OptError) as e:
        ob.opt_pointwise_plan_create([], BF16)
    assert e.value.status == ob.OPT_ERR_INVALID_ARG
    assert ob.opt_launch_count() == n0


# ---------------------------------------------- Table-1 patterns beyond relu/tanh/sigmoid --
def _special(a_bits):
    """sprinkle NaN / +inf / -inf / -0 into a bf16 bit array."""
    a = a_bits.copy().reshape(-1)
    a[3::97] = 0x7FC0; a[5::101] = 0x7F80; a[7::103] = 0xFF80; a[11::107] = 0x8000
    return a.reshape(a_bits.shape)


def test_table1_patterns_one_launch_mixed_group(ob):
    """batch_clamp, batch_nan_to_num, batch_aten_sub / div / mul and a relu member in ONE launch: dense tensors,
    strided column slices, special values; <= 2 bf16 ulp of the oracle, special values exactly."""
    ops = [(oracle.PW_CLAMP, [-0.75, 1.25]), (oracle.PW_NAN_TO_NUM, [0.5, 100.0, -100.0]), (oracle.PW_SUB, []),
           (oracle.PW_DIV, []), (oracle.PW_MUL, []), (oracle.PW_CLAMP, [2.0, 1.0]), (oracle.PW_MUL, [])]
    shapes = [(300, 512), (77, 200), (1000, 64), (129, 1032), (64, 8), (5, 4096), (513, 256)]
    host, chunks, keep = [], [], []
    for i, ((op, prm), (r, w)) in enumerate(zip(ops, shapes)):
        a = _special(wl.tensor_normal(41, 2 * i + 1, (r, w), 0.0, 2.0, BF16))
        b = wl.tensor_normal(41, 2 * i + 2, (r, w), 0.5, 1.5, BF16) if op >= oracle.PW_SUB else None
        strided = i % 2 == 1                               # odd members: column slices of wider buffers
        pad = 16 if strided else 0
        da = to_dev(np.pad(a, ((0, 0), (0, pad))), BF16)[:, :w] if strided else to_dev(a, BF16)
        db = None if b is None else (to_dev(np.pad(b, ((0, 0), (8, pad))), BF16)[:, 8:8 + w] if strided else to_dev(b, BF16))
        dd = empty_dev((r, w + pad), BF16, fill=float("nan"))[:, :w]
        chunks.append(ob.chunk(da, dd, op, db, prm))
        host.append((a, b, op, prm))
        keep.append((da, db, dd))
    x = wl.tensor_normal(41, 99, (256, 256), 0, 1, BF16)   # a plain relu member rides in the same launch
    dx, dy = to_dev(x, BF16), empty_dev((256, 256), BF16)
    chunks.append(ob.chunk(dx, dy, ob.OPT_PW_RELU))
    plan = ob.opt_pointwise_plan_create(chunks, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    for (a, b, op, prm), (_, _, dd) in zip(host, keep):
        ref = oracle.round_to_storage(oracle.pointwise_ext(a, b, op, prm, BF16), BF16)
        got = to_host(dd)
        d = bf16_ulp_distance(got, ref)
        assert d.max() <= 2, (op, int(d.max()))
        if op in (oracle.PW_CLAMP, oracle.PW_NAN_TO_NUM, oracle.PW_MUL):
            nan = (ref & 0x7FFF) > 0x7F80                  # NaN stays NaN (payload is not part of the contract)
            assert np.array_equal(got[~nan], ref[~nan]) and np.all((got[nan] & 0x7FFF) > 0x7F80)   # else exact
    assert bf16_ulp_distance(to_host(dy), oracle.round_to_storage(oracle.pointwise(x, 1, BF16), BF16)).max() == 0


def test_table1_patterns_fp32_and_errors(ob):
    a = wl.tensor_normal(42, 1, (100, 36), 0, 2, F32)
    b = wl.tensor_normal(42, 2, (100, 36), 1, 1, F32)
    da, db = to_dev(a, F32), to_dev(b, F32)
    outs = [empty_dev((100, 36), F32) for _ in range(3)]
    plan = ob.opt_pointwise_plan_create([ob.chunk(da, outs[0], ob.OPT_PW_DIV, db), ob.chunk(da, outs[1], ob.OPT_PW_SUB, db),
                                         ob.chunk(da, outs[2], ob.OPT_PW_CLAMP, None, [-1.0, 0.5])], F32)
    plan.launch()
    torch.cuda.synchronize()
    for o, op, prm in zip(outs, (oracle.PW_DIV, oracle.PW_SUB, oracle.PW_CLAMP), ([], [], [-1.0, 0.5])):
        ref = oracle.round_to_storage(oracle.pointwise_ext(a, b if op != oracle.PW_CLAMP else None, op, prm, F32), F32)
        assert np.array_equal(to_host(o), ref)             # fp32: IEEE sub / div, correctly rounded
    with pytest.raises(ob.OptError) as e:                  # binary op without a second operand
        ob.opt_pointwise_plan_create([ob.chunk(da, outs[0], ob.OPT_PW_MUL)], F32)
    assert e.value.status == ob.OPT_ERR_INVALID_ARG
    with pytest.raises(ob.OptError) as e:                  # second operand overlaps another member's output
        ob.opt_pointwise_plan_create([ob.chunk(da, outs[0], ob.OPT_PW_MUL, db), ob.chunk(da, outs[1], ob.OPT_PW_MUL, outs[0])], F32)
    assert e.value.status == ob.OPT_ERR_ALIAS


def _quant_case(seed, i, rows, w, std, strided):
    a = _special(wl.tensor_normal(seed, i, (rows, w), 0.0, std, BF16))
    pad = 16 if strided else 0
    da = to_dev(np.pad(a, ((0, 0), (0, pad))), BF16)[:, :w]
    dq = torch.full((rows, w + pad), 0xAA, dtype=torch.uint8, device="cuda")[:, :w]
    return a, da, dq


def test_fp8_e4m3_quant_dequant_one_launch_each(ob):
    """activation_quantization_aten_pass: a group of saved activations -> FP8 E4M3 codes in one
    launch, and back in one launch.  The code is an integer decided by floating point: both sides decide it on the
    kernel's fp32 product x * scale (bit-exact); with a power-of-two scale that product is exact and the fp64 oracle
    on (x, scale) agrees too.  Dequantised values: exact (a 4-bit significand times a power of two fits bf16) for
    power-of-two scales, <= 1 bf16 ulp otherwise."""
    shapes = [(300, 512), (77, 200), (1000, 64), (129, 1032), (64, 8), (5, 4096), (2048, 256)]
    scales = [1.0, 0.25, 16.0, 0.7310791015625, 3.3, 1.0 / 448.0, 37.0]
    stds = [2.0, 100.0, 0.05, 1.0, 300.0, 1000.0, 3.0]
    host, chunks, keep = [], [], []
    for i, ((r, w), sc, sd) in enumerate(zip(shapes, scales, stds)):
        a, da, dq = _quant_case(51, i, r, w, sd, strided=i % 2 == 1)
        chunks.append(ob.chunk(da, dq, ob.OPT_PW_QUANT_E4M3, None, [sc]))
        host.append((a, sc))
        keep.append((da, dq))
    plan = ob.opt_pointwise_plan_create(chunks, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    codes = []
    for (a, sc), (_, dq) in zip(host, keep):
        got = dq.cpu().numpy()
        prod32 = (wl.f32_from_bf16_bits(a) * np.float32(sc)).astype(np.float32)       # the kernel's precision
        ref = oracle.quant_e4m3(prod32, 1.0, F32)
        assert np.array_equal(got, ref), (sc, int((got != ref).sum()))
        ref64 = oracle.quant_e4m3(a, sc, BF16)                                        # the plain fp64 definition
        bad = got != ref64
        if np.log2(sc) == np.round(np.log2(sc)):
            assert not bad.any()
        else:   # rounding the product to fp32 first can only move it onto / off a tie: adjacent code.  (Not always
            #       rare: with scale = fp32(1/448), x = 7 * odd * 2^n puts the fp32 product exactly on a tie.)
            assert bad.mean() < 0.05 and np.all(np.abs(got[bad].astype(int) - ref64[bad].astype(int)) <= 1)
        assert (got == 0x7F).sum() + (got == 0xFF).sum() == ((a & 0x7FFF) > 0x7F80).sum()   # NaN <-> NaN only
        codes.append(got)
    # untouched padding of the strided outputs
    for i, (_, dq) in enumerate(keep):
        if i % 2 == 1:
            base = dq.as_strided((dq.shape[0], dq.shape[1] + 16), (dq.stride(0), 1))
            assert bool((base[:, dq.shape[1]:] == 0xAA).all())

    # dequantise the codes back, one launch
    chunks, outs = [], []
    for i, ((a, sc), (_, dq)) in enumerate(zip(host, keep)):
        pad = 8 if i % 2 == 0 else 0
        dy = empty_dev((dq.shape[0], dq.shape[1] + pad), BF16, fill=float("nan"))[:, :dq.shape[1]]
        chunks.append(ob.chunk(dq, dy, ob.OPT_PW_DEQUANT_E4M3, None, [1.0 / sc]))
        outs.append(dy)
    plan = ob.opt_pointwise_plan_create(chunks, BF16)
    n0 = ob.opt_launch_count()
    plan.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 1
    for (a, sc), c, dy in zip(host, codes, outs):
        ref = oracle.round_to_storage(oracle.dequant_e4m3(c, 1.0 / sc), BF16)
        got = to_host(dy)
        d = bf16_ulp_distance(got, ref)
        pow2 = np.log2(sc) == np.round(np.log2(sc))
        assert d.max() <= (0 if pow2 else 1), (sc, int(d.max()))


def test_fp8_e4m3_all_codes_and_rounding_boundaries(ob):
    """every one of the 256 codes through dequantise (exact), and every bf16 value in [-2^10, 2^10] through quantise
    (all rounding ties, subnormal codes, saturation at 448, signed zero) bit-exact against the fp64 oracle."""
    c = np.arange(256, dtype=np.uint8).reshape(1, 256).repeat(3, 0)
    dc = torch.from_numpy(c).cuda()
    dy = empty_dev((3, 256), BF16)
    ob.opt_pointwise_plan_create([ob.chunk(dc, dy, ob.OPT_PW_DEQUANT_E4M3, None, [1.0])], BF16).launch()
    torch.cuda.synchronize()
    ref = oracle.round_to_storage(oracle.dequant_e4m3(c, 1.0), BF16)
    assert bf16_ulp_distance(to_host(dy), ref).max() == 0
    assert np.array_equal(to_host(dy)[:, :0x7F], ref[:, :0x7F]) and np.array_equal(to_host(dy)[:, 0x80:0xFF], ref[:, 0x80:0xFF])

    allb = np.arange(65536, dtype=np.uint32).astype(np.uint16).reshape(64, 1024)
    da = to_dev(allb, BF16)
    dq = torch.empty((64, 1024), dtype=torch.uint8, device="cuda")
    ob.opt_pointwise_plan_create([ob.chunk(da, dq, ob.OPT_PW_QUANT_E4M3, None, [1.0])], BF16).launch()
    torch.cuda.synchronize()
    got, ref = dq.cpu().numpy(), oracle.quant_e4m3(allb, 1.0, BF16)
    nan = (ref & 0x7F) == 0x7F                             # NaN -> NaN (the sign of a NaN code is not part of the contract)
    assert np.array_equal(got[~nan], ref[~nan]) and np.all((got[nan] & 0x7F) == 0x7F)


def test_fp8_errors(ob):
    a = empty_dev((16, 64), F32, fill=1.0)
    q = torch.empty((16, 64), dtype=torch.uint8, device="cuda")
    with pytest.raises(ob.OptError) as e:                  # fp32 activations: not implemented
        ob.opt_pointwise_plan_create([ob.chunk(a, q, ob.OPT_PW_QUANT_E4M3, None, [1.0])], F32)
    assert e.value.status == ob.OPT_ERR_UNSUPPORTED
    b = empty_dev((16, 64), BF16, fill=1.0)
    with pytest.raises(ob.OptError) as e:                  # fp8 row stride must keep 8-byte vectors aligned
        ob.opt_pointwise_plan_create([ob.chunk(b, torch.empty((16, 68), dtype=torch.uint8, device="cuda")[:, :64],
                                               ob.OPT_PW_QUANT_E4M3, None, [1.0])], BF16)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
