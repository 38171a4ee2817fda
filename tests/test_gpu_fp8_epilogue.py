"""GPU parity: the FP8 (E4M3) copy of the output written by the grouped Linear's and the batched LayerNorm's own
epilogue (activation_quantization_aten_pass fused into the op that produces the saved activation, PAPER.md:341-345,
:487-489).  Reading Q29: the codes are the quantisation of the ROUNDED bf16 output, so they must
equal, bit for bit, (a) the two-launch path (op, then OPT_PW_QUANT_E4M3 on its stored output) and (b) the oracle's
quant_e4m3 fed with the GPU's own bf16 output (the decision on the kernel's fp32 product, reading Q24); the bf16
output itself is gated against the oracle as in the plain tests and must not change when the FP8 copy is requested."""
import numpy as np
import pytest
import torch

import oracle
from oracle import graphs
import workloads as wl
from util import BF16, F32, bf16_ulp_distance, empty_dev, row_l2_rel_err, to_dev, to_host

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def codes_of(y_bits, scale):
    """oracle codes of a stored bf16 tensor, decided on the kernel's fp32 product (reading Q24)."""
    prod32 = (wl.f32_from_bf16_bits(y_bits) * np.float32(scale)).astype(np.float32)
    return oracle.quant_e4m3(prod32, 1.0, F32)


def same_codes(got, ref):
    nan = (ref & 0x7F) == 0x7F              # the sign of a NaN code is not part of the contract
    return np.array_equal(got[~nan], ref[~nan]) and np.all((got[nan] & 0x7F) == 0x7F)


def mk(seed, i, M, N, K, act, std=1.0):
    return dict(M=M, N=N, K=K, act=act,
                x=wl.tensor_normal(seed, 3 * i + 1, (M, K), 0, std, BF16),
                w=wl.tensor_normal(seed, 3 * i + 2, (N, K), 0, K ** -0.5, BF16),
                b=wl.tensor_normal(seed, 3 * i + 3, (N,), 0, 0.1, BF16))


@pytest.mark.parametrize("cta_pair", [0, 1])
def test_linear_fp8_copy_equals_two_launch_path_and_oracle(ob, cta_pair):
    shapes = [(300, 64, 64, 1), (257, 256, 128, 0), (513, 512, 72, 2), (130, 144, 200, 3), (1000, 1024, 256, 1), (64, 16, 32, 0)]
    scales = [16.0, 3.3, 0.25, 100.0, 7.0, 448.0]
    members = [mk(71, i, M, N, K, act, std=1.0 + i) for i, (M, N, K, act) in enumerate(shapes)]
    dev, descs, plain = [], [], []
    for m, sc in zip(members, scales):
        x, w, b = to_dev(m["x"], BF16), to_dev(m["w"], BF16), to_dev(m["b"], BF16)
        y = empty_dev((m["M"], m["N"]), BF16, fill=float("nan"))
        y0 = empty_dev((m["M"], m["N"]), BF16, fill=float("nan"))
        y8 = torch.full((m["M"], m["N"] + 16), 0xAA, dtype=torch.uint8, device="cuda")        # padded rows: ldy8 > N
        y8only = torch.full((m["M"], m["N"]), 0xAA, dtype=torch.uint8, device="cuda")
        dev.append((x, w, b, y, y0, y8, y8only))
        descs.append(ob.linear_member(x, w, b, y, m["act"], 0, y8[:, :m["N"]], sc))
        plain.append(ob.linear_member(x, w, b, y0, m["act"]))
    opts = ob.opt_linear_options(cta_pair=cta_pair)
    p = ob.opt_linear_plan_create_ex(descs, BF16, 0, opts)
    p0 = ob.opt_linear_plan_create_ex(plain, BF16, 0, opts)
    only = ob.opt_linear_plan_create_ex([ob.linear_member(x, w, b, None, m["act"], 0, y8only, sc)
                                         for (x, w, b, _, _, _, y8only), m, sc in zip(dev, members, scales)], BF16, 0, opts)
    n0 = ob.opt_launch_count()
    p.launch(); p0.launch(); only.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 3
    info, info0, info_only = p.info(), p0.info(), only.info()
    mn = sum(m["M"] * m["N"] for m in members)
    assert info["bytes"] - info0["bytes"] == mn and info0["bytes"] - info_only["bytes"] == mn      # +1 byte / -2 +1 bytes per element
    # two-launch path: quantise the stored output of the plain plan
    q2 = [torch.empty((m["M"], m["N"]), dtype=torch.uint8, device="cuda") for m in members]
    ob.opt_pointwise_plan_create([ob.chunk(d[4], q, ob.OPT_PW_QUANT_E4M3, None, [sc]) for d, q, sc in zip(dev, q2, scales)], BF16).launch()
    torch.cuda.synchronize()
    for (x, w, b, y, y0, y8, y8only), m, sc, q in zip(dev, members, scales, q2):
        yb = to_host(y)
        assert yb.tobytes() == to_host(y0).tobytes()                       # asking for the FP8 copy does not change Y
        assert row_l2_rel_err(yb, graphs.linear_member(m, BF16), BF16) <= 1e-2
        got = y8.cpu().numpy()
        assert np.all(got[:, m["N"]:] == 0xAA), "wrote outside the member's columns"
        assert np.array_equal(got[:, :m["N"]], q.cpu().numpy())            # == op then OPT_PW_QUANT_E4M3, bit for bit
        assert same_codes(got[:, :m["N"]], codes_of(yb, sc))               # == oracle on the GPU's own bf16 output
        assert np.array_equal(y8only.cpu().numpy(), got[:, :m["N"]])       # FP8-only members write the same codes


def test_linear_fp8_copy_into_a_concat_slot_and_mixed_members(ob):
    """members with and without an FP8 copy in one group; the copies land in column slots of ONE uint8 concat buffer."""
    cfg = wl.config2(M=384, n=10)
    ms = cfg["members"]
    width = cfg["concat_width"]
    ycat = empty_dev((384, width), BF16, fill=float("nan"))
    y8cat = torch.full((384, width), 0xAA, dtype=torch.uint8, device="cuda")
    keep, descs = [], []
    for i, m in enumerate(ms):
        x, w, b = to_dev(m["x"], BF16), to_dev(m["w"], BF16), to_dev(m["b"], BF16)
        keep.append((x, w, b))
        sl = slice(m["col_off"], m["col_off"] + m["N"])
        descs.append(ob.linear_member(x, w, b, ycat[:, sl], m["act"], 0, y8cat[:, sl] if i % 3 != 1 else None, 8.0))
    ob.opt_linear_plan_create(descs, BF16).launch()
    torch.cuda.synchronize()
    y, y8 = to_host(ycat), y8cat.cpu().numpy()
    for i, m in enumerate(ms):
        sl = slice(m["col_off"], m["col_off"] + m["N"])
        assert row_l2_rel_err(y[:, sl], graphs.linear_member(m, BF16), BF16) <= 1e-2
        if i % 3 != 1:
            assert same_codes(y8[:, sl], codes_of(y[:, sl], 8.0))
        else:
            assert np.all(y8[:, sl] == 0xAA)


def test_linear_fp8_integers_bit_exact_against_the_oracle_graph(ob):
    """small integers: Y and its codes are exact, so the whole fused op must equal graphs.linear_member_fp8 bit for bit."""
    rng = np.random.default_rng(5)
    members = []
    for (M, N, K) in [(200, 64, 16), (129, 128, 24), (300, 256, 8)]:
        members.append(dict(M=M, N=N, K=K, act=1, x=wl.bf16_bits_from_f32(rng.integers(-1, 2, (M, K)).astype(np.float32)),
                            w=wl.bf16_bits_from_f32(rng.integers(-1, 2, (N, K)).astype(np.float32)),
                            b=wl.bf16_bits_from_f32(rng.integers(-2, 3, (N,)).astype(np.float32))))
    dev = [(to_dev(m["x"], BF16), to_dev(m["w"], BF16), to_dev(m["b"], BF16), empty_dev((m["M"], m["N"]), BF16),
            torch.empty((m["M"], m["N"]), dtype=torch.uint8, device="cuda")) for m in members]
    ob.opt_linear_plan_create([ob.linear_member(x, w, b, y, 1, 0, y8, 0.5) for x, w, b, y, y8 in dev], BF16).launch()
    torch.cuda.synchronize()
    for (x, w, b, y, y8), m in zip(dev, members):
        _, yref, cref = graphs.linear_member_fp8(m, 0.5, BF16)
        assert to_host(y).tobytes() == yref.tobytes() and y8.cpu().numpy().tobytes() == cref.tobytes()


def test_layernorm_fp8_copy_equals_two_launch_path_and_oracle(ob):
    shapes = [(300, 32), (1000, 64), (77, 128), (2048, 256), (129, 512), (64, 1032), (5, 2048), (513, 200), (8192, 64)]
    scales = [16.0, 3.3, 0.25, 100.0, 7.0, 30.0, 1.0, 64.0, 12.0]
    ms, dev, descs, plain, only = [], [], [], [], []
    for i, ((rows, D), sc) in enumerate(zip(shapes, scales)):
        m = dict(x=wl.tensor_normal(81, 4 * i + 1, (rows, D), 0.3 * i, 1.0 + i, BF16), gamma=wl.tensor_normal(81, 4 * i + 2, (D,), 1.0, 0.3, BF16),
                 beta=wl.tensor_normal(81, 4 * i + 3, (D,), 0.0, 0.3, BF16), eps=1e-5)
        if i == 2:
            m["gamma"] = None
        ms.append(m)
        x = to_dev(m["x"], BF16)
        g = to_dev(m["gamma"], BF16) if m["gamma"] is not None else None
        b = to_dev(m["beta"], BF16)
        y, y0 = empty_dev((rows, D), BF16, fill=float("nan")), empty_dev((rows, D), BF16, fill=float("nan"))
        y8 = torch.full((rows, D + 8), 0xAA, dtype=torch.uint8, device="cuda")
        y8o = torch.full((rows, D), 0xAA, dtype=torch.uint8, device="cuda")
        dev.append((x, g, b, y, y0, y8, y8o))
        want8 = i != 3                                           # one member of the group without an FP8 copy
        descs.append(ob.layernorm_member(x, y, g, b, 1e-5, y8[:, :D] if want8 else None, sc))
        plain.append(ob.layernorm_member(x, y0, g, b, 1e-5))
        only.append(ob.layernorm_member(x, None, g, b, 1e-5, y8o, sc))
    p, p0, po = (ob.opt_layernorm_plan_create(d, BF16) for d in (descs, plain, only))
    n0 = ob.opt_launch_count()
    p.launch(); p0.launch(); po.launch()
    torch.cuda.synchronize()
    assert ob.opt_launch_count() - n0 == 3
    for i, ((x, g, b, y, y0, y8, y8o), m, sc) in enumerate(zip(dev, ms, scales)):
        D = m["x"].shape[1]
        yb = to_host(y)
        assert yb.tobytes() == to_host(y0).tobytes()
        got = y8.cpu().numpy()
        assert np.all(got[:, D:] == 0xAA)
        if i == 3:
            assert np.all(got == 0xAA)
        else:
            assert same_codes(got[:, :D], codes_of(yb, sc))
        assert same_codes(y8o.cpu().numpy(), codes_of(yb, sc))
        ref = oracle.round_to_storage(oracle.layernorm(m["x"], m.get("gamma"), m["beta"], 1e-5, BF16), BF16)
        assert np.percentile(bf16_ulp_distance(yb, ref), 99.9) <= 2


def test_fp8_epilogue_errors(ob):
    x = empty_dev((64, 64), BF16, fill=1.0); w = empty_dev((64, 64), BF16, fill=1.0); y = empty_dev((64, 64), BF16)
    y8 = torch.empty((64, 64), dtype=torch.uint8, device="cuda")
    for bad_scale in (0.0, -1.0, float("inf"), float("nan")):
        with pytest.raises(ob.OptError) as e:
            ob.opt_linear_plan_create([ob.linear_member(x, w, None, y, 0, 0, y8, bad_scale)], BF16)
        assert e.value.status == ob.OPT_ERR_INVALID_ARG
        with pytest.raises(ob.OptError) as e:
            ob.opt_layernorm_plan_create([ob.layernorm_member(x, y, None, None, 1e-5, y8, bad_scale)], BF16)
        assert e.value.status == ob.OPT_ERR_INVALID_ARG
    with pytest.raises(ob.OptError) as e:                       # N % 16
        ob.opt_linear_plan_create([ob.linear_member(x[:, :64], w[:24], None, y[:, :24], 0, 0, y8[:, :24], 1.0)], BF16)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
    with pytest.raises(ob.OptError) as e:                       # neither output
        ob.opt_linear_plan_create([ob.opt_linear_member(x.data_ptr(), 64, w.data_ptr(), 64, None, None, 0, 64, 64, 64, 0, 0, None, 0, 0.0)], BF16)
    assert e.value.status == ob.OPT_ERR_INVALID_ARG
    xf = empty_dev((64, 64), F32, fill=1.0); yf = empty_dev((64, 64), F32)
    with pytest.raises(ob.OptError) as e:                       # fp32 activations: not implemented
        ob.opt_layernorm_plan_create([ob.layernorm_member(xf, yf, None, None, 1e-5, y8, 1.0)], F32)
    assert e.value.status == ob.OPT_ERR_UNSUPPORTED
