"""Plans are independent of one another (include/optimus_b200.h: "Different plans are independent"): a plan that
needs a lot of dynamic shared memory still launches after a LATER plan of the same kind was created with a small
request (the shared-memory opt-in is an attribute of the kernel function -- the last cudaFuncSetAttribute wins -- so
the library always sets the fixed maximum).  Every kernel that opts in is covered: staged LayerNorm, staged
split/cat, the chained Linear, the grouped GEMM."""
import numpy as np
import pytest
import torch

from util import BF16, to_host

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def _randn(shape, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    return torch.randn(*shape, device="cuda", generator=g).to(torch.bfloat16)


def _launch_bits(plan, out):
    out.fill_(float("nan"))
    plan.launch()
    torch.cuda.synchronize()          # a failed launch raises from plan.launch(); a fault would surface here
    return to_host(out).tobytes()


def test_layernorm_large_plan_survives_a_later_small_plan(ob):
    x = _randn((4096, 512), 1); y = torch.empty_like(x)
    g = _randn((512,), 2); b = _randn((512,), 3)
    big = ob.opt_layernorm_plan_create([ob.layernorm_member(x, y, g, b, 1e-5)], BF16)      # 4 stages x ~18 KB
    first = _launch_bits(big, y)
    xs = _randn((8, 64), 4); ys = torch.empty_like(xs)
    small = ob.opt_layernorm_plan_create([ob.layernorm_member(xs, ys, None, None, 1e-5)], BF16)   # a few KB
    small.launch()
    torch.cuda.synchronize()
    assert _launch_bits(big, y) == first
    # and the other order: a small plan first, then a large one, both stay launchable
    assert _launch_bits(small, ys) == _launch_bits(small, ys)
    assert _launch_bits(big, y) == first


def test_staged_splitcat_large_plan_survives_a_later_small_plan(ob):
    def plan_for(width, chunk, rows, seed):
        x = _randn((rows, width), seed); out = torch.empty_like(x)
        n = width // chunk
        perm = list(np.random.default_rng(seed).permutation(n))
        chunks = ob.split_cat_chunks(x, out, [chunk] * n, [ob.OPT_PW_COPY] * n, perm)
        ref = torch.cat([x[:, p * chunk:(p + 1) * chunk] for p in perm], dim=1)
        return ob.opt_pointwise_plan_create(chunks, BF16), out, to_host(ref).tobytes()
    big, big_out, big_ref = plan_for(8192, 32, 512, 5)       # 5 x 16 KB staged rows per block
    assert _launch_bits(big, big_out) == big_ref
    small, small_out, small_ref = plan_for(4096, 32, 64, 6)   # half of that: must not lower the big plan's limit
    assert _launch_bits(small, small_out) == small_ref
    assert _launch_bits(big, big_out) == big_ref
    wide, wide_out, wide_ref = plan_for(16384, 32, 300, 7)    # 32 KB rows: the staged destination row is given up
    assert _launch_bits(wide, wide_out) == wide_ref
    assert _launch_bits(big, big_out) == big_ref
    assert _launch_bits(small, small_out) == small_ref


def test_grouped_gemm_and_chained_linear_plans_are_independent(ob):
    x = _randn((512, 256), 8)
    w_wide = _randn((1024, 256), 9); y_wide = torch.empty(512, 1024, device="cuda", dtype=torch.bfloat16)
    w_narrow = _randn((16, 256), 10); y_narrow = torch.empty(512, 16, device="cuda", dtype=torch.bfloat16)
    wide = ob.opt_linear_plan_create([ob.linear_member(x, w_wide, None, y_wide, ob.OPT_ACT_RELU)], BF16)     # 6 x 32 KB ring
    first = _launch_bits(wide, y_wide)
    narrow = ob.opt_linear_plan_create([ob.linear_member(x, w_narrow, None, y_narrow, ob.OPT_ACT_NONE)], BF16)
    narrow.launch()
    w1 = _randn((128, 256), 11); w2 = _randn((64, 128), 12); y2 = torch.empty(512, 64, device="cuda", dtype=torch.bfloat16)
    chain = ob.opt_linear2_plan_create([ob.linear2_member(x, w1, None, w2, None, y2)], BF16)
    chain_first = _launch_bits(chain, y2)
    lnchain = ob.opt_ln_linear2_plan_create([ob.ln_linear2_member(x, None, None, 1e-5, w1, None, w2, None, y2)], BF16)
    lnchain.launch()
    torch.cuda.synchronize()
    assert _launch_bits(wide, y_wide) == first
    assert _launch_bits(chain, y2) == chain_first


def test_plan_create_leaves_the_current_device_alone(ob):
    before = torch.cuda.current_device()
    x = _randn((64, 64), 13); y = torch.empty_like(x)
    ob.opt_layernorm_plan_create([ob.layernorm_member(x, y, None, None, 1e-5)], BF16, None, before).launch()
    torch.cuda.synchronize()
    assert torch.cuda.current_device() == before
