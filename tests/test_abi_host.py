"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU,
exports every symbol include/optimus_b200.h declares, and validates descriptors on the host
before the first CUDA call (no compute here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    ob.lib()
    return ob


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "optimus_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(opt_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(ob):
    names = declared_symbols()
    assert {"opt_linear_plan_create", "opt_layernorm_plan_create", "opt_pointwise_plan_create", "opt_plan_launch",
            "opt_plan_launch_host", "opt_plan_info", "opt_plan_destroy", "opt_last_error", "opt_launch_count",
            "opt_version"} <= set(names)
    L = ctypes.CDLL(ob.lib_path())
    for n in names:
        assert hasattr(L, n), "symbol %s declared in the header but not exported" % n
    # and the Python binding carries the same names
    for n in names:
        assert hasattr(ob, n), "binding lacks %s" % n


def test_struct_layouts_match_header(ob):
    assert ctypes.sizeof(ob.opt_linear_member) == 104      # + y8, ldy8, scale8 (tests/test_header_is_c.py checks every offset against gcc)
    assert ctypes.sizeof(ob.opt_layernorm_member) == 88
    assert ctypes.sizeof(ob.opt_chunk) == 80
    assert ctypes.sizeof(ob.opt_linear2_member) == 104 and ctypes.sizeof(ob.opt_ln_linear2_member) == 128
    assert ctypes.sizeof(ob.opt_host_copy) == 32
    assert ctypes.sizeof(ob.opt_bias_grad_member) == 72 and ctypes.sizeof(ob.opt_layernorm_bwd_member) == 88


def test_sass_is_blackwell_native():
    """tcgen05.mma / tcgen05.ld / TMA show up as UTC*MMA / LDTM / UTMALDG+UTMASTG in the SASS."""
    import shutil
    import subprocess
    import paper_2607_02945_b200 as ob
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not installed")
    sass = subprocess.run([cuobjdump, "-sass", ob.lib_path()], capture_output=True, text=True).stdout
    for mnemonic in ("UTCHMMA", "LDTM", "UTMALDG", "UTMASTG"):
        assert mnemonic in sass, mnemonic
    assert "sm_100a" in sass


def dummy(addr):
    return ctypes.c_void_p(addr)


def test_host_validation_runs_before_any_cuda_call(ob):
    """INVALID_ARG / ALIGNMENT / ALIAS come back on a machine without a GPU; a valid group then
    fails with NO_DEVICE (never a CPU fallback)."""
    import torch
    A, B, Cc = 0x10000000, 0x20000000, 0x30000000
    mk = lambda **kw: ob.opt_linear_member(**{**dict(x=A, ldx=64, w=B, ldw=64, bias=None, y=Cc, ldy=64, M=128, N=64, K=64, act=0), **kw})
    for member, status in [(mk(ldx=60), ob.OPT_ERR_INVALID_ARG), (mk(ldx=68), ob.OPT_ERR_ALIGNMENT), (mk(x=A + 2), ob.OPT_ERR_ALIGNMENT),
                           (mk(M=0), ob.OPT_ERR_INVALID_ARG), (mk(act=9), ob.OPT_ERR_INVALID_ARG),
                           (mk(y=A), ob.OPT_ERR_ALIAS), (mk(ldy=32), ob.OPT_ERR_INVALID_ARG)]:
        with pytest.raises(ob.OptError) as e:
            ob.opt_linear_plan_create([member], ob.OPT_BF16)
        assert e.value.status == status, (e.value, status)
    with pytest.raises(ob.OptError) as e:     # two members writing overlapping concat slots
        ob.opt_linear_plan_create([mk(y=Cc, ldy=128), mk(y=Cc + 64, ldy=128)], ob.OPT_BF16)
    assert e.value.status == ob.OPT_ERR_ALIAS
    # adjacent, non-overlapping slots pass the host checks:
    if not torch.cuda.is_available():
        with pytest.raises(ob.OptError) as e:
            ob.opt_linear_plan_create([mk(y=Cc, ldy=128), mk(y=Cc + 128, ldy=128)], ob.OPT_BF16)
        assert e.value.status == ob.OPT_ERR_NO_DEVICE
        ln = ob.opt_layernorm_member(x=A, ldx=64, y=B, ldy=64, gamma=None, beta=None, rows=4, D=64, eps=1e-5)
        with pytest.raises(ob.OptError) as e:
            ob.opt_layernorm_plan_create([ln], ob.OPT_BF16)
        assert e.value.status == ob.OPT_ERR_NO_DEVICE
        ch = ob.opt_chunk(src=A, lds=64, dst=B, ldd=64, rows=4, width=64, op=0)
        with pytest.raises(ob.OptError) as e:
            ob.opt_pointwise_plan_create([ch], ob.OPT_BF16)
        assert e.value.status == ob.OPT_ERR_NO_DEVICE
    ln = ob.opt_layernorm_member(x=A, ldx=64, y=B, ldy=64, gamma=None, beta=None, rows=4, D=60, eps=1e-5)
    with pytest.raises(ob.OptError) as e:
        ob.opt_layernorm_plan_create([ln], ob.OPT_BF16)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
    ch = ob.opt_chunk(src=A, lds=64, dst=A + 64, ldd=64, rows=4, width=64, op=0)   # dst overlaps src rows
    with pytest.raises(ob.OptError) as e:
        ob.opt_pointwise_plan_create([ch], ob.OPT_BF16)
    assert e.value.status == ob.OPT_ERR_ALIAS
    assert ob.lib().opt_plan_launch(None, None) == ob.OPT_ERR_INVALID_ARG      # NULL plan: error, no launch
    assert "NULL" in ob.opt_last_error()
    assert ob.opt_launch_count() == 0


def test_host_validation_of_the_next_row_entry_points(ob):
    """the section-8(f) entry points validate on the host too: chained Linear (+ LayerNorm), LayerNorm backward,
    skinny groups (relaxed stride rule), extended / FP8 pointwise ops -- no GPU needed, nothing launched."""
    import torch
    A, B, Cc, D, E = 0x10000000, 0x20000000, 0x30000000, 0x40000000, 0x50000000
    l2 = lambda **kw: ob.opt_linear2_member(**{**dict(x=A, ldx=64, w1=B, ldw1=64, b1=None, w2=Cc, ldw2=128, b2=None, y=D, ldy=64,
                                                      M=256, K=64, H=128, N=64, act1=1, act2=0), **kw})
    for member, status in [(l2(K=512, ldx=512, ldw1=512), ob.OPT_ERR_UNSUPPORTED), (l2(H=1024, ldw2=1024), ob.OPT_ERR_UNSUPPORTED),
                           (l2(N=128, ldy=128), ob.OPT_ERR_UNSUPPORTED), (l2(H=120, ldw2=120), ob.OPT_ERR_ALIGNMENT),
                           (l2(y=A), ob.OPT_ERR_ALIAS), (l2(act1=7), ob.OPT_ERR_INVALID_ARG), (l2(ldw2=64), ob.OPT_ERR_INVALID_ARG)]:
        with pytest.raises(ob.OptError) as e:
            ob.opt_linear2_plan_create([member], ob.OPT_BF16)
        assert e.value.status == status, (e.value, status)
    with pytest.raises(ob.OptError) as e:
        ob.opt_linear2_plan_create([l2()], ob.OPT_F32)
    assert e.value.status == ob.OPT_ERR_UNSUPPORTED
    lnl = lambda chain, **kw: ob.opt_ln_linear2_member(**{**dict(chain=chain, gamma=E, beta=None, eps=1e-5, reserved=0), **kw})
    for member, status in [(lnl(l2(), eps=-1.0), ob.OPT_ERR_INVALID_ARG), (lnl(l2(), gamma=E + 2), ob.OPT_ERR_ALIGNMENT),
                           (lnl(l2(y=E)), ob.OPT_ERR_ALIAS), (lnl(l2(K=512, ldx=512, ldw1=512)), ob.OPT_ERR_UNSUPPORTED)]:
        with pytest.raises(ob.OptError) as e:
            ob.opt_ln_linear2_plan_create([member], ob.OPT_BF16)
        assert e.value.status == status, (e.value, status)
    # skinny groups: even row strides are enough, odd ones are not; a non-skinny member in the group restores ld % 8
    sk = lambda **kw: ob.opt_linear_member(**{**dict(x=A, ldx=4, w=B, ldw=4, bias=None, y=Cc, ldy=2, M=1000, N=2, K=4, act=0, layout=0), **kw})
    with pytest.raises(ob.OptError) as e:
        ob.opt_linear_plan_create([sk(ldx=5)], ob.OPT_BF16)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
    big = ob.opt_linear_member(x=D, ldx=64, w=E, ldw=64, bias=None, y=0x60000000, ldy=64, M=128, N=64, K=64, act=0, layout=0)
    with pytest.raises(ob.OptError) as e:
        ob.opt_linear_plan_create([sk(), big], ob.OPT_BF16)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
    if not torch.cuda.is_available():
        with pytest.raises(ob.OptError) as e:      # valid skinny group: only the device is missing
            ob.opt_linear_plan_create([sk()], ob.OPT_BF16)
        assert e.value.status == ob.OPT_ERR_NO_DEVICE
    # LayerNorm backward: D <= 512, multiples of 8
    lb = lambda **kw: ob.opt_layernorm_bwd_member(**{**dict(x=A, ldx=64, dy=B, lddy=64, gamma=None, dx=Cc, lddx=64, dgamma=None, dbeta=None,
                                                            rows=16, D=64, eps=1e-5), **kw})
    for member, status in [(lb(D=4096, ldx=4096, lddy=4096, lddx=4096), ob.OPT_ERR_UNSUPPORTED), (lb(D=60), ob.OPT_ERR_ALIGNMENT),
                           (lb(dx=A), ob.OPT_ERR_ALIAS)]:
        with pytest.raises(ob.OptError) as e:
            ob.opt_layernorm_bwd_plan_create([member], ob.OPT_BF16)
        assert e.value.status == status, (e.value, status)
    # bias gradient: N % 8 (fp32 activations: % 4), aligned pointers and strides, db must not lie inside dz
    bgm = lambda **kw: ob.opt_bias_grad_member(**{**dict(dz=A, ldz=64, db=B, M=16, N=64, y=None, ldy=0, dz_out=None, lddz_out=0, act=0), **kw})
    for member, io, status in [(bgm(N=60), ob.OPT_BF16, ob.OPT_ERR_ALIGNMENT), (bgm(ldz=68), ob.OPT_BF16, ob.OPT_ERR_ALIGNMENT), (bgm(db=B + 8), ob.OPT_BF16, ob.OPT_ERR_ALIGNMENT),
                               (bgm(db=A + 128), ob.OPT_BF16, ob.OPT_ERR_ALIAS), (bgm(ldz=32), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (bgm(M=0), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG),
                               (bgm(dz=None), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (bgm(N=62), ob.OPT_F32, ob.OPT_ERR_ALIGNMENT), (bgm(act=1), ob.OPT_F32, ob.OPT_ERR_INVALID_ARG),
                               (bgm(dz_out=Cc, lddz_out=64), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (bgm(y=Cc, ldy=60), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (bgm(act=2), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (bgm(y=Cc, ldy=64, act=4), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG),
                               (bgm(y=Cc, ldy=64, dz_out=A + 16, lddz_out=64), ob.OPT_BF16, ob.OPT_ERR_ALIAS)]:
        with pytest.raises(ob.OptError) as e:
            ob.opt_bias_grad_plan_create([member], io)
        assert e.value.status == status, (e.value, status)
    if not torch.cuda.is_available():
        with pytest.raises(ob.OptError) as e:      # valid group: only the device is missing
            ob.opt_bias_grad_plan_create([bgm()], ob.OPT_BF16, ob.OPT_F32)
        assert e.value.status == ob.OPT_ERR_NO_DEVICE
    # pointwise: binary op without a second operand, FP8 on fp32 activations, unknown op
    ch = lambda **kw: ob.opt_chunk(**{**dict(src=A, lds=64, dst=B, ldd=64, rows=4, width=64, op=0, src2=None, lds2=0, p0=0.0, p1=0.0, p2=0.0), **kw})
    for chunk, io, status in [(ch(op=ob.OPT_PW_MUL), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (ch(op=ob.OPT_PW_QUANT_E4M3, p0=1.0), ob.OPT_F32, ob.OPT_ERR_UNSUPPORTED),
                              (ch(op=14), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (ch(op=ob.OPT_PW_RELU_BWD), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (ch(op=ob.OPT_PW_TANH_BWD), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (ch(op=ob.OPT_PW_SIGMOID_BWD), ob.OPT_BF16, ob.OPT_ERR_INVALID_ARG), (ch(op=ob.OPT_PW_SUB, src2=B + 64, lds2=64), ob.OPT_BF16, ob.OPT_ERR_ALIAS)]:
        with pytest.raises(ob.OptError) as e:
            ob.opt_pointwise_plan_create([chunk], io)
        assert e.value.status == status, (e.value, status)
    assert ob.opt_launch_count() == 0


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_02945_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "optimus_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2607_02945_b200" not in txt and "from paper_2607_02945_b200" not in txt, f
            assert "csrc" not in txt and "optimus_b200.h" not in txt, f


def test_no_alloc_entry_point_validates_on_the_host(ob):
    """opt_bias_grad_noalloc: the limit of its static scratch and the argument rules are reported before any CUDA call."""
    L = ob.lib()
    dz, db = ctypes.c_void_p(0x10000000), ctypes.c_void_p(0x20000000)          # never dereferenced: validation only
    call = lambda dz_, ldz, db_, M, N, param=ob.OPT_F32: L.opt_bias_grad_noalloc(dz_, ldz, db_, M, N, param, 0, None)
    n0 = ob.opt_launch_count()
    assert call(dz, 8192, db, 64, ob.OPT_NOALLOC_BIAS_GRAD_MAX_N + 8) == ob.OPT_ERR_UNSUPPORTED
    assert "OPT_NOALLOC_BIAS_GRAD_MAX_N" in ob.opt_last_error()
    assert call(None, 64, db, 64, 64) == ob.OPT_ERR_INVALID_ARG
    assert call(dz, 64, db, 0, 64) == ob.OPT_ERR_INVALID_ARG
    assert call(dz, 32, db, 64, 64) == ob.OPT_ERR_INVALID_ARG                   # ldz < N
    assert call(dz, 64, db, 64, 64, 7) == ob.OPT_ERR_INVALID_ARG                # bad dtype
    assert call(dz, 64, db, 64, 60) == ob.OPT_ERR_ALIGNMENT                     # N % 8
    assert call(dz, 68, db, 64, 64) == ob.OPT_ERR_ALIGNMENT                     # ldz % 8
    assert call(ctypes.c_void_p(0x10000008), 64, db, 64, 64) == ob.OPT_ERR_ALIGNMENT
    assert call(dz, 64, ctypes.c_void_p(0x10000000 + 64 * 8), 64, 64) == ob.OPT_ERR_ALIAS   # db inside dz
    assert ob.opt_launch_count() == n0
