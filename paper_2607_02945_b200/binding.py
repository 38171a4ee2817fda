"""ctypes binding: same names as the C ABI, argument marshalling only."""
import ctypes as C
import os

from . import build as _build

OPT_F32, OPT_BF16 = 0, 1
OPT_ACT_NONE, OPT_ACT_RELU, OPT_ACT_TANH, OPT_ACT_SIGMOID = 0, 1, 2, 3
OPT_PW_COPY, OPT_PW_RELU, OPT_PW_TANH, OPT_PW_SIGMOID = 0, 1, 2, 3
OPT_PW_CLAMP, OPT_PW_NAN_TO_NUM, OPT_PW_SUB, OPT_PW_DIV, OPT_PW_MUL = 4, 5, 6, 7, 8
OPT_PW_QUANT_E4M3, OPT_PW_DEQUANT_E4M3 = 9, 10
OPT_PW_RELU_BWD = 11
OPT_PW_TANH_BWD, OPT_PW_SIGMOID_BWD = 12, 13
OPT_LAYOUT_X_TRANSPOSED, OPT_LAYOUT_W_TRANSPOSED = 1, 2
(OPT_OK, OPT_ERR_INVALID_ARG, OPT_ERR_UNSUPPORTED, OPT_ERR_ALIGNMENT, OPT_ERR_ALIAS, OPT_ERR_CUDA,
 OPT_ERR_NO_DEVICE) = range(7)
_STATUS_NAMES = ["OPT_OK", "OPT_ERR_INVALID_ARG", "OPT_ERR_UNSUPPORTED", "OPT_ERR_ALIGNMENT", "OPT_ERR_ALIAS",
                 "OPT_ERR_CUDA", "OPT_ERR_NO_DEVICE"]


class opt_linear_member(C.Structure):
    _fields_ = [("x", C.c_void_p), ("ldx", C.c_int64), ("w", C.c_void_p), ("ldw", C.c_int64),
                ("bias", C.c_void_p), ("y", C.c_void_p), ("ldy", C.c_int64),
                ("M", C.c_int32), ("N", C.c_int32), ("K", C.c_int32), ("act", C.c_int32), ("layout", C.c_int32),
                ("y8", C.c_void_p), ("ldy8", C.c_int64), ("scale8", C.c_float)]


class opt_linear_options(C.Structure):
    _fields_ = [("cta_pair", C.c_int32), ("no_skinny", C.c_int32), ("no_lhs_order", C.c_int32), ("reserved", C.c_int32 * 5)]


class opt_linear2_member(C.Structure):
    _fields_ = [("x", C.c_void_p), ("ldx", C.c_int64), ("w1", C.c_void_p), ("ldw1", C.c_int64), ("b1", C.c_void_p),
                ("w2", C.c_void_p), ("ldw2", C.c_int64), ("b2", C.c_void_p), ("y", C.c_void_p), ("ldy", C.c_int64),
                ("M", C.c_int32), ("K", C.c_int32), ("H", C.c_int32), ("N", C.c_int32),
                ("act1", C.c_int32), ("act2", C.c_int32)]


class opt_ln_linear2_member(C.Structure):
    _fields_ = [("chain", opt_linear2_member), ("gamma", C.c_void_p), ("beta", C.c_void_p), ("eps", C.c_float),
                ("reserved", C.c_int32)]


class opt_layernorm_member(C.Structure):
    _fields_ = [("x", C.c_void_p), ("ldx", C.c_int64), ("y", C.c_void_p), ("ldy", C.c_int64),
                ("gamma", C.c_void_p), ("beta", C.c_void_p),
                ("rows", C.c_int32), ("D", C.c_int32), ("eps", C.c_float),
                ("y8", C.c_void_p), ("ldy8", C.c_int64), ("scale8", C.c_float)]


class opt_layernorm_bwd_member(C.Structure):
    _fields_ = [("x", C.c_void_p), ("ldx", C.c_int64), ("dy", C.c_void_p), ("lddy", C.c_int64), ("gamma", C.c_void_p),
                ("dx", C.c_void_p), ("lddx", C.c_int64), ("dgamma", C.c_void_p), ("dbeta", C.c_void_p),
                ("rows", C.c_int32), ("D", C.c_int32), ("eps", C.c_float)]


class opt_bias_grad_member(C.Structure):
    _fields_ = [("dz", C.c_void_p), ("ldz", C.c_int64), ("db", C.c_void_p), ("M", C.c_int32), ("N", C.c_int32),
                ("y", C.c_void_p), ("ldy", C.c_int64), ("dz_out", C.c_void_p), ("lddz_out", C.c_int64), ("act", C.c_int32)]


class opt_chunk(C.Structure):
    _fields_ = [("src", C.c_void_p), ("lds", C.c_int64), ("dst", C.c_void_p), ("ldd", C.c_int64),
                ("rows", C.c_int32), ("width", C.c_int32), ("op", C.c_int32),
                ("src2", C.c_void_p), ("lds2", C.c_int64), ("p0", C.c_float), ("p1", C.c_float), ("p2", C.c_float)]


class opt_host_copy(C.Structure):
    _fields_ = [("host", C.c_void_p), ("device", C.c_void_p), ("bytes", C.c_size_t), ("to_device", C.c_int32)]


class OptError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("%s: %s" % (_STATUS_NAMES[status] if 0 <= status < 7 else status, message))
        self.status = status
        self.message = message


_lib = None


def lib_path():
    return _lib_path or _build.LIB


_lib_path = None


def use_trace_library():
    """Measurement aid (bench.py --side gemm_trace): make this process load the pipeline-trace build of the library
    (liboptimus_b200_trace.so: same kernels + wait-cycle counters in the grouped GEMM).  Call before the first use."""
    global _lib_path
    assert _lib is None, "the library is already loaded"
    _lib_path = _build.build(trace=True)


def lib():
    """Load (building if needed) liboptimus_b200.so.  Raises if it cannot be had: no fallback."""
    global _lib
    if _lib is None:
        if _lib_path is None and (not os.path.exists(_build.LIB) or not _build.up_to_date()):
            try:
                _build.build()
            except Exception as e:  # noqa: BLE001
                if not os.path.exists(_build.LIB):
                    raise ImportError("liboptimus_b200.so is missing and could not be built with nvcc: %r" % (e,))
        L = C.CDLL(_lib_path or _build.LIB)
        pp = C.POINTER(C.c_void_p)
        L.opt_linear_plan_create.argtypes = [C.POINTER(opt_linear_member), C.c_int32, C.c_int, C.c_int, pp]
        L.opt_linear_plan_create_ex.argtypes = [C.POINTER(opt_linear_member), C.c_int32, C.c_int, C.c_int,
                                                C.POINTER(opt_linear_options), pp]
        L.opt_linear2_plan_create.argtypes = [C.POINTER(opt_linear2_member), C.c_int32, C.c_int, C.c_int, pp]
        L.opt_ln_linear2_plan_create.argtypes = [C.POINTER(opt_ln_linear2_member), C.c_int32, C.c_int, C.c_int, pp]
        L.opt_layernorm_plan_create.argtypes = [C.POINTER(opt_layernorm_member), C.c_int32, C.c_int, C.c_int,
                                                C.c_int, pp]
        L.opt_layernorm_bwd_plan_create.argtypes = [C.POINTER(opt_layernorm_bwd_member), C.c_int32, C.c_int, C.c_int,
                                                    C.c_int, pp]
        L.opt_bias_grad_plan_create.argtypes = [C.POINTER(opt_bias_grad_member), C.c_int32, C.c_int, C.c_int, C.c_int, pp]
        L.opt_pointwise_plan_create.argtypes = [C.POINTER(opt_chunk), C.c_int32, C.c_int, C.c_int, pp]
        L.opt_bias_grad_noalloc.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_int32, C.c_int32, C.c_int, C.c_int, C.c_void_p]
        L.opt_bias_grad_noalloc.restype = C.c_int
        L.opt_plan_launch.argtypes = [C.c_void_p, C.c_void_p]
        L.opt_plan_launch_host.argtypes = [C.c_void_p, C.POINTER(opt_host_copy), C.c_int32, C.c_void_p]
        L.opt_plan_info.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int32),
                                    C.POINTER(C.c_int32)]
        L.opt_plan_destroy.argtypes = [C.c_void_p]
        L.opt_last_error.restype = C.c_char_p
        L.opt_launch_count.restype = C.c_uint64
        L.opt_version.restype = C.c_char_p
        for f in (L.opt_linear_plan_create, L.opt_linear_plan_create_ex, L.opt_linear2_plan_create, L.opt_ln_linear2_plan_create, L.opt_layernorm_plan_create, L.opt_layernorm_bwd_plan_create, L.opt_bias_grad_plan_create, L.opt_pointwise_plan_create,
                  L.opt_plan_launch, L.opt_plan_launch_host, L.opt_plan_info, L.opt_plan_destroy):
            f.restype = C.c_int
        _lib = L
    return _lib


def opt_last_error():
    return lib().opt_last_error().decode()


def opt_launch_count():
    return int(lib().opt_launch_count())


def opt_version():
    return lib().opt_version().decode()


def _check(st):
    if st != OPT_OK:
        raise OptError(st, opt_last_error())


def _array(ctype, items):
    items = list(items)
    return (ctype * max(len(items), 1))(*items), len(items)


class Plan:
    """Opaque opt_plan handle.  launch() = opt_plan_launch: exactly one kernel launch."""

    def __init__(self, handle):
        self._h = handle

    def launch(self, stream=None):
        opt_plan_launch(self, stream)

    def launch_host(self, copies, stream=None):
        opt_plan_launch_host(self, copies, stream)

    def info(self):
        return opt_plan_info(self)

    def destroy(self):
        opt_plan_destroy(self)

    def __del__(self):
        try:
            self.destroy()
        except Exception:  # noqa: BLE001
            pass


def _create(fn, ctype, members, *dtype_and_device):
    arr, n = _array(ctype, members)
    h = C.c_void_p()
    _check(fn(arr, n, *dtype_and_device, C.byref(h)))
    return Plan(h)


def opt_linear_plan_create(members, io, device=0):
    return _create(lib().opt_linear_plan_create, opt_linear_member, members, io, device)


def opt_linear_plan_create_ex(members, io, device=0, options=None):
    """options: an opt_linear_options (or None for the defaults)."""
    arr, n = _array(opt_linear_member, members)
    h = C.c_void_p()
    _check(lib().opt_linear_plan_create_ex(arr, n, io, device, None if options is None else C.byref(options), C.byref(h)))
    return Plan(h)


def opt_linear2_plan_create(members, io, device=0):
    return _create(lib().opt_linear2_plan_create, opt_linear2_member, members, io, device)


def opt_ln_linear2_plan_create(members, io, device=0):
    return _create(lib().opt_ln_linear2_plan_create, opt_ln_linear2_member, members, io, device)


def opt_layernorm_plan_create(members, io, param=None, device=0):
    return _create(lib().opt_layernorm_plan_create, opt_layernorm_member, members, io,
                   io if param is None else param, device)


def opt_layernorm_bwd_plan_create(members, io, param=None, device=0):
    return _create(lib().opt_layernorm_bwd_plan_create, opt_layernorm_bwd_member, members, io,
                   io if param is None else param, device)


def opt_bias_grad_plan_create(members, io, param=None, device=0):
    return _create(lib().opt_bias_grad_plan_create, opt_bias_grad_member, members, io,
                   io if param is None else param, device)


OPT_NOALLOC_BIAS_GRAD_MAX_N = 4096


def opt_bias_grad_noalloc(dz, db, param=OPT_F32, device=0, stream=None):
    """db = column sums of the bf16 tensor dz [M, N] without any allocation (scratch in a static device array of the
    library; N <= OPT_NOALLOC_BIAS_GRAD_MAX_N; calls that overlap on the GPU race on that scratch)."""
    M, N = dz.shape
    assert tuple(db.shape) == (N,)
    _check(lib().opt_bias_grad_noalloc(dz.data_ptr(), _ld(dz), db.data_ptr(), M, N, int(param), device, _stream_ptr(stream)))


def opt_pointwise_plan_create(chunks, io, device=0):
    return _create(lib().opt_pointwise_plan_create, opt_chunk, chunks, io, device)


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    return C.c_void_p(int(stream))


def opt_plan_launch(plan, stream=None):
    _check(lib().opt_plan_launch(plan._h, _stream_ptr(stream)))


def opt_plan_launch_host(plan, copies, stream=None):
    arr, n = _array(opt_host_copy, copies)
    _check(lib().opt_plan_launch_host(plan._h, arr, n, _stream_ptr(stream)))


def opt_plan_info(plan):
    fl, by, la, ti = C.c_int64(), C.c_int64(), C.c_int32(), C.c_int32()
    _check(lib().opt_plan_info(plan._h, C.byref(fl), C.byref(by), C.byref(la), C.byref(ti)))
    return dict(flops=fl.value, bytes=by.value, launches=la.value, tiles=ti.value)


def opt_plan_destroy(plan):
    if plan._h is not None and plan._h.value:
        lib().opt_plan_destroy(plan._h)
    plan._h = None


# ---- descriptor helpers: read data_ptr / strides off torch tensors (marshalling only) ----
def _ld(t):
    assert t.dim() == 2 and t.stride(1) == 1, "2-D tensor with unit column stride required"
    return t.stride(0)


def linear_member(x, w, bias, y, act=OPT_ACT_NONE, layout=0, y8=None, scale8=0.0):
    """layout: OPT_LAYOUT_* flags; a transposed operand is passed as it is stored ([K,M] / [K,N]).
    y8: optional uint8 [M,N] tensor for the FP8 (E4M3) copy of the output (y may then be None)."""
    M, N = (y if y is not None else y8).shape
    K = x.shape[0] if layout & OPT_LAYOUT_X_TRANSPOSED else x.shape[1]
    assert tuple(x.shape) == ((K, M) if layout & OPT_LAYOUT_X_TRANSPOSED else (M, K))
    assert tuple(w.shape) == ((K, N) if layout & OPT_LAYOUT_W_TRANSPOSED else (N, K))
    assert y8 is None or (tuple(y8.shape) == (M, N) and y8.element_size() == 1)
    return opt_linear_member(x.data_ptr(), _ld(x), w.data_ptr(), _ld(w),
                             None if bias is None else bias.data_ptr(), None if y is None else y.data_ptr(),
                             0 if y is None else _ld(y), M, N, K, int(act), int(layout),
                             None if y8 is None else y8.data_ptr(), 0 if y8 is None else _ld(y8), float(scale8))


def linear2_member(x, w1, b1, w2, b2, y, act1=OPT_ACT_RELU, act2=OPT_ACT_NONE):
    M, K = x.shape
    H, N = w1.shape[0], w2.shape[0]
    assert w1.shape[1] == K and w2.shape[1] == H and tuple(y.shape) == (M, N)
    return opt_linear2_member(x.data_ptr(), _ld(x), w1.data_ptr(), _ld(w1), None if b1 is None else b1.data_ptr(),
                              w2.data_ptr(), _ld(w2), None if b2 is None else b2.data_ptr(), y.data_ptr(), _ld(y),
                              M, K, H, N, int(act1), int(act2))


def ln_linear2_member(x, gamma, beta, eps, w1, b1, w2, b2, y, act1=OPT_ACT_RELU, act2=OPT_ACT_NONE):
    assert gamma is None or tuple(gamma.shape) == (x.shape[1],)
    assert beta is None or tuple(beta.shape) == (x.shape[1],)
    return opt_ln_linear2_member(linear2_member(x, w1, b1, w2, b2, y, act1, act2), None if gamma is None else gamma.data_ptr(),
                                 None if beta is None else beta.data_ptr(), float(eps), 0)


def layernorm_member(x, y, gamma, beta, eps, y8=None, scale8=0.0):
    """y8: optional uint8 [rows,D] tensor for the FP8 (E4M3) copy of the output (y may then be None)."""
    rows, D = x.shape
    assert y is None or tuple(y.shape) == (rows, D)
    assert y8 is None or (tuple(y8.shape) == (rows, D) and y8.element_size() == 1)
    return opt_layernorm_member(x.data_ptr(), _ld(x), None if y is None else y.data_ptr(), 0 if y is None else _ld(y),
                                None if gamma is None else gamma.data_ptr(),
                                None if beta is None else beta.data_ptr(), rows, D, float(eps),
                                None if y8 is None else y8.data_ptr(), 0 if y8 is None else _ld(y8), float(scale8))


def layernorm_bwd_member(x, dy, gamma, dx, dgamma, dbeta, eps):
    rows, D = x.shape
    assert tuple(dy.shape) == (rows, D) and tuple(dx.shape) == (rows, D)
    ptr = lambda t: None if t is None else t.data_ptr()
    return opt_layernorm_bwd_member(x.data_ptr(), _ld(x), dy.data_ptr(), _ld(dy), ptr(gamma), dx.data_ptr(), _ld(dx),
                                    ptr(dgamma), ptr(dbeta), rows, D, float(eps))


def bias_grad_member(dz, db, y=None, dz_out=None, act=0):
    """db = column sums of dz; with y (stored ReLU output): of the masked gradient (act 2 / 3: of dz times the tanh / sigmoid derivative), which goes to dz_out if given."""
    M, N = dz.shape
    assert tuple(db.shape) == (N,)
    assert y is None or tuple(y.shape) == (M, N)
    assert dz_out is None or (y is not None and tuple(dz_out.shape) == (M, N))
    return opt_bias_grad_member(dz.data_ptr(), _ld(dz), db.data_ptr(), M, N,
                                None if y is None else y.data_ptr(), 0 if y is None else _ld(y),
                                None if dz_out is None else dz_out.data_ptr(), 0 if dz_out is None else _ld(dz_out), int(act))


def chunk(src, dst, op=OPT_PW_COPY, src2=None, params=()):
    rows, width = src.shape
    assert tuple(dst.shape) == (rows, width)
    p = (list(params) + [0.0, 0.0, 0.0])[:3]
    if src2 is not None:
        assert tuple(src2.shape) == (rows, width)
    return opt_chunk(src.data_ptr(), _ld(src), dst.data_ptr(), _ld(dst), rows, width, int(op),
                     None if src2 is None else src2.data_ptr(), 0 if src2 is None else _ld(src2),
                     float(p[0]), float(p[1]), float(p[2]))


def split_cat_chunks(x, out, widths, ops, perm):
    """Chunk list of split(x, widths, dim=1) -> ops[j] on chunk j -> cat in order perm
    (perm[j] = source chunk at output position j)."""
    starts = [0]
    for w in widths:
        starts.append(starts[-1] + w)
    chunks, d = [], 0
    for p in perm:
        w = widths[p]
        chunks.append(chunk(x[:, starts[p]:starts[p] + w], out[:, d:d + w], ops[p]))
        d += w
    return chunks
