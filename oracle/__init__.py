"""CPU ORACLE -- test infrastructure, not the product.

ctypes access to oracle/optimus_oracle.cpp (plain C++17, fp64, the unfused graph
one op at a time).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package; the product
package paper_2607_02945_b200 never does, and this package never imports it.

`build()` compiles liboptimus_oracle.so next to the source with g++ (OpenMP for
the timed run; OpenMP only splits independent rows, never a floating-point sum).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "optimus_oracle.cpp")
_LIB = os.path.join(_HERE, "liboptimus_oracle.so")
_lib = None

F32, BF16 = 0, 1
_NP = {F32: np.float32, BF16: np.uint16}
_ESZ = {F32: 4, BF16: 2}


def build(force=False):
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-fno-fast-math",
           "-o", _LIB, _SRC]
    subprocess.check_call(cmd)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        c = ctypes
        vp, i64, i32, dbl = c.c_void_p, c.c_int64, c.c_int32, c.c_double
        L.oracle_set_threads.argtypes = [c.c_int]
        L.oracle_get_max_threads.restype = c.c_int
        L.oracle_round_to_storage.argtypes = [vp, i64, c.c_int, vp]
        L.oracle_widen.argtypes = [vp, i64, c.c_int, vp]
        L.oracle_linear.argtypes = [vp, i64, vp, i64, vp, i32, i32, i32, c.c_int, vp]
        L.oracle_linear_f64x.argtypes = [vp, vp, i64, vp, i32, i32, i32, c.c_int, vp]
        L.oracle_colsum.argtypes = [vp, i64, i32, i32, c.c_int, vp]
        L.oracle_linear_mulreduce.argtypes = [vp, i64, vp, i64, vp, i32, i32, i32, c.c_int, vp]
        L.oracle_activation.argtypes = [vp, i64, c.c_int]
        L.oracle_pointwise.argtypes = [vp, i64, i32, i32, c.c_int, c.c_int, vp]
        L.oracle_pointwise_ext.argtypes = [vp, i64, vp, i64, i32, i32, c.c_int, dbl, dbl, dbl, c.c_int, vp]
        L.oracle_layernorm.argtypes = [vp, i64, vp, vp, i32, i32, dbl, c.c_int, c.c_int, vp, vp]
        L.oracle_quant_e4m3.argtypes = [vp, i64, i32, i32, dbl, c.c_int, vp]
        L.oracle_dequant_e4m3.argtypes = [vp, i64, i32, i32, dbl, vp]
        L.oracle_layernorm_backward.argtypes = [vp, i64, vp, i64, vp, i32, i32, dbl, c.c_int, c.c_int, vp, vp, vp]
        L.oracle_split.argtypes = [vp, i64, i32, i32, i32, vp, i32, vp]
        L.oracle_split.restype = c.c_int
        L.oracle_cat.argtypes = [vp, vp, i32, i32, i32, vp, i64]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _chk(a, dt, ndim=None):
    assert a.dtype == _NP[dt], (a.dtype, dt)
    assert a.strides[-1] == a.itemsize, "unit inner stride required"
    if ndim is not None:
        assert a.ndim == ndim
    return a


def _ld(a):
    return a.strides[0] // a.itemsize if a.ndim == 2 else a.shape[-1]


def set_threads(n):
    lib().oracle_set_threads(int(n))


def max_threads():
    return int(lib().oracle_get_max_threads())


# ------------------------------------------------------------------- ops ----
def round_to_storage(z, dt):
    """fp64 array -> storage dtype (fp32, or bf16 bits as uint16), direct RNE."""
    z = np.ascontiguousarray(z, dtype=np.float64)
    out = np.empty(z.shape, dtype=_NP[dt])
    lib().oracle_round_to_storage(_ptr(z), z.size, dt, _ptr(out))
    return out


def widen(a, dt):
    a = np.ascontiguousarray(a)
    assert a.dtype == _NP[dt]
    out = np.empty(a.shape, dtype=np.float64)
    lib().oracle_widen(_ptr(a), a.size, dt, _ptr(out))
    return out


def linear(x, w, b, dt, mulreduce=False):
    """Z = X W^T + b in fp64; x:[M,K], w:[N,K], b:[N] or None, storage dtype dt."""
    _chk(x, dt, 2), _chk(w, dt, 2)
    M, K = x.shape
    N, K2 = w.shape
    assert K == K2
    if b is not None:
        b = np.ascontiguousarray(_chk(b, dt, 1))
        assert b.shape == (N,)
    z = np.empty((M, N), dtype=np.float64)
    fn = lib().oracle_linear_mulreduce if mulreduce else lib().oracle_linear
    fn(_ptr(x), _ld(x), _ptr(w), _ld(w), _ptr(b), M, N, K, dt, _ptr(z))
    return z


def linear_f64x(x64, w, b, dt):
    """Z = X W^T + b in fp64 for an activation matrix that is already fp64 (the unrounded LayerNorm output inside a
    vertically fused chain, reading Q25); w:[N,K], b:[N] or None in storage dtype dt.  Same summation order as linear."""
    x64 = np.ascontiguousarray(x64, dtype=np.float64)
    _chk(w, dt, 2)
    M, K = x64.shape
    N, K2 = w.shape
    assert K == K2
    if b is not None:
        b = np.ascontiguousarray(_chk(b, dt, 1))
        assert b.shape == (N,)
    z = np.empty((M, N), dtype=np.float64)
    lib().oracle_linear_f64x(_ptr(x64), _ptr(w), _ld(w), _ptr(b), M, N, K, dt, _ptr(z))
    return z


def colsum(dz, dt):
    """db[n] = sum over rows of dz[m, n], rows added in index order, fp64 (the bias gradient of a Linear)."""
    _chk(dz, dt, 2)
    M, N = dz.shape
    db = np.empty((N,), dtype=np.float64)
    lib().oracle_colsum(_ptr(dz), _ld(dz), M, N, dt, _ptr(db))
    return db


def activation(z, act):
    """elementwise on fp64, returns a new array; act: 0 none, 1 relu, 2 tanh, 3 sigmoid."""
    z = np.array(z, dtype=np.float64, order="C", copy=True)
    lib().oracle_activation(_ptr(z), z.size, int(act))
    return z


def pointwise(src, op, dt):
    """f(src) in fp64 for a 2-D storage tensor with unit inner stride."""
    _chk(src, dt, 2)
    rows, width = src.shape
    out = np.empty((rows, width), dtype=np.float64)
    lib().oracle_pointwise(_ptr(src), _ld(src), rows, width, int(op), dt, _ptr(out))
    return out


PW_CLAMP, PW_NAN_TO_NUM, PW_SUB, PW_DIV, PW_MUL = 4, 5, 6, 7, 8
PW_RELU_BWD = 11
PW_TANH_BWD = 12
PW_SIGMOID_BWD = 13


def pointwise_ext(a, b, op, params, dt):
    """Table-1 pointwise patterns beyond relu/tanh/sigmoid, fp64, torch semantics:
    op 4 clamp(a, lo=params[0], hi=params[1]); op 5 nan_to_num(a, nan=params[0], posinf=params[1],
    neginf=params[2]); op 6/7/8 a - b, a / b, a * b; op 11 ReLU backward: a where b > 0 (or b is NaN), else 0
    (a = incoming gradient, b = the ReLU's output or input); op 12 tanh backward a (1 - b^2), op 13 sigmoid backward
    a (1 - b) b (b = the stored forward OUTPUT; torch tanh_backward / sigmoid_backward).  Parameters are the fp32 values the descriptor carries."""
    _chk(a, dt, 2)
    rows, width = a.shape
    if b is not None:
        _chk(b, dt, 2)
        assert b.shape == a.shape
    p = [float(np.float32(v)) for v in (list(params) + [0.0, 0.0, 0.0])[:3]]
    out = np.empty((rows, width), dtype=np.float64)
    lib().oracle_pointwise_ext(_ptr(a), _ld(a), _ptr(b), 0 if b is None else _ld(b), rows, width, int(op),
                               p[0], p[1], p[2], dt, _ptr(out))
    return out


def quant_e4m3(src, scale, dt):
    """FP8 E4M3 codes (uint8) of src * scale, round-to-nearest-even, saturating at +-448."""
    _chk(src, dt, 2)
    rows, width = src.shape
    out = np.empty((rows, width), dtype=np.uint8)
    lib().oracle_quant_e4m3(_ptr(src), _ld(src), rows, width, float(np.float32(scale)), dt, _ptr(out))
    return out


def dequant_e4m3(codes, scale):
    """fp64 values of FP8 E4M3 codes times scale."""
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    rows, width = codes.shape
    out = np.empty((rows, width), dtype=np.float64)
    lib().oracle_dequant_e4m3(_ptr(codes), width, rows, width, float(np.float32(scale)), _ptr(out))
    return out


def layernorm(x, gamma, beta, eps, dt, param_dt=None, return_xhat=False):
    """torch layer_norm over the last dim, fp64.  eps is the fp32 value the
    descriptor carries, widened (np.float32(eps))."""
    param_dt = dt if param_dt is None else param_dt
    _chk(x, dt, 2)
    rows, D = x.shape
    if gamma is not None:
        gamma = np.ascontiguousarray(_chk(gamma, param_dt, 1))
    if beta is not None:
        beta = np.ascontiguousarray(_chk(beta, param_dt, 1))
    y = np.empty((rows, D), dtype=np.float64)
    xh = np.empty((rows, D), dtype=np.float64) if return_xhat else None
    lib().oracle_layernorm(_ptr(x), _ld(x), _ptr(gamma), _ptr(beta), rows, D,
                           float(np.float32(eps)), dt, param_dt, _ptr(y), _ptr(xh))
    return (y, xh) if return_xhat else y


def layernorm_backward(x, dy, gamma, eps, dt, param_dt=None):
    """torch layer_norm backward over the last dim, fp64 -> (dx [rows,D], dgamma [D], dbeta [D])."""
    param_dt = dt if param_dt is None else param_dt
    _chk(x, dt, 2)
    _chk(dy, dt, 2)
    assert x.shape == dy.shape
    rows, D = x.shape
    if gamma is not None:
        gamma = np.ascontiguousarray(_chk(gamma, param_dt, 1))
    dx = np.empty((rows, D), dtype=np.float64)
    dg = np.empty((D,), dtype=np.float64)
    db = np.empty((D,), dtype=np.float64)
    lib().oracle_layernorm_backward(_ptr(x), _ld(x), _ptr(dy), _ld(dy), _ptr(gamma), rows, D, float(np.float32(eps)),
                                    dt, param_dt, _ptr(dx), _ptr(dg), _ptr(db))
    return dx, dg, db


def split(x, sizes):
    """torch.split(x, sizes, dim=1) on raw storage elements; returns dense pieces."""
    assert x.ndim == 2 and x.strides[1] == x.itemsize
    rows, width = x.shape
    sizes = [int(s) for s in sizes]
    pieces = [np.empty((rows, s), dtype=x.dtype) for s in sizes]
    arr = (ctypes.c_void_p * len(sizes))(*[p.ctypes.data for p in pieces])
    sz = (ctypes.c_int32 * len(sizes))(*sizes)
    rc = lib().oracle_split(_ptr(x), _ld(x), rows, width, x.itemsize, sz, len(sizes), arr)
    if rc != 0:
        raise ValueError("split sizes do not sum to the width")
    return pieces


def cat(pieces):
    """torch.cat(pieces, dim=1) on raw storage elements."""
    pieces = [np.ascontiguousarray(p) for p in pieces]
    rows = pieces[0].shape[0]
    assert all(p.ndim == 2 and p.shape[0] == rows and p.dtype == pieces[0].dtype for p in pieces)
    sizes = [p.shape[1] for p in pieces]
    out = np.empty((rows, sum(sizes)), dtype=pieces[0].dtype)
    arr = (ctypes.c_void_p * len(sizes))(*[p.ctypes.data for p in pieces])
    sz = (ctypes.c_int32 * len(sizes))(*sizes)
    lib().oracle_cat(arr, sz, len(sizes), rows, out.itemsize, _ptr(out), out.shape[1])
    return out
