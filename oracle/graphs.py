"""CPU ORACLE (test infrastructure) -- the UNFUSED graphs of BASELINE.json's
configs, run one op at a time through oracle/optimus_oracle.cpp.

Each function mirrors the graph a PyTorch user writes before Optimus rewrites
it (PAPER.md:148 group fusion; :166 chained transformations; :403-416 Listing
2): N independent ops, then torch.cat.  Rounding to the storage dtype happens
once per *group* output (linear+bias+activation is one group: reading Q2), and
between the groups of configs[4] (reading Q3).
"""
import numpy as np

from . import (BF16, F32, activation, cat, colsum, layernorm, linear, linear_f64x, pointwise,  # noqa: F401
               quant_e4m3, round_to_storage, split)


def linear_member(m, dt):
    """fp64 result of one member: act(x W^T + b)."""
    z = linear(m["x"], m["w"], m.get("b"), dt)
    return activation(z, m["act"])


def linear_group(members, dt):
    """-> (list of fp64 outputs, list of storage-dtype outputs)."""
    z64 = [linear_member(m, dt) for m in members]
    return z64, [round_to_storage(z, dt) for z in z64]


def linear_group_concat(members, dt):
    z64, ys = linear_group(members, dt)
    return z64, cat(ys)


def saved_activation_fp8(y_storage, scale, dt=BF16):
    """activation_quantization_aten_pass as the unfused graph runs it: the op's output
    is first materialised in the storage dtype, THEN quantised -- code = e4m3_rne_satfinite(y_storage * scale).
    A fused epilogue that also emits the FP8 copy must produce exactly these codes (reading Q29).  No new arithmetic:
    `quant_e4m3` applied to the rounded output."""
    return quant_e4m3(y_storage, scale, dt)


def linear_member_fp8(m, scale, dt=BF16):
    """Linear + bias + activation, rounded to storage, and the FP8 copy of that rounded tensor.  -> (y64, y, codes)."""
    y64 = linear_member(m, dt)
    y = round_to_storage(y64, dt)
    return y64, y, saved_activation_fp8(y, scale, dt)


def layernorm_fp8(m, scale, dt=BF16):
    """LayerNorm, rounded to storage, and the FP8 copy of that rounded tensor.  -> (y64, y, codes)."""
    y64 = layernorm(m["x"], m.get("gamma"), m.get("beta"), m["eps"], dt)
    y = round_to_storage(y64, dt)
    return y64, y, saved_activation_fp8(y, scale, dt)


def layernorm_group(members, dt):
    y64 = [layernorm(m["x"], m.get("gamma"), m.get("beta"), m["eps"], dt) for m in members]
    return y64, [round_to_storage(y, dt) for y in y64]


def split_pointwise_cat(x, widths, ops, perm, dt):
    """split(x, widths, dim=1) -> f_j on chunk j -> cat([f_perm[0], f_perm[1], ...], dim=1).
    perm[j] = source chunk placed at output position j (reading Q14).
    Returns (fp64 [rows,width] in output order, storage-dtype output)."""
    pieces = split(x, widths)
    f64 = [pointwise(p, op, dt) for p, op in zip(pieces, ops)]
    fst = [round_to_storage(f, dt) for f in f64]
    out = cat([fst[p] for p in perm])
    out64 = np.concatenate([f64[p] for p in perm], axis=1)
    return out64, out


def split_copy_cat(x, widths, perm):
    """movement only: split -> cat in permuted order, raw bits."""
    pieces = split(x, widths)
    return cat([pieces[p] for p in perm])


def recsys_tower(t, dt=BF16):
    """LayerNorm -> Linear+ReLU -> Linear for one tower, intermediates
    materialised in the storage dtype between groups (Q3).
    Returns dict of storage-dtype stage outputs and fp64 stage outputs, where
    stage g's fp64 output is computed from stage g-1's *rounded* output."""
    ln64 = layernorm(t["x"], t["gamma"], t["beta"], t["eps"], dt)
    ln = round_to_storage(ln64, dt)
    h64 = activation(linear(ln, t["w1"], t["b1"], dt), 1)
    h = round_to_storage(h64, dt)
    o64 = linear(h, t["w2"], t["b2"], dt)
    o = round_to_storage(o64, dt)
    return dict(ln=ln, h=h, out=o, ln64=ln64, h64=h64, out64=o64)


def linear2(m, dt=BF16):
    """Two chained Linear layers of one member, the unfused graph op by op ("chained
    transformations", Fig. 5):
        h = act1(x W1^T + b1)  -> rounded to the storage dtype (the intermediate tensor the unfused graph
                                  materialises, reading Q3)
        y = act2(h W2^T + b2)  -> rounded to the storage dtype
    Returns dict(h64, h, y64, y); y64 is computed from the ROUNDED h."""
    h64 = activation(linear(m["x"], m["w1"], m.get("b1"), dt), m["act1"])
    h = round_to_storage(h64, dt)
    y64 = activation(linear(h, m["w2"], m.get("b2"), dt), m["act2"])
    return dict(h64=h64, h=h, y64=y64, y=round_to_storage(y64, dt))


def ln_linear2(m, dt=BF16):
    """LayerNorm -> Linear + act1 -> Linear + act2 of one tower as ONE vertically fused op ("chained
    transformations", Fig. 5, the LayerNorm folded in).  Reading Q25: the
    fused op never materialises the normalised tensor, so it is NOT rounded here; the hidden tensor is still
    rounded to the storage dtype (as in `linear2`, reading Q3):
        xn = layer_norm(x; gamma, beta, eps)          fp64, unrounded
        h  = act1(xn W1^T + b1)  -> rounded            (first layer: oracle_linear_f64x, the plain index-order loop
                                                        of `linear` on the unrounded xn)
        y  = act2(h W2^T + b2)   -> rounded
    Returns dict(xn64, h64, h, y64, y)."""
    xn64 = layernorm(m["x"], m.get("gamma"), m.get("beta"), m["eps"], dt)
    h64 = activation(linear_f64x(xn64, m["w1"], m.get("b1"), dt), m["act1"])
    h = round_to_storage(h64, dt)
    y64 = activation(linear(h, m["w2"], m.get("b2"), dt), m["act2"])
    return dict(xn64=xn64, h64=h64, h=h, y64=y64, y=round_to_storage(y64, dt))


def _transposed(a):
    return np.ascontiguousarray(a.T)


def linear_dgrad(dy, w, dt=BF16):
    """Backward of y = x W^T w.r.t. the input: dX[M,K] = dY[M,N] W[N,K] (sum over n in index order), fp64.
    It is `linear` applied to the transposed weight: dX = dY (W^T)^T (PAPER.md:292 batch_linear_post_grad,
    PAPER.md:437 training)."""
    return linear(dy, _transposed(w), None, dt)


def linear_wgrad(dy, x, dt=BF16):
    """Backward w.r.t. the weight: dW[N,K] = dY[M,N]^T X[M,K] (sum over m in index order), fp64."""
    return linear(_transposed(dy), _transposed(x), None, dt)


def linear_bias_grad(dz, dt=BF16):
    """Backward of y = x W^T + b w.r.t. the bias: db[n] = sum_m dZ[m, n], rows added in index order, fp64
    (PAPER.md:292 batch_linear_post_grad; PAPER.md:437 training)."""
    return colsum(dz, dt)


def linear_relu_backward(m, dy, dt=BF16):
    """The whole backward of one member y = relu(x W^T + b), one op at a time, the mask taken from the STORED forward
    output y (reading Q26): dz = dy where y > 0 else 0 (storage dtype: a select, exact); db = column sums of dz;
    dX = dz W; dW = dz^T x.  -> dict(dz (storage), db64, dx64, dw64)."""
    from . import PW_RELU_BWD, pointwise_ext
    y = round_to_storage(linear_member(dict(m, act=1), dt), dt)
    dz = round_to_storage(pointwise_ext(dy, y, PW_RELU_BWD, [], dt), dt)
    return dict(y=y, dz=dz, db64=linear_bias_grad(dz, dt), dx64=linear_dgrad(dz, m["w"], dt), dw64=linear_wgrad(dz, m["x"], dt))


def linear_act_backward(m, dy, act, dt=BF16):
    """The whole backward of one member y = act(x W^T + b) for act in {1 relu, 2 tanh, 3 sigmoid}, one op at a time,
    the activation's derivative taken from the STORED forward output y (pointwise_ext ops 11 / 12 / 13):
    dz (storage), db = column sums of dz, dX = dz W, dW = dz^T x.  -> dict(y, dz, db64, dx64, dw64)."""
    from . import PW_RELU_BWD, PW_SIGMOID_BWD, PW_TANH_BWD, pointwise_ext
    op = {1: PW_RELU_BWD, 2: PW_TANH_BWD, 3: PW_SIGMOID_BWD}[act]
    y = round_to_storage(linear_member(dict(m, act=act), dt), dt)
    dz = round_to_storage(pointwise_ext(dy, y, op, [], dt), dt)
    return dict(y=y, dz=dz, db64=linear_bias_grad(dz, dt), dx64=linear_dgrad(dz, m["w"], dt), dw64=linear_wgrad(dz, m["x"], dt))
