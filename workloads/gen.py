"""Seeded shape and value draws for BASELINE.json configs[0..4].

No method arithmetic lives here (no linear, no LayerNorm, no activation, no
split/cat): only random draws and storage-format packing.  Every tensor comes
from its own counter-based stream, numpy Philox keyed by (seed, tensor id), so
a tensor's values do not depend on the order or number of other draws.
Structure draws (D_i, K_i, N_i, H_i, widths, ops, permutation) use tensor id 0.

Storage formats: F32 -> numpy float32; BF16 -> numpy uint16 holding the raw
bf16 bits (numpy has no bf16).  "N(a, b)" in BASELINE.json is read as mean a,
VARIANCE b.
"""
import numpy as np

F32 = 0   # matches opt_dtype OPT_F32
BF16 = 1  # matches opt_dtype OPT_BF16

ACT_NONE, ACT_RELU, ACT_TANH, ACT_SIGMOID = 0, 1, 2, 3      # opt_act
PW_COPY, PW_RELU, PW_TANH, PW_SIGMOID = 0, 1, 2, 3          # opt_pw_op


# ----------------------------------------------------------------- storage --
def bf16_bits_from_f32(a):
    """float32 array -> uint16 bf16 bits, round-to-nearest-even (finite inputs)."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def f32_from_bf16_bits(u):
    """uint16 bf16 bits -> float32 (exact widening)."""
    return (np.ascontiguousarray(u, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def _store(a32, dtype):
    return a32 if dtype == F32 else bf16_bits_from_f32(a32)


def _stream(seed, tid):
    return np.random.Generator(np.random.Philox(key=[int(seed) & (2**64 - 1), int(tid)]))


def tensor_normal(seed, tid, shape, mean, std, dtype):
    g = _stream(seed, tid)
    a = g.standard_normal(size=shape, dtype=np.float32)
    if std != 1.0:
        a *= np.float32(std)
    if mean != 0.0:
        a += np.float32(mean)
    return _store(a, dtype)


def tensor_uniform(seed, tid, shape, lo, hi, dtype):
    g = _stream(seed, tid)
    a = g.random(size=shape, dtype=np.float32)
    a = a * np.float32(hi - lo) + np.float32(lo)
    return _store(a, dtype)


def _tid(member, role):
    return 1 + member * 16 + role


# ----------------------------------------------------------------- configs --
def config0(seed=0):
    """configs[0]: 4 Linear+bias+tanh members, fp32, M=64.
    X~N(0,1), W~N(0,1/K), b~U(-0.1,0.1)."""
    M = 64
    shapes = [(16, 32), (32, 16), (64, 64), (32, 48)]
    members = []
    for i, (K, N) in enumerate(shapes):
        members.append(dict(
            M=M, K=K, N=N, act=ACT_TANH,
            x=tensor_normal(seed, _tid(i, 0), (M, K), 0.0, 1.0, F32),
            w=tensor_normal(seed, _tid(i, 1), (N, K), 0.0, K ** -0.5, F32),
            b=tensor_uniform(seed, _tid(i, 2), (N,), -0.1, 0.1, F32)))
    return dict(name="config0_tiny_group_linear", dtype=F32, M=M, members=members)


def config1(seed=1, rows=2048, n=64, dims=(64, 128, 192, 256, 384, 512)):
    """configs[1]: n LayerNorm members [rows, D_i] bf16; x~N(mu_i, sigma_i^2),
    mu_i~U(-2,2), sigma_i~U(0.5,4), gamma~N(1,0.1), beta~N(0,0.1), eps=1e-5."""
    s = _stream(seed, 0)
    D = s.choice(np.asarray(dims), size=n)
    mu = s.uniform(-2.0, 2.0, size=n)
    sigma = s.uniform(0.5, 4.0, size=n)
    members = []
    for i in range(n):
        d = int(D[i])
        members.append(dict(
            rows=rows, D=d, eps=1e-5, mu=float(mu[i]), sigma=float(sigma[i]),
            x=tensor_normal(seed, _tid(i, 0), (rows, d), float(mu[i]), float(sigma[i]), BF16),
            gamma=tensor_normal(seed, _tid(i, 1), (d,), 1.0, 0.1 ** 0.5, BF16),
            beta=tensor_normal(seed, _tid(i, 2), (d,), 0.0, 0.1 ** 0.5, BF16)))
    return dict(name="config1_batched_layernorm", dtype=BF16, members=members)


def config2(seed=2, M=4096, n=128, sizes=(128, 256, 512, 1024)):
    """configs[2]: n Linear+bias+ReLU members, bf16, batch M; K_i,N_i iid from
    sizes; X~N(0,1), W~N(0,1/K_i), b~N(0,0.01); concat along dim 1."""
    s = _stream(seed, 0)
    Ks = s.choice(np.asarray(sizes), size=n)
    Ns = s.choice(np.asarray(sizes), size=n)
    members, off = [], 0
    for i in range(n):
        K, N = int(Ks[i]), int(Ns[i])
        members.append(dict(
            M=M, K=K, N=N, act=ACT_RELU, col_off=off,
            x=tensor_normal(seed, _tid(i, 0), (M, K), 0.0, 1.0, BF16),
            w=tensor_normal(seed, _tid(i, 1), (N, K), 0.0, K ** -0.5, BF16),
            b=tensor_normal(seed, _tid(i, 2), (N,), 0.0, 0.1, BF16)))
        off += N
    return dict(name="config2_grouped_linear_tower", dtype=BF16, M=M, members=members,
                concat_width=off)


def config3(seed=3, rows=8192, width=8192, nchunks=256):
    """configs[3]: one [rows,width] bf16 tensor ~N(0,2) split along dim 1 into
    nchunks uneven chunks (multiples of 8, uniform random composition), each
    chunk gets sigmoid/tanh/ReLU (iid), chunks concatenated in a Fisher-Yates
    permutation.  perm[j] = SOURCE chunk placed at output position j (Q14)."""
    s = _stream(seed, 0)
    units = width // 8
    assert units >= nchunks and width % 8 == 0
    cuts = np.sort(s.choice(np.arange(1, units), size=nchunks - 1, replace=False))
    parts = np.diff(np.concatenate(([0], cuts, [units])))
    widths = (parts * 8).astype(np.int64)
    ops = s.choice(np.asarray([PW_SIGMOID, PW_TANH, PW_RELU]), size=nchunks)
    perm = np.arange(nchunks)
    for i in range(nchunks - 1, 0, -1):          # Fisher-Yates
        j = int(s.integers(0, i + 1))
        perm[i], perm[j] = perm[j], perm[i]
    x = tensor_normal(seed, _tid(0, 0), (rows, width), 0.0, 2.0 ** 0.5, BF16)
    return dict(name="config3_split_pointwise_cat", dtype=BF16, rows=rows, width=width,
                x=x, widths=[int(w) for w in widths], ops=[int(o) for o in ops],
                perm=[int(p) for p in perm])


def config4(seed=4, B=8192, n=512, dims=(32, 64, 128, 256), hids=(128, 256, 512), out=64):
    """configs[4]: n towers LayerNorm(D_i) -> Linear(D_i->H_i)+ReLU ->
    Linear(H_i->out); bf16.  BASELINE.json gives shapes only; values reuse the
    laws of configs[1]/[2] (Q22): x~N(0,1), gamma~N(1,0.1), beta~N(0,0.1),
    eps=1e-5, W~N(0,1/fan_in), b~N(0,0.01)."""
    s = _stream(seed, 0)
    D = s.choice(np.asarray(dims), size=n)
    H = s.choice(np.asarray(hids), size=n)
    towers = []
    for i in range(n):
        d, h = int(D[i]), int(H[i])
        towers.append(dict(
            B=B, D=d, H=h, out=out, eps=1e-5,
            x=tensor_normal(seed, _tid(i, 0), (B, d), 0.0, 1.0, BF16),
            gamma=tensor_normal(seed, _tid(i, 1), (d,), 1.0, 0.1 ** 0.5, BF16),
            beta=tensor_normal(seed, _tid(i, 2), (d,), 0.0, 0.1 ** 0.5, BF16),
            w1=tensor_normal(seed, _tid(i, 3), (h, d), 0.0, d ** -0.5, BF16),
            b1=tensor_normal(seed, _tid(i, 4), (h,), 0.0, 0.1, BF16),
            w2=tensor_normal(seed, _tid(i, 5), (out, h), 0.0, h ** -0.5, BF16),
            b2=tensor_normal(seed, _tid(i, 6), (out,), 0.0, 0.1, BF16)))
    return dict(name="config4_recsys_interaction_block", dtype=BF16, B=B, towers=towers,
                concat_width=out * n)


def listing2_example(seed=7, dtype=BF16):
    """Shape of the paper's worked example (Listing 2):
    x:[2,6]; split [2,4] along dim 1; second piece split (2,2); cat of the three
    pieces along dim 1.  Values are arbitrary (the paper uses torch.randn)."""
    x = tensor_normal(seed, 1, (2, 6), 0.0, 1.0, dtype)
    return dict(x=x, first_split=[2, 4], second_split=[2, 2])
