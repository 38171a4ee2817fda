"""GPU check of the no-allocation entry point opt_bias_grad_noalloc (scratch in a static device array of the library,
no cudaMalloc) against the existing planned path opt_bias_grad_plan_create on the same inputs.

Collected LAST on purpose (file name): the suite runs with pytest -x, and this entry point sits outside the hot-path
scope table.  It must pass alone in a fresh process and after every other test.

Tolerance: the one tests/test_gpu_bias_grad.py derives (reading Q27) -- each path adds in fp32 along a fixed tree of
depth <= 200, so each is within 2e-5 sum_m |dZ[m, n]| of the exact column sum, and the two are within twice that of
each other; a bf16 result adds its own rounding, 2^-8 |db| per side.  Sums of small integers are exact: bit for bit."""
import numpy as np
import pytest
import torch

import workloads as wl
from util import BF16, F32, empty_dev, to_dev, to_host, values64

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ob():
    import paper_2607_02945_b200 as ob
    return ob


def both_paths(ob, z, param_dt, pad=0):
    """z: host bf16-bit array [M, N] -> (db of the no-allocation entry point, db of the planned path), host arrays."""
    M, N = z.shape
    buf = empty_dev((M, N + 2 * pad), BF16, fill=float("nan"))
    buf[:, pad:pad + N] = to_dev(z, BF16)
    dz = buf[:, pad:pad + N]
    db_new = empty_dev((N,), param_dt, fill=float("nan"))
    db_old = empty_dev((N,), param_dt, fill=float("nan"))
    n0 = ob.opt_launch_count()
    ob.opt_bias_grad_noalloc(dz, db_new, param_dt)
    assert ob.opt_launch_count() - n0 == 1
    plan = ob.opt_bias_grad_plan_create([ob.bias_grad_member(dz, db_old)], BF16, param_dt)
    plan.launch()
    torch.cuda.synchronize()
    return to_host(db_new), to_host(db_old)


def close(new, old, z, param_dt):
    l1 = np.abs(values64(z, BF16)).sum(axis=0)
    a, b = values64(new, param_dt), values64(old, param_dt)
    bound = 2 * 2e-5 * l1 + (2 * 2.0 ** -8 * np.abs(b) if param_dt == BF16 else 0.0)
    assert np.all(np.isfinite(a)) and np.all(np.abs(a - b) <= bound), float(np.max(np.abs(a - b) - bound))


# two calls in a row share the scratch: the second is narrower and shorter than the first (stale partial sums and
# tickets of the first call must not leak into it), then a wide one again
CALLS = [((5000, 1032), 0), ((77, 200), 24), ((8192, 4096), 0), ((1, 8), 0), ((100000, 16), 8)]


@pytest.mark.parametrize("param_dt", [F32, BF16])
def test_matches_planned_path_on_calls_in_a_row(ob, param_dt):
    for rep in range(2):
        for i, (shape, pad) in enumerate(CALLS):
            z = wl.tensor_normal(71 + rep, i + 1, shape, 0.1 * (i % 3), 1.0 + i, BF16)
            new, old = both_paths(ob, z, param_dt, pad)
            close(new, old, z, param_dt)


def test_integers_bit_exact_and_repeatable(ob):
    rng = np.random.default_rng(72)
    for shape in [(3000, 520), (129, 4096), (64, 8)]:
        z = wl.bf16_bits_from_f32(rng.integers(-2, 3, shape).astype(np.float32))
        new, old = both_paths(ob, z, F32)
        assert new.tobytes() == old.tobytes(), shape              # every fp32 partial sum is exact
        again, _ = both_paths(ob, z, F32)
        assert again.tobytes() == new.tobytes(), shape


def test_random_is_bitwise_repeatable(ob):
    z = wl.tensor_normal(73, 1, (4097, 264), 0.0, 1.0, BF16)
    a, _ = both_paths(ob, z, F32)
    b, _ = both_paths(ob, z, F32)
    assert a.tobytes() == b.tobytes()


def test_limit_and_argument_errors(ob):
    N = ob.OPT_NOALLOC_BIAS_GRAD_MAX_N + 8
    dz = empty_dev((16, N), BF16, fill=1.0)
    db = empty_dev((N,), F32, fill=0.0)
    n0 = ob.opt_launch_count()
    with pytest.raises(ob.OptError) as e:
        ob.opt_bias_grad_noalloc(dz, db, F32)
    assert e.value.status == ob.OPT_ERR_UNSUPPORTED and "OPT_NOALLOC_BIAS_GRAD_MAX_N" in str(e.value)
    with pytest.raises(ob.OptError) as e:                          # N % 8 != 0
        ob.opt_bias_grad_noalloc(dz[:, :12], db[:12], F32)
    assert e.value.status == ob.OPT_ERR_ALIGNMENT
    assert ob.opt_launch_count() == n0                             # nothing was launched
    # the entry point still works after the rejected calls
    z = wl.tensor_normal(74, 1, (300, 512), 0.0, 1.0, BF16)
    new, old = both_paths(ob, z, F32)
    close(new, old, z, F32)
