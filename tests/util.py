"""Helpers for the GPU parity tests: host<->device marshalling and the error
metrics of DESIGN.md.  No method arithmetic."""
import numpy as np
import torch

import workloads as wl

BF16, F32 = wl.BF16, wl.F32


def to_dev(a, dt, device="cuda"):
    """host storage array (uint16 bf16 bits or float32) -> device tensor (same bits)."""
    a = np.ascontiguousarray(a)
    if dt == BF16:
        assert a.dtype == np.uint16
        return torch.from_numpy(a.view(np.int16)).to(device).view(torch.bfloat16)
    assert a.dtype == np.float32
    return torch.from_numpy(a).to(device)


def to_host(t):
    """device tensor -> host storage array (uint16 bits for bf16)."""
    t = t.detach().contiguous().cpu()
    if t.dtype == torch.bfloat16:
        return t.view(torch.int16).numpy().view(np.uint16).copy()
    return t.numpy().copy()


def empty_dev(shape, dt, device="cuda", fill=None):
    t = torch.empty(shape, dtype=torch.bfloat16 if dt == BF16 else torch.float32, device=device)
    if fill is not None:
        t.fill_(fill)
    return t


def bf16_ordinal(u):
    """Q11: map bf16 bits to a signed integer line; +-0 coincide."""
    u = np.asarray(u, dtype=np.uint16).astype(np.int32)
    mag = u & 0x7FFF
    return np.where(u & 0x8000, -mag, mag)


def bf16_ulp_distance(a_bits, b_bits):
    """ulp distance between bf16 patterns; NaN matches only NaN (distance 0), else huge."""
    a, b = np.asarray(a_bits, np.uint16), np.asarray(b_bits, np.uint16)
    d = np.abs(bf16_ordinal(a) - bf16_ordinal(b))
    an, bn = (a & 0x7FFF) > 0x7F80, (b & 0x7FFF) > 0x7F80
    d = np.where(an & bn, 0, d)
    d = np.where(an ^ bn, 1 << 20, d)
    return d


def values64(bits_or_f32, dt):
    if dt == BF16:
        return wl.f32_from_bf16_bits(bits_or_f32).astype(np.float64)
    return np.asarray(bits_or_f32, dtype=np.float64)


def row_l2_rel_err(y, ref64, dt):
    """Q9: max over rows of ||y - ref||_2 / max(||ref||_2, 1e-30), over the member's own columns."""
    y64 = values64(y, dt)
    num = np.linalg.norm(y64 - ref64, axis=1)
    den = np.maximum(np.linalg.norm(ref64, axis=1), 1e-30)
    return float((num / den).max())
