"""The same counter-based generators as gen.py, written with torch integer ops so that the largest
config (c5: 10^5 x 10^5, 40 GB) can be produced straight into device memory, row block by row block.

Bit-identical to gen.py (tests/test_inputs.py compares them on the CPU).  torch has no uint64, so the
64-bit counters live in int64: multiplication and addition wrap mod 2^64 exactly as in uint64, logical
right shifts are an arithmetic shift followed by a mask, and unsigned comparison flips the sign bit.
Like gen.py this module holds none of the method's arithmetic.
"""
from __future__ import annotations

import torch

from . import gen

_I64 = torch.int64


def _c(v: int) -> int:
    """Python int (mod 2^64) -> the int64 with the same bits."""
    v &= 0xFFFFFFFFFFFFFFFF
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    return (x >> k) & ((1 << (64 - k)) - 1)


def splitmix64(seed: int, idx: torch.Tensor) -> torch.Tensor:
    z = idx.to(_I64) + 1
    z = z * _c(0x9E3779B97F4A7C15) + _c(seed)
    z = (z ^ _lsr(z, 30)) * _c(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _c(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def uniform_mod_p(h: torch.Tensor, p: int) -> torch.Tensor:
    """mulhi64(h, p) for p < 2^31 (every term below stays under 2^63).  Returns int64 in [0, p)."""
    assert 0 < p < (1 << 31)
    hi = _lsr(h, 32)
    lo = h & 0xFFFFFFFF
    t = hi * p + _lsr(lo * p, 32)
    return _lsr(t, 32)


def _ult(a: torch.Tensor, b: int) -> torch.Tensor:
    """unsigned a < b for int64-held uint64 values."""
    flip = _c(1 << 63)
    return (a ^ flip) < (_c(b) ^ flip)


def _counters(row_idx: torch.Tensor, cols: int) -> torch.Tensor:
    c = torch.arange(cols, dtype=_I64, device=row_idx.device)
    return row_idx.to(_I64)[:, None] * cols + c[None, :]


def uniform_rows(row0: int, nrows: int, cols: int, p: int, seed: int, device) -> torch.Tensor:
    """int32 tensor holding the uint32 bits of gen.uniform_rows."""
    idx = torch.arange(row0, row0 + nrows, dtype=_I64, device=device)
    return uniform_mod_p(splitmix64(seed, _counters(idx, cols)), p).to(torch.int32)


def _sparse_base_rows(row_idx: torch.Tensor, cols: int, p: int, seed: int) -> torch.Tensor:
    ctr = _counters(row_idx, cols)
    val = uniform_mod_p(splitmix64(seed, ctr), p)
    keep = _ult(splitmix64(seed ^ gen.SPARSE_MASK_TWEAK, ctr), gen.SPARSE_THRESHOLD)
    return torch.where(keep, val, torch.zeros_like(val))


def sparse_dependent_rows(row0: int, nrows: int, rows: int, cols: int, p: int, seed: int, seed_dep: int,
                          period: int = 50, terms: int = 3, device="cpu", plan=None) -> torch.Tensor:
    """Rows [row0, row0+nrows) of config c5's matrix (see gen.sparse_dependent_rows), int32 bits of uint32."""
    idx = torch.arange(row0, row0 + nrows, dtype=_I64, device=device)
    out = _sparse_base_rows(idx, cols, p, seed)
    dep_local = torch.nonzero((idx % period) == (period - 1)).flatten()
    if dep_local.numel():
        if plan is None:
            plan = gen.sparse_dependent_plan(rows, p, seed_dep, period, terms)
        _, src, alpha = plan
        d = (idx[dep_local] // period).cpu().numpy()
        src_t = torch.from_numpy(src[d]).to(device)                    # [nd, terms]
        alpha_t = torch.from_numpy(alpha[d].astype("int64")).to(device)
        acc = torch.zeros((dep_local.numel(), cols), dtype=_I64, device=device)
        for t in range(terms):
            base = _sparse_base_rows(src_t[:, t], cols, p, seed)       # < 2^31, alpha < 2^31: product < 2^62
            acc = (acc + base * alpha_t[:, t:t + 1] % p) % p
        out[dep_local] = acc
    return out.to(torch.int32)


def fill_c5(dst: torch.Tensor, cfg: dict, block_rows: int = 512) -> None:
    """Writes config c5 (or any sparse_dep config) into the device tensor dst (rows x cols int32)."""
    rows, cols = dst.shape
    plan = gen.sparse_dependent_plan(rows, cfg["p"], cfg["seed_dep"], cfg["period"], cfg["terms"])
    for r0 in range(0, rows, block_rows):
        n = min(block_rows, rows - r0)
        dst[r0:r0 + n] = sparse_dependent_rows(r0, n, rows, cols, cfg["p"], cfg["seed"], cfg["seed_dep"],
                                               cfg["period"], cfg["terms"], device=dst.device, plan=plan)
