"""Helpers for the -m gpu parity tests: numpy <-> device plumbing around the C-ABI binding."""
from __future__ import annotations

import numpy as np
import torch

SENTINEL = 0xDEADBEEF


def require_cuda():
    if not torch.cuda.is_available():
        raise RuntimeError("GPU test selected but no CUDA device is visible (there is no CPU fallback)")


def to_device_padded(a: np.ndarray, ld: int | None = None) -> torch.Tensor:
    """rows x ld device buffer (uint32 viewed as int32 for torch), padding columns = SENTINEL."""
    rows, cols = a.shape
    ld = cols if ld is None else ld
    buf = np.full((rows, ld), SENTINEL, dtype=np.uint32)
    buf[:, :cols] = a
    return torch.from_numpy(buf.view(np.int32)).cuda()


def from_device(t: torch.Tensor) -> np.ndarray:
    return t.cpu().numpy().view(np.uint32)


def gpu_rref(a: np.ndarray, p: int, ld: int | None = None):
    import paper_2605_25863_b200 as L
    rows, cols = a.shape
    buf = to_device_padded(a, ld)
    view = buf[:, :cols] if cols else buf
    rank, piv = L.rref_u32(view, p)
    out = from_device(buf)
    if out.shape[1] > cols:
        assert (out[:, cols:] == SENTINEL).all(), "padding columns were written"
    return out[:, :cols].copy(), rank, piv.numpy().copy(), L.last_stats()
