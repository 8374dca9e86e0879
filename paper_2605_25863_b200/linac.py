"""Thin Python binding of the C ABI in include/linac.h (ctypes; argument marshalling only).

PyTorch is used for device memory and streams, nothing else: every step of the path runs in the
library's CUDA kernels.  There is NO CPU fallback -- importing this module on a box where
`liblinac.so` cannot be loaded, or calling it without a CUDA device, raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblinac.so")

OK, ERR_INVALID_ARG, ERR_BAD_MODULUS, ERR_WORKSPACE, ERR_CUDA = 0, 1, 2, 3, 4
ERR_SINGULAR, ERR_BUFFER_TOO_SMALL, ERR_UNSUPPORTED_DEVICE, ERR_INTERNAL = 5, 6, 7, 8
ERR_TOO_LARGE = 9
STATIC_SCRATCH_BYTES = 32 << 20          # linac.h: LINAC_STATIC_SCRATCH_BYTES

#: every symbol include/linac.h declares (checked by tests/test_abi.py)
SYMBOLS = [
    "linac_status_string", "linac_last_cuda_error", "linac_version",
    "linac_rref_u32_workspace", "linac_solve_f64_workspace", "linac_set_workspace", "linac_release",
    "linac_rref_u64_workspace", "linac_rref_u64",
    "linac_rref_u32", "linac_nullspace_u32", "linac_nullspace_from_rref_u32", "linac_solve_u32", "linac_rank_factor_u32", "linac_load_matrix_u32", "linac_gemm_sub_u32",
    "linac_gemm_sub_u32_static",
    "linac_solve_f64", "linac_rref_f64_workspace", "linac_rref_f64", "linac_rref_c128_workspace", "linac_rref_c128",
    "linac_get_last_stats", "linac_get_last_marks", "linac_set_option", "linac_measure_peak",
]


class LinacError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = _lib().linac_status_string(status).decode()
        if status == ERR_CUDA:
            msg += ": " + _lib().linac_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} (status {status})")


class Stats(C.Structure):
    _fields_ = [("kernel_launches", C.c_int64), ("host_syncs", C.c_int64), ("panels", C.c_int64),
                ("row_swaps", C.c_int64), ("update_macs", C.c_int64), ("residual_nonzero", C.c_int64), ("tc_launches", C.c_int64),
                ("ms_update", C.c_double), ("ms_total", C.c_double),
                ("ms_strip", C.c_double), ("ms_trsm", C.c_double), ("ms_update_top", C.c_double),
                ("top_m", C.c_int64), ("top_n", C.c_int64), ("top_k", C.c_int64),
                ("ms_overlap", C.c_double), ("lookahead_strips", C.c_int64), ("winv_solves", C.c_int64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_LIB = None


def _lib() -> C.CDLL:
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2605_25863_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i64, u32, sz = C.c_void_p, C.c_int64, C.c_uint32, C.c_size_t
        L.linac_status_string.restype = C.c_char_p
        L.linac_status_string.argtypes = [C.c_int]
        L.linac_last_cuda_error.restype = C.c_char_p
        L.linac_version.restype = C.c_int
        L.linac_rref_u32_workspace.argtypes = [i64, i64, C.POINTER(sz)]
        L.linac_solve_f64_workspace.argtypes = [i64, i64, C.POINTER(sz)]
        L.linac_set_workspace.argtypes = [vp, sz]
        L.linac_rref_u32.argtypes = [vp, i64, i64, i64, u32, vp, C.POINTER(i64), vp]
        L.linac_rref_u64_workspace.argtypes = [i64, i64, C.POINTER(sz)]
        L.linac_rref_u64.argtypes = [vp, i64, i64, i64, C.c_uint64, vp, C.POINTER(i64), vp]
        L.linac_nullspace_u32.argtypes = [vp, i64, i64, i64, u32, vp, C.POINTER(i64), vp, vp, i64, i64, C.POINTER(i64)]
        L.linac_nullspace_from_rref_u32.argtypes = [vp, i64, i64, i64, u32, i64, vp, vp, i64, vp]
        L.linac_solve_u32.argtypes = [vp, i64, i64, i64, i64, u32, vp, C.POINTER(i64), vp, vp, vp, i64]
        L.linac_rank_factor_u32.argtypes = [vp, i64, i64, i64, u32, vp, vp, i64, vp, i64, C.POINTER(i64), vp]
        L.linac_load_matrix_u32.argtypes = [vp, i64, i64, i64, vp, i64, i64, vp, i64, u32, vp]
        L.linac_gemm_sub_u32.argtypes = [vp, i64, vp, i64, vp, i64, i64, i64, i64, u32, C.c_int, vp]
        L.linac_gemm_sub_u32_static.argtypes = [vp, i64, vp, i64, vp, i64, i64, i64, i64, u32, vp]
        L.linac_solve_f64.argtypes = [vp, i64, i64, vp, i64, i64, C.c_double, vp, C.POINTER(i64)]
        L.linac_rref_f64_workspace.argtypes = [i64, i64, C.POINTER(sz)]
        L.linac_rref_f64.argtypes = [vp, i64, i64, i64, C.c_double, vp, C.POINTER(i64), vp]
        L.linac_rref_c128_workspace.argtypes = [i64, i64, C.POINTER(sz)]
        L.linac_rref_c128.argtypes = [vp, i64, i64, i64, C.c_double, vp, C.POINTER(i64), vp]
        L.linac_measure_peak.argtypes = [C.c_char_p, C.c_double, vp, sz, vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.linac_get_last_stats.argtypes = [C.POINTER(Stats)]
        L.linac_get_last_marks.argtypes = [C.POINTER(Mark), i64, C.POINTER(i64)]
        L.linac_set_option.argtypes = [C.c_char_p, i64]
        _LIB = L
    return _LIB


def version() -> int:
    return int(_lib().linac_version())


def set_option(name: str, value: int) -> None:
    rc = _lib().linac_set_option(name.encode(), int(value))
    if rc:
        raise LinacError(rc, f"linac_set_option({name})")


class Mark(C.Structure):
    _fields_ = [("cls", C.c_int32), ("stream", C.c_int32), ("m", C.c_int64), ("n", C.c_int64), ("k", C.c_int64),
                ("t0_ms", C.c_float), ("t1_ms", C.c_float)]


def last_marks() -> list:
    """Per-launch intervals of this thread's last rref_u32 call made with set_option("timing", 2) (mirrors
    linac_get_last_marks): dicts with cls (0 update, 1 strip kernel, 2 row-block solve), stream, m, n, k, t0_ms, t1_ms."""
    n = C.c_int64(0)
    _lib().linac_get_last_marks(None, 0, C.byref(n))
    buf = (Mark * max(1, n.value))()
    _lib().linac_get_last_marks(buf, n.value, C.byref(n))
    return [{k: getattr(buf[i], k) for k, _ in Mark._fields_} for i in range(n.value)]


def last_stats() -> dict:
    s = Stats()
    _lib().linac_get_last_stats(C.byref(s))
    return s.as_dict()


import threading

_tls = threading.local()      # the library keeps its workspace binding per host thread; so does this binding


def _ensure_workspace(nbytes: int, device) -> None:
    """Workspace is a torch allocation handed to the library (the caller owns device memory); one per Python thread."""
    if nbytes == 0:
        return
    ws = getattr(_tls, "ws", None)
    if ws is None or ws.numel() < nbytes or ws.device != device:
        _lib().linac_set_workspace(None, 0)
        _tls.ws = None
        _tls.ws = torch.empty(nbytes, dtype=torch.uint8, device=device)
        rc = _lib().linac_set_workspace(_tls.ws.data_ptr(), _tls.ws.numel())
        if rc:
            raise LinacError(rc, "linac_set_workspace")


def release_workspace() -> None:
    _lib().linac_set_workspace(None, 0)
    _lib().linac_release()
    _tls.ws = None


def _check_matrix(t: torch.Tensor, dtypes, what: str):
    if not t.is_cuda:
        raise ValueError(f"{what} must be a CUDA tensor (there is no CPU path)")
    if t.dtype not in dtypes:
        raise TypeError(f"{what}: dtype {t.dtype} not in {dtypes}")
    if t.dim() != 2 or (t.numel() and t.stride(1) != 1):
        raise ValueError(f"{what} must be 2-D with unit column stride")
    ld = t.stride(0) if t.shape[0] > 1 else max(t.shape[1], t.stride(0) if t.shape[0] else 0)
    return t.shape[0], t.shape[1], max(ld, t.shape[1])


def _stream_ptr(device):
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


_U32 = (torch.uint32, torch.int32)


def rref_u32(a: torch.Tensor, p: int):
    """In place: `a` (CUDA, uint32/int32 storage, rows x cols, row stride = ld) -> its RREF over F_p.

    Returns (rank, pivot_cols) with pivot_cols a host int32 tensor.  Mirrors linac_rref_u32.
    """
    rows, cols, ld = _check_matrix(a, _U32, "a")
    with torch.cuda.device(a.device):
        need = C.c_size_t(0)
        _lib().linac_rref_u32_workspace(rows, cols, C.byref(need))
        _ensure_workspace(need.value, a.device)
        rank = C.c_int64(0)
        piv = torch.empty(max(1, min(rows, cols)), dtype=torch.int32)
        rc = _lib().linac_rref_u32(a.data_ptr(), rows, cols, ld, p, _stream_ptr(a.device), C.byref(rank), piv.data_ptr())
    if rc:
        raise LinacError(rc, "linac_rref_u32")
    return int(rank.value), piv[: rank.value].clone()


def rref_u64(a: torch.Tensor, p: int):
    """In place: `a` (CUDA, int64/uint64 storage holding uint64 residues) -> its RREF over F_p, odd prime p < 2^63
    (the 64-bit backend of PAPER.md:163).  Returns (rank, pivot_cols).  Mirrors linac_rref_u64."""
    rows, cols, ld = _check_matrix(a, (torch.int64, torch.uint64), "a")
    with torch.cuda.device(a.device):
        need = C.c_size_t(0)
        _lib().linac_rref_u64_workspace(rows, cols, C.byref(need))
        _ensure_workspace(need.value, a.device)
        rank = C.c_int64(0)
        piv = torch.empty(max(1, min(rows, cols)), dtype=torch.int32)
        rc = _lib().linac_rref_u64(a.data_ptr(), rows, cols, ld, p, _stream_ptr(a.device), C.byref(rank), piv.data_ptr())
    if rc:
        raise LinacError(rc, "linac_rref_u64")
    return int(rank.value), piv[: rank.value].clone()


def nullspace_u32(a: torch.Tensor, p: int, k: torch.Tensor | None = None):
    """Reduce `a` in place and return (rank, pivot_cols, K) with K = cols x nullity on the device.

    If `k` is given it is used as the output buffer (cols x capacity); too small -> LinacError with
    status ERR_BUFFER_TOO_SMALL (a then holds the RREF).  If `k` is None the nullity is found first
    with a capacity-0 call semantics: the RREF is computed once, K allocated, then filled by
    linac_nullspace_from_rref_u32.
    """
    rows, cols, ld = _check_matrix(a, _U32, "a")
    with torch.cuda.device(a.device):
        need = C.c_size_t(0)
        _lib().linac_rref_u32_workspace(rows, cols, C.byref(need))
        _ensure_workspace(need.value, a.device)
        rank, nullity = C.c_int64(0), C.c_int64(0)
        piv = torch.empty(max(1, min(rows, cols)), dtype=torch.int32)
        if k is not None:
            krows, kcap, ldk = _check_matrix(k, _U32, "k")
            if krows != cols:
                raise ValueError("k must have `cols` rows")
            rc = _lib().linac_nullspace_u32(a.data_ptr(), rows, cols, ld, p, _stream_ptr(a.device), C.byref(rank),
                                            piv.data_ptr(), k.data_ptr(), ldk, kcap, C.byref(nullity))
            if rc:
                raise LinacError(rc, "linac_nullspace_u32")
            return int(rank.value), piv[: rank.value].clone(), k[:, : nullity.value]
        rc = _lib().linac_nullspace_u32(a.data_ptr(), rows, cols, ld, p, _stream_ptr(a.device), C.byref(rank),
                                        piv.data_ptr(), None, 0, 0, C.byref(nullity))
        if rc not in (OK, ERR_BUFFER_TOO_SMALL):
            raise LinacError(rc, "linac_nullspace_u32")
        d = int(nullity.value)
        kk = torch.empty((cols, d), dtype=a.dtype, device=a.device)
        if d:
            rc = _lib().linac_nullspace_from_rref_u32(a.data_ptr(), rows, cols, ld, p, rank.value, piv.data_ptr(),
                                                      kk.data_ptr(), d, _stream_ptr(a.device))
            if rc:
                raise LinacError(rc, "linac_nullspace_from_rref_u32")
    return int(rank.value), piv[: rank.value].clone(), kk


def solve_u32(m: torch.Tensor, cols: int, p: int):
    """In place: `m` = (A | B) (CUDA, uint32/int32 storage, rows x (cols + nrhs)) -> its RREF over F_p.

    Returns (rank_a, pivot_cols, consistent, X): X is cols x nrhs on the device (particular solutions, free variables
    zero; zero columns for inconsistent right-hand sides), `consistent` a host bool tensor.  Mirrors linac_solve_u32.
    """
    rows, wide, ld = _check_matrix(m, _U32, "m")
    nrhs = wide - cols
    if cols < 0 or nrhs < 0:
        raise ValueError("cols must lie in [0, m.shape[1]]")
    with torch.cuda.device(m.device):
        need = C.c_size_t(0)
        _lib().linac_rref_u32_workspace(rows, wide, C.byref(need))
        _ensure_workspace(need.value, m.device)
        rank_a = C.c_int64(0)
        piv = torch.empty(max(1, min(rows, wide)), dtype=torch.int32)
        cons = torch.zeros(max(1, nrhs), dtype=torch.uint8)
        x = torch.zeros((cols, nrhs), dtype=m.dtype, device=m.device)
        rc = _lib().linac_solve_u32(m.data_ptr(), rows, cols, nrhs, ld, p, _stream_ptr(m.device), C.byref(rank_a),
                                    piv.data_ptr(), cons.data_ptr(), x.data_ptr() if x.numel() else None, max(1, nrhs))
        if rc:
            raise LinacError(rc, "linac_solve_u32")
    return int(rank_a.value), piv, cons[:nrhs].bool(), x


def rank_factor_u32(a: torch.Tensor, p: int):
    """Rank factorisation A = C.R over F_p (eq. 7): `a` is left untouched.  Returns (rank, pivot_cols, C, R) with
    C = a[:, pivot_cols] mod p (rows x rank) and R the non-zero rows of the RREF (rank x cols), both on the device
    (views of freshly allocated buffers).  Mirrors linac_rank_factor_u32."""
    rows, cols, ld = _check_matrix(a, _U32, "a")
    cap = min(rows, cols)
    with torch.cuda.device(a.device):
        need = C.c_size_t(0)
        _lib().linac_rref_u32_workspace(rows, cols, C.byref(need))
        _ensure_workspace(need.value, a.device)
        rank = C.c_int64(0)
        piv = torch.empty(max(1, cap), dtype=torch.int32)
        r = torch.empty((rows, cols), dtype=a.dtype, device=a.device)
        c = torch.empty((rows, cap), dtype=a.dtype, device=a.device)
        rc = _lib().linac_rank_factor_u32(a.data_ptr() if a.numel() else None, rows, cols, ld, p, _stream_ptr(a.device),
                                          r.data_ptr() if r.numel() else None, max(cols, 1),
                                          c.data_ptr() if c.numel() else None, max(cap, 1), C.byref(rank), piv.data_ptr())
    if rc:
        raise LinacError(rc, "linac_rank_factor_u32")
    k = int(rank.value)
    return k, piv[:k].clone(), c[:, :k], r[:k]


def load_matrix_u32(bases: torch.Tensor, lindices: torch.Tensor, p: int, out: torch.Tensor | None = None) -> torch.Tensor:
    """A[r][c] = prod_t bases[r][lindices[c][t]] mod p on the device (mirrors linac_load_matrix_u32).

    bases: CUDA n_rows x n_basis (uint32/int32 storage); lindices: CUDA n_cols x d int32, contiguous; an index outside
    [0, n_basis) means "no factor".  Returns the n_rows x n_cols matrix (uint32 bits in an int32 tensor unless `out`)."""
    n_rows, n_basis, ldb = _check_matrix(bases, _U32, "bases")
    if lindices.dtype != torch.int32 or lindices.dim() != 2 or not lindices.is_cuda or not lindices.is_contiguous():
        raise ValueError("lindices must be a contiguous CUDA int32 tensor of shape (n_cols, d)")
    n_cols, d = lindices.shape
    if out is None:
        out = torch.empty((n_rows, n_cols), dtype=torch.int32, device=bases.device)
    orow, ocol, ld = _check_matrix(out, _U32, "out")
    if (orow, ocol) != (n_rows, n_cols):
        raise ValueError("out has the wrong shape")
    with torch.cuda.device(bases.device):
        rc = _lib().linac_load_matrix_u32(out.data_ptr(), n_rows, n_cols, ld, bases.data_ptr(), n_basis, ldb,
                                          lindices.data_ptr() if lindices.numel() else None, d, p, _stream_ptr(bases.device))
    if rc:
        raise LinacError(rc, "linac_load_matrix_u32")
    return out


def nullspace_from_rref_u32(r: torch.Tensor, p: int, rank: int, pivot_cols: torch.Tensor) -> torch.Tensor:
    rows, cols, ld = _check_matrix(r, _U32, "r")
    piv = pivot_cols.to(dtype=torch.int32, device="cpu").contiguous()
    d = cols - rank
    k = torch.empty((cols, d), dtype=r.dtype, device=r.device)
    with torch.cuda.device(r.device):
        rc = _lib().linac_nullspace_from_rref_u32(r.data_ptr(), rows, cols, ld, p, rank, piv.data_ptr(),
                                                  k.data_ptr() if d else None, max(d, 1), _stream_ptr(r.device))
    if rc:
        raise LinacError(rc, "linac_nullspace_from_rref_u32")
    return k


def gemm_sub_u32(c: torch.Tensor, a: torch.Tensor, b: torch.Tensor, p: int, path: int = 0) -> None:
    """In place: c <- c - a.b (mod p) on the device (S5 primitive).  path 0 auto, 1 CUDA cores, 2 tensor cores."""
    m, n, ldc = _check_matrix(c, _U32, "c")
    m2, k, lda = _check_matrix(a, _U32, "a")
    k2, n2, ldb = _check_matrix(b, _U32, "b")
    if m != m2 or n != n2 or k != k2:
        raise ValueError("shape mismatch")
    with torch.cuda.device(c.device):
        rc = _lib().linac_gemm_sub_u32(c.data_ptr(), ldc, a.data_ptr(), lda, b.data_ptr(), ldb, m, n, k, p, path,
                                       _stream_ptr(c.device))
    if rc:
        raise LinacError(rc, "linac_gemm_sub_u32")


def gemm_sub_u32_static(c: torch.Tensor, a: torch.Tensor, b: torch.Tensor, p: int) -> None:
    """In place: c <- c - a.b (mod p), enqueued on the current stream WITHOUT allocating device memory and without a
    synchronisation (scratch in the library's static 32 MiB device array; LinacError(ERR_TOO_LARGE) beyond it).
    Calls on one device share that array: do not let two of them overlap on the GPU."""
    m, n, ldc = _check_matrix(c, _U32, "c")
    m2, k, lda = _check_matrix(a, _U32, "a")
    k2, n2, ldb = _check_matrix(b, _U32, "b")
    if m != m2 or n != n2 or k != k2:
        raise ValueError("shape mismatch")
    with torch.cuda.device(c.device):
        rc = _lib().linac_gemm_sub_u32_static(c.data_ptr(), ldc, a.data_ptr(), lda, b.data_ptr(), ldb, m, n, k, p,
                                              _stream_ptr(c.device))
    if rc:
        raise LinacError(rc, "linac_gemm_sub_u32_static")


def solve_f64(a: torch.Tensor, b: torch.Tensor, tol: float = -1.0) -> int:
    """In place: solves a x = b (a: n x n float64 CUDA, overwritten by factors; b: n x nrhs, becomes x).

    Returns info (0).  A singular pivot raises LinacError(status ERR_SINGULAR) with `.info` set.
    """
    n, n2, lda = _check_matrix(a, (torch.float64,), "a")
    nb, nrhs, ldb = _check_matrix(b, (torch.float64,), "b")
    if n != n2 or nb != n:
        raise ValueError("a must be n x n and b n x nrhs")
    with torch.cuda.device(a.device):
        need = C.c_size_t(0)
        _lib().linac_solve_f64_workspace(n, nrhs, C.byref(need))
        _ensure_workspace(need.value, a.device)
        info = C.c_int64(0)
        rc = _lib().linac_solve_f64(a.data_ptr(), n, lda, b.data_ptr(), nrhs, ldb, float(tol), _stream_ptr(a.device),
                                    C.byref(info))
    if rc:
        err = LinacError(rc, "linac_solve_f64")
        err.info = int(info.value)
        raise err
    return int(info.value)


def rref_f64(a: torch.Tensor, tol: float = -1.0):
    """In place: `a` (CUDA float64, rows x cols) -> its reduced row-echelon form with the threshold `tol` on the
    row-scaled matrix (the paper's floating-point mode).  Returns (rank, pivot_cols).  Mirrors linac_rref_f64."""
    rows, cols, ld = _check_matrix(a, (torch.float64,), "a")
    with torch.cuda.device(a.device):
        need = C.c_size_t(0)
        _lib().linac_rref_f64_workspace(rows, cols, C.byref(need))
        _ensure_workspace(need.value, a.device)
        rank = C.c_int64(0)
        piv = torch.empty(max(1, min(rows, cols)), dtype=torch.int32)
        rc = _lib().linac_rref_f64(a.data_ptr(), rows, cols, ld, float(tol), _stream_ptr(a.device), C.byref(rank),
                                   piv.data_ptr())
    if rc:
        raise LinacError(rc, "linac_rref_f64")
    return int(rank.value), piv[: rank.value].clone()


def rref_c128(a: torch.Tensor, tol: float = -1.0):
    """In place: `a` (CUDA complex128, rows x cols) -> its reduced row-echelon form with the threshold `tol` on the
    row-scaled matrix.  Returns (rank, pivot_cols).  Mirrors linac_rref_c128."""
    rows, cols, ld = _check_matrix(a, (torch.complex128,), "a")
    with torch.cuda.device(a.device):
        need = C.c_size_t(0)
        _lib().linac_rref_c128_workspace(rows, cols, C.byref(need))
        _ensure_workspace(need.value, a.device)
        rank = C.c_int64(0)
        piv = torch.empty(max(1, min(rows, cols)), dtype=torch.int32)
        rc = _lib().linac_rref_c128(a.data_ptr(), rows, cols, ld, float(tol), _stream_ptr(a.device), C.byref(rank),
                                    piv.data_ptr())
    if rc:
        raise LinacError(rc, "linac_rref_c128")
    return int(rank.value), piv[: rank.value].clone()


def measure_peak(what: str, ms_target: float = 2.0, scratch: torch.Tensor | None = None):
    """Microbenchmark of one pipe (mirrors linac_measure_peak).  Returns (value, sm_mhz)."""
    dev = scratch.device if scratch is not None else torch.device("cuda", torch.cuda.current_device())
    with torch.cuda.device(dev):
        val, mhz = C.c_double(0), C.c_double(0)
        rc = _lib().linac_measure_peak(what.encode(), float(ms_target), scratch.data_ptr() if scratch is not None else None,
                                       scratch.numel() * scratch.element_size() if scratch is not None else 0,
                                       _stream_ptr(dev), C.byref(val), C.byref(mhz))
    if rc:
        raise LinacError(rc, f"linac_measure_peak({what})")
    return float(val.value), float(mhz.value)
