"""CPU oracle for the Linac hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes/numpy wrappers over `oracle/linac_oracle.c` (plain C, `%` arithmetic, the paper's
one-column-at-a-time Gauss-Jordan loop; citations are in the C file's header).  Only
`tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this package; nothing under `paper_2605_25863_b200/` does, and this package
imports nothing from there.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): every function here is pinned against
something other than itself -- brute force over tiny fields, Leibniz determinants, closed
forms (Vandermonde), Python big-int arithmetic, sympy's GF(p) RREF as a black box, LAPACK
for fp64, exact rational RREF and SVD rank for the floating-point RREF.  No function is "parity unpinned".
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

PIVOT_FIRST, PIVOT_LAST, PIVOT_MAX = 0, 1, 2

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        u32p, i32p, i64p, f64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_int32), C.POINTER(C.c_int64),
                                  C.POINTER(C.c_double))
        L.oracle_inv_modp.restype = C.c_uint32
        L.oracle_inv_modp.argtypes = [C.c_uint32, C.c_uint32]
        L.oracle_pow_modp.restype = C.c_uint32
        L.oracle_pow_modp.argtypes = [C.c_uint32, C.c_uint64, C.c_uint32]
        L.oracle_max_threads.restype = C.c_int
        L.oracle_rref_modp.restype = C.c_int
        L.oracle_rref_modp.argtypes = [u32p, C.c_int64, C.c_int64, C.c_int64, C.c_uint32, C.c_int, C.c_int, i64p, i32p]
        L.oracle_det_modp.restype = C.c_int
        L.oracle_det_modp.argtypes = [u32p, C.c_int64, C.c_int64, C.c_uint32, u32p]
        L.oracle_nullspace_modp.restype = C.c_int
        L.oracle_nullspace_modp.argtypes = [u32p, C.c_int64, C.c_int64, C.c_int64, C.c_uint32, C.c_int64, i32p, u32p,
                                            C.c_int64]
        L.oracle_matmul_modp.restype = C.c_int
        L.oracle_matmul_modp.argtypes = [u32p, C.c_int64, u32p, C.c_int64, u32p, C.c_int64, C.c_int64, C.c_int64,
                                         C.c_int64, C.c_uint32, C.c_int]
        L.oracle_solve_f64.restype = C.c_int
        L.oracle_solve_f64.argtypes = [f64p, C.c_int64, C.c_int64, f64p, C.c_int64, C.c_int64, C.c_double, C.c_int, i64p]
        u64p = C.POINTER(C.c_uint64)
        L.oracle_inv_modp64.restype = C.c_uint64
        L.oracle_inv_modp64.argtypes = [C.c_uint64, C.c_uint64]
        L.oracle_rref_modp64.restype = C.c_int
        L.oracle_rref_modp64.argtypes = [u64p, C.c_int64, C.c_int64, C.c_int64, C.c_uint64, C.c_int, C.c_int, i64p, i32p]
        L.oracle_matmul_modp64.restype = C.c_int
        L.oracle_matmul_modp64.argtypes = [u64p, C.c_int64, u64p, C.c_int64, u64p, C.c_int64, C.c_int64, C.c_int64,
                                           C.c_int64, C.c_uint64, C.c_int]
        L.oracle_rref_f64.restype = C.c_int
        L.oracle_rref_f64.argtypes = [f64p, C.c_int64, C.c_int64, C.c_int64, C.c_double, C.c_int, i64p, i32p]
        L.oracle_rref_c128.restype = C.c_int
        L.oracle_rref_c128.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_double, C.c_int, i64p, i32p]
        L.oracle_backward_error.restype = C.c_double
        L.oracle_backward_error.argtypes = [f64p, C.c_int64, C.c_int64, f64p, C.c_int64, f64p, C.c_int64, C.c_int64,
                                            C.c_int]
        _lib = L
    return _lib


def _u32(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint32))


def _f64(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def inv_modp(a: int, p: int) -> int:
    return int(lib().oracle_inv_modp(a, p))


def pow_modp(a: int, e: int, p: int) -> int:
    return int(lib().oracle_pow_modp(a, e, p))


def rref_modp(a: np.ndarray, p: int, pivot_rule: int = PIVOT_FIRST, nthreads: int = 1, ld: int | None = None):
    """RREF over F_p of the 2-D uint32 array `a` (not modified).  Returns (R, rank, pivot_cols).

    With `ld` > cols the matrix is embedded in a padded buffer (padding filled with a sentinel)
    and the test that padding is untouched is left to the caller via the returned full buffer.
    """
    a = np.ascontiguousarray(a, dtype=np.uint32)
    rows, cols = a.shape
    r = a.copy()
    rank = C.c_int64(0)
    piv = np.zeros(max(1, min(rows, cols)), dtype=np.int32)
    rc = lib().oracle_rref_modp(_u32(r), rows, cols, cols if ld is None else ld, p, pivot_rule, nthreads,
                                C.byref(rank), piv.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc != 0:
        raise ValueError(f"oracle_rref_modp failed: {rc}")
    return r, int(rank.value), piv[: rank.value].copy()


def det_modp(a: np.ndarray, p: int) -> int:
    a = np.ascontiguousarray(a, dtype=np.uint32).copy()
    n = a.shape[0]
    assert a.shape == (n, n)
    d = C.c_uint32(0)
    rc = lib().oracle_det_modp(_u32(a), n, n, p, C.byref(d))
    if rc != 0:
        raise ValueError(f"oracle_det_modp failed: {rc}")
    return int(d.value)


def nullspace_modp(r: np.ndarray, p: int, rank: int, pivot_cols: np.ndarray) -> np.ndarray:
    """Canonical kernel basis K (cols x (cols-rank)) from an RREF `r`."""
    r = np.ascontiguousarray(r, dtype=np.uint32)
    rows, cols = r.shape
    d = cols - rank
    k = np.zeros((cols, max(d, 0)), dtype=np.uint32)
    piv = np.ascontiguousarray(pivot_cols, dtype=np.int32)
    if piv.size == 0:
        piv = np.zeros(1, dtype=np.int32)
    kbuf = k if d > 0 else np.zeros((max(cols, 1), 1), dtype=np.uint32)
    rc = lib().oracle_nullspace_modp(_u32(r), rows, cols, cols, p, rank, piv.ctypes.data_as(C.POINTER(C.c_int32)),
                                     _u32(kbuf), max(d, 1) if d == 0 else d)
    if rc != 0:
        raise ValueError(f"oracle_nullspace_modp failed: {rc}")
    return k


def solve_modp(a: np.ndarray, b: np.ndarray, p: int, nthreads: int = 1):
    """A X = B over F_p, ONE right-hand side at a time, exactly as the paper states it:
    reduce M = (A | b) (eq. 11); the system is consistent iff the augmented column is not a pivot column (eq. 13-14);
    then the pivot columns of A are the solved variables, the free variables are set to zero.
    Returns (consistent bool[nrhs], X uint32[cols, nrhs]) with zero columns for inconsistent right-hand sides.
    Pinned in tests/test_oracle_modp.py: A.x = b by a plain product, and consistency against brute-force
    enumeration of all p^cols vectors over tiny fields."""
    a = np.ascontiguousarray(a, dtype=np.uint32)
    b = np.ascontiguousarray(b, dtype=np.uint32)
    rows, cols = a.shape
    nrhs = b.shape[1]
    cons = np.zeros(nrhs, dtype=bool)
    x = np.zeros((cols, nrhs), dtype=np.uint32)
    for j in range(nrhs):
        m = np.ascontiguousarray(np.hstack([a, b[:, j:j + 1]]))
        r, rank, piv = rref_modp(m, p, nthreads=nthreads)
        if rank > 0 and piv[rank - 1] == cols:          # the augmented column became a pivot column: (0 ... 0 | 1)
            continue
        cons[j] = True
        for k in range(rank):
            x[piv[k], j] = r[k, cols]
    return cons, x


def rank_factor_modp(a: np.ndarray, p: int, nthreads: int = 1):
    """Rank factorisation A = C.R exactly as the paper states it (eq. 7): R = the RREF of A with its
    bottom zero rows dropped, J = its pivot columns, C = A[:, J] (entries reduced to [0,p)).  Returns (C, R, J).
    Pinned in tests/test_oracle_modp.py: C.R = A by a plain product, C has full column rank (brute force over a tiny
    field), and the textbook 3x3 example worked by hand."""
    a = np.ascontiguousarray(a, dtype=np.uint32)
    r, rank, piv = rref_modp(a, p, nthreads=nthreads)
    c = (a[:, piv].astype(np.uint64) % np.uint64(p)).astype(np.uint32)
    return np.ascontiguousarray(c), np.ascontiguousarray(r[:rank]), piv


def load_matrix_modp(bases: np.ndarray, lindices: np.ndarray, p: int) -> np.ndarray:
    """A[r][c] = prod_t bases[r][lindices[c][t]] mod p, the definition written out with plain
    numpy integer arithmetic, one factor at a time.  An index outside [0, n_basis) means "no factor" (the reading
    stated in include/linac.h).  Pinned in tests/test_oracle_modp.py against Python big-int products and the closed
    form of a Vandermonde matrix."""
    bases = np.asarray(bases, dtype=np.uint64) % np.uint64(p)
    lind = np.asarray(lindices, dtype=np.int64)
    n_rows, n_basis = bases.shape
    n_cols, d = lind.shape
    a = np.full((n_rows, n_cols), 1 % p, dtype=np.uint64)
    for t in range(d):
        idx = lind[:, t]
        ok = (idx >= 0) & (idx < n_basis)
        factor = np.ones((n_rows, n_cols), dtype=np.uint64)
        if ok.any():
            factor[:, ok] = bases[:, idx[ok]]
        a = a * factor % np.uint64(p)
    return a.astype(np.uint32)


def matmul_modp(a: np.ndarray, b: np.ndarray, p: int, nthreads: int = 1) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.uint32)
    b = np.ascontiguousarray(b, dtype=np.uint32)
    m, k = a.shape
    k2, n = b.shape
    assert k == k2
    c = np.zeros((m, n), dtype=np.uint32)
    if m and n:
        lib().oracle_matmul_modp(_u32(a), max(k, 1), _u32(b), max(n, 1), _u32(c), max(n, 1), m, k, n, p, nthreads)
    return c


def solve_f64(a: np.ndarray, b: np.ndarray, tol: float = -1.0, nthreads: int = 1):
    """Row-scaled partial-pivot Gauss-Jordan solve.  Returns (status, info, X); inputs untouched."""
    a = np.ascontiguousarray(a, dtype=np.float64).copy()
    b2 = np.ascontiguousarray(b, dtype=np.float64)
    x = (b2.reshape(-1, 1) if b2.ndim == 1 else b2).copy()
    n = a.shape[0]
    info = C.c_int64(0)
    rc = lib().oracle_solve_f64(_f64(a), n, n, _f64(x), x.shape[1], x.shape[1], tol, nthreads, C.byref(info))
    if rc < 0:
        raise ValueError("oracle_solve_f64: bad arguments")
    return rc, int(info.value), (x.reshape(b2.shape) if rc == 0 else None)


def backward_error(a0: np.ndarray, x: np.ndarray, b0: np.ndarray, nthreads: int = 1) -> float:
    a0 = np.ascontiguousarray(a0, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.float64)
    b0 = np.ascontiguousarray(b0, dtype=np.float64)
    if x.ndim == 1:
        x = x.reshape(-1, 1)
        b0 = b0.reshape(-1, 1)
    n = a0.shape[0]
    return float(lib().oracle_backward_error(_f64(a0), n, n, _f64(x), x.shape[1], _f64(b0), b0.shape[1],
                                             x.shape[1], nthreads))


# ---- 64-bit backend ---------------------------------------------------

def _u64(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint64))


def inv_modp64(a: int, p: int) -> int:
    return int(lib().oracle_inv_modp64(a, p))


def rref_modp64(a: np.ndarray, p: int, pivot_rule: int = PIVOT_FIRST, nthreads: int = 1):
    """RREF over F_p of a 2-D uint64 array, p < 2^64: the loop of rref_modp with uint64 storage and `%` on
    unsigned __int128.  Returns (R, rank, pivot_cols).  Pinned in tests/test_oracle_wide.py (Python big-int
    arithmetic, sympy GF(p), agreement with rref_modp for p < 2^32, brute force over tiny fields)."""
    a = np.ascontiguousarray(a, dtype=np.uint64)
    rows, cols = a.shape
    r = a.copy()
    rank = C.c_int64(0)
    piv = np.zeros(max(1, min(rows, cols)), dtype=np.int32)
    rc = lib().oracle_rref_modp64(_u64(r), rows, cols, cols, p, pivot_rule, nthreads, C.byref(rank),
                                  piv.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc != 0:
        raise ValueError(f"oracle_rref_modp64 failed: {rc}")
    return r, int(rank.value), piv[: rank.value].copy()


def matmul_modp64(a: np.ndarray, b: np.ndarray, p: int, nthreads: int = 1) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.uint64)
    b = np.ascontiguousarray(b, dtype=np.uint64)
    m, k = a.shape
    k2, n = b.shape
    assert k == k2
    c = np.zeros((m, n), dtype=np.uint64)
    if m and n:
        lib().oracle_matmul_modp64(_u64(a), max(k, 1), _u64(b), max(n, 1), _u64(c), max(n, 1), m, k, n, p, nthreads)
    return c


# ---- floating-point RREF with a threshold ------------------------

def rref_f64(a: np.ndarray, tol: float = -1.0, nthreads: int = 1):
    """Row-rescaled, partially pivoted Gauss-Jordan reduction of a rectangular float64 matrix with the head compared
    to `tol` (citations in linac_oracle.c).  Returns (R, rank, pivot_cols); the input is untouched.
    Pinned in tests/test_oracle_f64.py: exact rational RREF (sympy) of small integer matrices, numpy SVD rank of
    low-rank products, (A | I) -> (I | A^-1) against LAPACK, the threshold semantics on a planted tiny pivot."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    rows, cols = a.shape
    r = a.copy()
    rank = C.c_int64(0)
    piv = np.zeros(max(1, min(rows, cols)), dtype=np.int32)
    rc = lib().oracle_rref_f64(_f64(r), rows, cols, max(cols, 1), tol, nthreads, C.byref(rank),
                               piv.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc != 0:
        raise ValueError(f"oracle_rref_f64 failed: {rc}")
    return r, int(rank.value), piv[: rank.value].copy()


def rref_c128(a: np.ndarray, tol: float = -1.0, nthreads: int = 1):
    """The same reduction on a complex128 matrix (rows rescaled by their largest real or imaginary part,
    reading Q21; pivot = largest modulus).  Returns (R, rank, pivot_cols); the input is untouched.
    Pinned in tests/test_oracle_c128.py: exact RREF over Q(i) (sympy) of Gaussian-integer matrices, agreement with
    rref_f64 on real input and through the real 2 x 2 block embedding, numpy SVD rank, invariance under row phases."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    rows, cols = a.shape
    r = a.copy()
    rank = C.c_int64(0)
    piv = np.zeros(max(1, min(rows, cols)), dtype=np.int32)
    rc = lib().oracle_rref_c128(r.ctypes.data_as(C.c_void_p), rows, cols, max(cols, 1), tol, nthreads, C.byref(rank),
                                piv.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc != 0:
        raise ValueError(f"oracle_rref_c128 failed: {rc}")
    return r, int(rank.value), piv[: rank.value].copy()
