"""Counter-based seeded generators (numpy, host side).  See the package docstring.

Nothing here eliminates, inverts or reduces a matrix; the only modular arithmetic is what
the *definition of an input* needs (a product of two random factors for the exact-rank
config, a linear combination of rows for the rank-deficient config), written with plain
Python/numpy integer `%`.
"""
from __future__ import annotations

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_MASK32 = np.uint64(0xFFFFFFFF)

#: seed tweak for the independent "is this entry non-zero" draw of the sparse config
SPARSE_MASK_TWEAK = 0x5851F42D4C957F2D
#: floor(0.1 * 2^64): an entry is non-zero iff its mask draw is below this
SPARSE_THRESHOLD = 1844674407370955161

#: The five BASELINE.json configs (sizes, modulus, seeds).  Names follow SURVEY.md 8(d).
CONFIGS = {
    "c1": dict(kind="uniform", rows=512, cols=512, p=2147483647, seed=1),
    "c2": dict(kind="lowrank", rows=4096, cols=4096, inner=3000, p=2147483629, seed_b=2, seed_c=3),
    "c3": dict(kind="uniform", rows=10000, cols=10000, p=2147483647, seed=4),
    "c4": dict(kind="f64", n=16384, nrhs=64, seed_a=5, seed_b=6),
    "c5": dict(kind="sparse_dep", rows=100000, cols=100000, p=2147483647, seed=7, seed_dep=8,
               period=50, terms=3),
}


def splitmix64(seed: int, idx) -> np.ndarray:
    """h(seed, idx) for an array of 64-bit counters `idx` (wraps mod 2^64)."""
    idx = np.asarray(idx, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + _GOLDEN * (idx + np.uint64(1))
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform_mod_p(h: np.ndarray, p: int) -> np.ndarray:
    """mulhi64(h, p) for p < 2^32: maps a 64-bit draw to [0, p).  Returns uint32."""
    assert 0 < p < (1 << 32)
    pp = np.uint64(p)
    hi = h >> np.uint64(32)
    lo = h & _MASK32
    # (hi*2^32 + lo) * p >> 64  ==  (hi*p + ((lo*p) >> 32)) >> 32   (all terms < 2^64)
    t = hi * pp + ((lo * pp) >> np.uint64(32))
    return (t >> np.uint64(32)).astype(np.uint32)


def uniform_mod_p64(h: np.ndarray, p: int) -> np.ndarray:
    """mulhi64(h, p) for any p < 2^64 (the 64-bit backend's inputs): 128-bit product by 32-bit halves.  uint64."""
    assert 0 < p < (1 << 64)
    p1, p0 = np.uint64(p >> 32), np.uint64(p & 0xFFFFFFFF)
    h1, h0 = h >> np.uint64(32), h & _MASK32
    with np.errstate(over="ignore"):
        mid = h1 * p0 + ((h0 * p0) >> np.uint64(32))          # < 2^64
        mid2 = (mid & _MASK32) + h0 * p1                      # < 2^64
        return h1 * p1 + (mid >> np.uint64(32)) + (mid2 >> np.uint64(32))


def uniform_matrix_u64(rows: int, cols: int, p: int, seed: int) -> np.ndarray:
    """rows x cols uint64, i.i.d. uniform in [0, p), p < 2^64; same counters as uniform_matrix."""
    return uniform_mod_p64(splitmix64(seed, _row_counters(0, rows, cols)), p)


def _row_counters(row0: int, nrows: int, cols: int) -> np.ndarray:
    r = np.arange(row0, row0 + nrows, dtype=np.uint64)[:, None]
    c = np.arange(cols, dtype=np.uint64)[None, :]
    return r * np.uint64(cols) + c


def uniform_rows(row0: int, nrows: int, cols: int, p: int, seed: int) -> np.ndarray:
    """Rows [row0, row0+nrows) of the rows x cols i.i.d. uniform-[0,p) matrix of `seed`."""
    return uniform_mod_p(splitmix64(seed, _row_counters(row0, nrows, cols)), p)


def uniform_matrix(rows: int, cols: int, p: int, seed: int, chunk_rows: int = 1024) -> np.ndarray:
    """rows x cols uint32, i.i.d. uniform in [0, p) (configs c1, c3 and the factors of c2)."""
    out = np.empty((rows, cols), dtype=np.uint32)
    for r0 in range(0, rows, chunk_rows):
        n = min(chunk_rows, rows - r0)
        out[r0:r0 + n] = uniform_rows(r0, n, cols, p, seed)
    return out


def _matmul_mod_p_exact(b: np.ndarray, c: np.ndarray, p: int) -> np.ndarray:
    """(b @ c) mod p for uint32 factors, exact: 16-bit halves through float64 BLAS.

    Each partial product sum is < inner * 2^32 <= 2^53 for inner <= 2^21, so float64 is exact.
    This is only how the *input* of the exact-rank config is defined (A = B.C mod p).
    """
    inner = b.shape[1]
    assert inner <= (1 << 21)
    b_lo = (b & 0xFFFF).astype(np.float64)
    b_hi = (b >> 16).astype(np.float64)
    c_lo = (c & 0xFFFF).astype(np.float64)
    c_hi = (c >> 16).astype(np.float64)
    pp = np.uint64(p)

    def red(x):  # float64 exact integer -> uint64 mod p
        return x.astype(np.uint64) % pp

    ll = red(b_lo @ c_lo)
    lh = red(b_lo @ c_hi) + red(b_hi @ c_lo)          # < 2p
    hh = red(b_hi @ c_hi)
    s16 = np.uint64((1 << 16) % p)
    s32 = np.uint64((1 << 32) % p)
    out = (ll + (lh % pp) * s16 % pp + hh * s32 % pp) % pp
    return out.astype(np.uint32)


def lowrank_factors(rows: int, inner: int, cols: int, p: int, seed_b: int, seed_c: int):
    """Config c2: returns (A, B, C) with A = B.C mod p, B rows x inner, C inner x cols uniform."""
    b = uniform_matrix(rows, inner, p, seed_b)
    c = uniform_matrix(inner, cols, p, seed_c)
    a = np.empty((rows, cols), dtype=np.uint32)
    step = 1024
    for r0 in range(0, rows, step):
        a[r0:r0 + step] = _matmul_mod_p_exact(b[r0:r0 + step], c, p)
    return a, b, c


def _sparse_base_rows(row_idx: np.ndarray, cols: int, p: int, seed: int) -> np.ndarray:
    """Independent sparse rows: entry (r,c) is uniform [0,p) with probability 0.1, else 0."""
    r = np.asarray(row_idx, dtype=np.uint64)[:, None]
    c = np.arange(cols, dtype=np.uint64)[None, :]
    ctr = r * np.uint64(cols) + c
    val = uniform_mod_p(splitmix64(seed, ctr), p)
    keep = splitmix64(seed ^ SPARSE_MASK_TWEAK, ctr) < np.uint64(SPARSE_THRESHOLD)
    return np.where(keep, val, np.uint32(0)).astype(np.uint32)


def sparse_dependent_plan(rows: int, p: int, seed_dep: int, period: int = 50, terms: int = 3):
    """For every dependent row i (i % period == period-1): source rows s_t and weights alpha_t.

    Sources are drawn among the independent rows (s % period != period-1), weights in [1, p).
    Returns (dep_rows int64[nd], src int64[nd, terms], alpha uint32[nd, terms]).
    """
    dep = np.arange(period - 1, rows, period, dtype=np.int64)
    n_indep = rows - dep.size
    k = np.arange(dep.size * terms, dtype=np.uint64)
    # rank among independent rows -> row index (skip every period-th row)
    rank = uniform_mod_p(splitmix64(seed_dep, np.uint64(2) * k), n_indep).astype(np.int64)
    src = rank + rank // (period - 1)
    alpha = uniform_mod_p(splitmix64(seed_dep, np.uint64(2) * k + np.uint64(1)), p - 1).astype(np.int64) + 1
    return dep, src.reshape(-1, terms), alpha.reshape(-1, terms).astype(np.uint32)


def sparse_dependent_rows(row0: int, nrows: int, rows: int, cols: int, p: int, seed: int,
                          seed_dep: int, period: int = 50, terms: int = 3) -> np.ndarray:
    """Config c5 (any size): rows [row0, row0+nrows) of the 90%-sparse rank-deficient matrix.

    Independent rows are `_sparse_base_rows`; every period-th row (i % period == period-1) is
    sum_t alpha_t * base_row(s_t) mod p, so the rank is at most rows - rows//period.
    """
    idx = np.arange(row0, row0 + nrows, dtype=np.int64)
    out = _sparse_base_rows(idx, cols, p, seed)
    is_dep = (idx % period) == (period - 1)
    if is_dep.any():
        _, src, alpha = sparse_dependent_plan(rows, p, seed_dep, period, terms)
        for local in np.nonzero(is_dep)[0]:
            d = int(idx[local]) // period
            acc = np.zeros(cols, dtype=np.uint64)
            base = _sparse_base_rows(src[d], cols, p, seed).astype(np.uint64)
            for t in range(terms):
                acc = (acc + base[t] * np.uint64(int(alpha[d, t])) % np.uint64(p)) % np.uint64(p)
            out[local] = acc.astype(np.uint32)
    return out


def normal_matrix(rows: int, cols: int, seed: int, chunk_rows: int = 1024) -> np.ndarray:
    """i.i.d. N(0,1) float64 by Box-Muller on two counter draws per element (host only)."""
    out = np.empty((rows, cols), dtype=np.float64)
    two53 = float(1 << 53)
    for r0 in range(0, rows, chunk_rows):
        n = min(chunk_rows, rows - r0)
        ctr = _row_counters(r0, n, cols)
        h1 = splitmix64(seed, np.uint64(2) * ctr)
        h2 = splitmix64(seed, np.uint64(2) * ctr + np.uint64(1))
        u1 = ((h1 >> np.uint64(11)).astype(np.float64) + 1.0) / two53      # (0, 1]
        u2 = (h2 >> np.uint64(11)).astype(np.float64) / two53              # [0, 1)
        out[r0:r0 + n] = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return out


def shifted_normal_system(n: int, nrhs: int, seed_a: int, seed_b: int):
    """Config c4: A = G + 4*sqrt(n)*I with G i.i.d. N(0,1); B n x nrhs N(0,1)."""
    a = normal_matrix(n, n, seed_a)
    a[np.arange(n), np.arange(n)] += 4.0 * np.sqrt(float(n))
    b = normal_matrix(n, nrhs, seed_b)
    return a, b
