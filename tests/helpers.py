"""Test-side reference helpers written independently of oracle/ and of the CUDA path.

Everything here is brute force or a definition (Python big ints, itertools), used to PIN the
oracle, never to generate expected values for the CUDA path.
"""
from __future__ import annotations

import itertools

import numpy as np


def is_rref(r: np.ndarray, p: int):
    """The four defining properties of a reduced row-echelon form; returns pivots or None."""
    rows, cols = r.shape
    if r.size and int(r.max()) >= p:
        return None
    pivots = []
    seen_zero_row = False
    last = -1
    for i in range(rows):
        nz = np.nonzero(r[i])[0]
        if nz.size == 0:
            seen_zero_row = True
            continue
        if seen_zero_row:                 # (1) non-zero rows precede zero rows
            return None
        c = int(nz[0])
        if r[i, c] != 1:                  # (2) pivot is 1
            return None
        if c <= last:                     # (3) pivot columns strictly increase
            return None
        if np.count_nonzero(r[:, c]) != 1:  # (4) pivot is the only non-zero in its column
            return None
        pivots.append(c)
        last = c
    return pivots


def row_space_set(a: np.ndarray, p: int) -> set:
    """All p^rows linear combinations of the rows of a (tiny fields only)."""
    rows, cols = a.shape
    out = set()
    aa = [[int(x) for x in row] for row in a]
    for coeffs in itertools.product(range(p), repeat=rows):
        v = tuple(sum(c * aa[i][j] for i, c in enumerate(coeffs)) % p for j in range(cols))
        out.add(v)
    return out


def kernel_count(a: np.ndarray, p: int) -> int:
    """#{x in F_p^cols : a x = 0} by enumeration."""
    rows, cols = a.shape
    aa = [[int(x) for x in row] for row in a]
    n = 0
    for x in itertools.product(range(p), repeat=cols):
        if all(sum(aa[i][j] * x[j] for j in range(cols)) % p == 0 for i in range(rows)):
            n += 1
    return n


def det_leibniz(a: np.ndarray, p: int) -> int:
    n = a.shape[0]
    aa = [[int(x) for x in row] for row in a]
    total = 0
    for perm in itertools.permutations(range(n)):
        inv = sum(1 for i in range(n) for j in range(i + 1, n) if perm[i] > perm[j])
        term = 1
        for i in range(n):
            term = term * aa[i][perm[i]] % p
        total += -term if inv & 1 else term
    return total % p


def matmul_big(a: np.ndarray, b: np.ndarray, p: int) -> np.ndarray:
    """Exact (a @ b) mod p through Python ints (object dtype)."""
    return ((a.astype(object) @ b.astype(object)) % p).astype(np.uint32)


def random_row_ops(a: np.ndarray, p: int, rng: np.random.Generator, nops: int = 40) -> np.ndarray:
    """G.a for G a random product of row swaps, non-zero scalings and row additions (Python ints)."""
    m = [[int(x) for x in row] for row in a]
    rows = len(m)
    if rows < 2:
        return a.copy()
    for _ in range(nops):
        op = rng.integers(3)
        i, j = (int(x) for x in rng.choice(rows, size=2, replace=False))
        if op == 0:
            m[i], m[j] = m[j], m[i]
        elif op == 1:
            s = int(rng.integers(1, p))
            m[i] = [x * s % p for x in m[i]]
        else:
            s = int(rng.integers(0, p))
            m[i] = [(x + s * y) % p for x, y in zip(m[i], m[j])]
    return np.array(m, dtype=np.uint32)
