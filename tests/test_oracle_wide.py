"""Pins for the wide-modulus oracle paths: oracle_rref_modp with
2^31 <= p < 2^32 and the 64-bit backend oracle_rref_modp64 / inv_modp64 / matmul_modp64.

As in test_oracle_modp.py every check is something other than the oracle: Python big-int arithmetic, brute
force over a tiny field, sympy's GF(p) RREF as a black box, closed forms.
"""
import itertools

import numpy as np
import pytest

import helpers as H
import linac_inputs as gen

P32 = 4294967291          # 2^32 - 5, the largest 32-bit prime
P32B = 2147483659         # the first prime above 2^31
P61 = (1 << 61) - 1       # Mersenne prime
P63 = 9223372036854775783 # 2^63 - 25, the largest prime below 2^63
P40 = 1099511627791       # a prime just above 2^40


def is_rref_big(r, p):
    """helpers.is_rref for object/uint64 matrices (the four defining properties)."""
    rows, cols = r.shape
    last, seen_zero = -1, False
    piv = []
    for i in range(rows):
        nz = [c for c in range(cols) if int(r[i, c]) != 0]
        if not nz:
            seen_zero = True
            continue
        if seen_zero or int(r[i, nz[0]]) != 1 or nz[0] <= last:
            return None
        if sum(1 for k in range(rows) if int(r[k, nz[0]]) != 0) != 1:
            return None
        if any(int(x) >= p for x in r[i]):
            return None
        piv.append(nz[0])
        last = nz[0]
    return piv


def rowspace_contains(r, rank, piv, a, p):
    """Every row of a equals a[pivots] . R (R is the identity on its pivot columns): Python ints."""
    rr = [[int(x) for x in row] for row in r[:rank]]
    for row in a:
        row = [int(x) % p for x in row]
        comb = [sum(row[piv[k]] * rr[k][c] for k in range(rank)) % p for c in range(len(row))]
        if comb != row:
            return False
    return True


@pytest.mark.parametrize("p", [P32, P32B, P40, P61, P63])
def test_inverse64_vs_python(oracle, p):
    rng = np.random.default_rng(5)
    for a in [1, 2, p - 1, p - 2, (p + 1) // 2] + [int(x) % p or 1 for x in rng.integers(1, 2**63 - 1, size=3000)]:
        inv = oracle.inv_modp64(a, p)
        assert 0 < inv < p and inv == pow(a, -1, p)


def test_matmul64_vs_bigint(oracle):
    rng = np.random.default_rng(6)
    for p in [7, P32, P61, P63]:
        a = (rng.integers(0, 2**63 - 1, size=(7, 11), dtype=np.uint64) % np.uint64(p)).astype(np.uint64)
        b = (rng.integers(0, 2**63 - 1, size=(11, 4), dtype=np.uint64) % np.uint64(p)).astype(np.uint64)
        want = (a.astype(object) @ b.astype(object)) % p
        assert np.array_equal(oracle.matmul_modp64(a, b, p).astype(object), want)
    a = np.full((2, 50), P63 - 1, dtype=np.uint64)          # worst-case operands
    b = np.full((50, 3), P63 - 1, dtype=np.uint64)
    assert np.array_equal(oracle.matmul_modp64(a, b, P63).astype(object), (a.astype(object) @ b.astype(object)) % P63)


@pytest.mark.parametrize("p", [P32, P32B])
def test_rref32_wide_p_structure_rowspace_and_64bit_agreement(oracle, p):
    """oracle_rref_modp with p >= 2^31: RREF structure, row-space containment with Python ints, rank of a
    product, and byte agreement with the independent 64-bit routine on the same data."""
    for shape, seed in [((9, 13), 1), ((13, 9), 2), ((12, 12), 3)]:
        a = gen.uniform_matrix(*shape, p, seed)
        a[0, 0] = p - 1; a[1, 1] = p - 1                   # worst-case operands somewhere
        r, rank, piv = oracle.rref_modp(a, p)
        assert rank == min(shape) and H.is_rref(r, p) == list(piv)
        assert rowspace_contains(r, rank, list(piv), a, p)
        r64, rank64, piv64 = oracle.rref_modp64(a.astype(np.uint64), p)
        assert rank64 == rank and np.array_equal(piv, piv64) and np.array_equal(r64, r.astype(np.uint64))
    b = gen.uniform_matrix(14, 5, p, 7)
    c = gen.uniform_matrix(5, 11, p, 8)
    a = ((b.astype(object) @ c.astype(object)) % p).astype(np.uint32)
    r, rank, piv = oracle.rref_modp(a, p)
    rc, rankc, pivc = oracle.rref_modp(c, p)
    assert rank == 5 and np.array_equal(r[:5], rc[:rankc]) and not r[5:].any()     # RREF(B.C) = RREF(C) padded


@pytest.mark.parametrize("p", [P40, P61, P63])
def test_rref64_structure_rowspace_product_rank(oracle, p):
    for shape, seed in [((8, 12), 1), ((12, 8), 2), ((10, 10), 3)]:
        a = gen.uniform_matrix_u64(*shape, p, seed)
        a[0, 0] = p - 1
        r, rank, piv = oracle.rref_modp64(a, p)
        assert rank == min(shape) and is_rref_big(r, p) == list(piv)
        assert rowspace_contains(r, rank, list(piv), a, p)
        for rule in (1, 2):                               # pivot-rule independence (uniqueness of the RREF)
            r2, rank2, piv2 = oracle.rref_modp64(a, p, pivot_rule=rule)
            assert rank2 == rank and np.array_equal(r2, r) and np.array_equal(piv2, piv)
        r3, _, _ = oracle.rref_modp64(a, p, nthreads=4)
        assert np.array_equal(r3, r)
    b = gen.uniform_matrix_u64(13, 4, p, 7)
    c = gen.uniform_matrix_u64(4, 10, p, 8)
    a = np.array((b.astype(object) @ c.astype(object)) % p, dtype=np.uint64)
    r, rank, piv = oracle.rref_modp64(a, p)
    rc, rankc, _ = oracle.rref_modp64(c, p)
    assert rank == 4 and np.array_equal(r[:4], rc[:rankc]) and not r[4:].any()


def test_rref64_small_field_agrees_with_bruteforce_and_32bit(oracle):
    """p small: the 64-bit loop against brute-force row spaces and against the pinned 32-bit oracle."""
    rng = np.random.default_rng(9)
    for p in [2, 3, 5]:
        for _ in range(6):
            rows, cols = int(rng.integers(1, 5)), int(rng.integers(1, 6))
            a = rng.integers(0, p, size=(rows, cols)).astype(np.uint64)
            r, rank, piv = oracle.rref_modp64(a, p)
            assert H.row_space_set(a.astype(np.uint32), p) == H.row_space_set(r.astype(np.uint32), p)
            assert H.is_rref(r.astype(np.uint32), p) == list(piv)
            r32, rank32, piv32 = oracle.rref_modp(a.astype(np.uint32), p)
            assert rank == rank32 and np.array_equal(r, r32.astype(np.uint64))


def test_rref64_vandermonde_interpolation(oracle):
    """(V | y) -> (I | coefficients) for y_i = q(x_i): a closed-form check of a non-trivial reduced block."""
    p = P61
    n = 9
    rng = np.random.default_rng(10)
    xs = [int(v) for v in rng.integers(1, 2**60, size=n)]
    coef = [int(v) for v in rng.integers(0, 2**60, size=n)]
    v = np.array([[pow(x, k, p) for k in range(n)] + [sum(c * pow(x, k, p) for k, c in enumerate(coef)) % p]
                  for x in xs], dtype=np.uint64)
    r, rank, piv = oracle.rref_modp64(v, p)
    assert rank == n and list(piv) == list(range(n))
    assert [int(r[k, n]) for k in range(n)] == [c % p for c in coef]


@pytest.mark.parametrize("p", [P32, P61])
def test_rref_wide_vs_sympy_blackbox(oracle, p):
    sympy = pytest.importorskip("sympy")
    from sympy.polys.domains import GF
    from sympy.polys.matrices import DomainMatrix
    a = gen.uniform_matrix_u64(7, 10, p, 21)
    a[3] = (a[0].astype(object) * 5 + a[1].astype(object) * 3) % p        # a dependent row
    dm = DomainMatrix([[GF(p)(int(x)) for x in row] for row in a], a.shape, GF(p))
    rr, pivs = dm.rref()
    want = np.array([[int(x) % p for x in row] for row in rr.to_list()], dtype=object)
    if p < 2**32:
        r, rank, piv = oracle.rref_modp(a.astype(np.uint32), p)
    else:
        r, rank, piv = oracle.rref_modp64(a, p)
    assert list(piv) == list(pivs) and rank == 6
    assert np.array_equal(r.astype(object), want)
