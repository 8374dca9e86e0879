"""Pins for the complex128 row reduction of the oracle (`oracle.rref_c128`).

Nothing here re-types the oracle's loop: the expected values come from sympy's exact arithmetic over Q(i), from the
oracle's REAL reduction applied to the 2 x 2 block embedding (a different routine on a different matrix), from numpy's
SVD / LAPACK, and from invariants of the reduced echelon form.
"""
import numpy as np
import pytest
import sympy

import linac_inputs as gen


def embed(a: np.ndarray) -> np.ndarray:
    """z = x + iy -> [[x, -y], [y, x]]: a ring homomorphism, so RREF(embed(A)) = embed(RREF(A)) by uniqueness."""
    rows, cols = a.shape
    e = np.empty((2 * rows, 2 * cols))
    e[0::2, 0::2] = a.real
    e[0::2, 1::2] = -a.imag
    e[1::2, 0::2] = a.imag
    e[1::2, 1::2] = a.real
    return e


def complex_normal(rows, cols, seed):
    return gen.normal_matrix(rows, cols, seed=seed) + 1j * gen.normal_matrix(rows, cols, seed=seed + 1000)


def test_vs_exact_rref_over_gaussian_rationals(oracle):
    rng = np.random.default_rng(11)
    for rows, cols, rk in [(3, 4, 2), (5, 5, 5), (6, 8, 4), (7, 5, 3)]:
        b = rng.integers(-3, 4, size=(rows, rk)) + 1j * rng.integers(-3, 4, size=(rows, rk))
        c = rng.integers(-3, 4, size=(rk, cols)) + 1j * rng.integers(-3, 4, size=(rk, cols))
        a = b @ c
        m = sympy.Matrix(rows, cols, lambda i, j: sympy.Integer(int(a[i, j].real)) + sympy.I * sympy.Integer(int(a[i, j].imag)))
        ref, piv_ref = m.rref()
        ref = np.array(ref.applyfunc(sympy.nsimplify).evalf(30).tolist(), dtype=np.complex128)
        r, rank, piv = oracle.rref_c128(a, tol=1e-9)
        assert rank == len(piv_ref) and list(piv) == list(piv_ref)
        assert np.allclose(r, ref, rtol=0, atol=1e-11)


def test_real_input_reduces_like_the_real_oracle(oracle):
    a = gen.normal_matrix(9, 6, seed=21) @ gen.normal_matrix(6, 13, seed=22)
    r_re, rank_re, piv_re = oracle.rref_f64(a, tol=1e-10)
    r, rank, piv = oracle.rref_c128(a.astype(np.complex128), tol=1e-10)
    assert rank == rank_re == 6 and np.array_equal(piv, piv_re)
    assert np.abs(r.imag).max() == 0.0
    assert np.allclose(r.real, r_re, rtol=0, atol=1e-12)


@pytest.mark.parametrize("rows,inner,cols", [(8, 8, 8), (10, 4, 14), (12, 7, 9)])
def test_block_embedding_commutes_with_the_reduction(oracle, rows, inner, cols):
    a = complex_normal(rows, inner, 31) @ complex_normal(inner, cols, 33)
    a *= (10.0 ** (2 * gen.normal_matrix(rows, 1, seed=35)))          # badly scaled rows: the rescaling must cope
    r, rank, piv = oracle.rref_c128(a, tol=1e-9)
    re, rank_e, piv_e = oracle.rref_f64(embed(a), tol=1e-9)
    assert rank == min(rows, inner, cols) and rank_e == 2 * rank
    assert np.array_equal(piv_e[0::2], 2 * piv) and np.array_equal(piv_e[1::2], 2 * piv + 1)
    assert np.allclose(embed(r), re, rtol=0, atol=1e-9 * max(1.0, np.abs(re).max()))


def test_rank_vs_svd_rowspace_and_structure(oracle):
    rows, inner, cols = 40, 17, 55
    a = complex_normal(rows, inner, 41) @ complex_normal(inner, cols, 43)
    r, rank, piv = oracle.rref_c128(a, tol=1e-9)
    assert rank == inner == int((np.linalg.svd(a, compute_uv=False) > 1e-9).sum())
    assert np.array_equal(r[:rank][:, piv], np.eye(rank))                      # exact unit pivot columns
    assert not r[rank:].any()
    for t in range(rank):
        assert not r[t, :piv[t]].any()
    assert np.allclose(a[:, piv] @ r[:rank], a, rtol=0, atol=1e-9 * np.abs(a).max())     # every row of A lies in the row space


def test_row_phases_and_row_operations_do_not_change_the_result(oracle):
    a = complex_normal(7, 4, 51) @ complex_normal(4, 9, 53)
    r0, rank0, piv0 = oracle.rref_c128(a, tol=1e-10)
    phases = np.exp(2j * np.pi * np.linspace(0.1, 0.9, 7))[:, None]
    mix = complex_normal(7, 7, 55)                                                # invertible with probability one
    for b in (phases * a, mix @ a, a[::-1]):
        r, rank, piv = oracle.rref_c128(b, tol=1e-10)
        assert rank == rank0 and np.array_equal(piv, piv0)
        assert np.allclose(r, r0, rtol=0, atol=1e-9)


def test_inverse_and_threshold(oracle):
    n = 12
    a = complex_normal(n, n, 61) + 4 * np.eye(n)
    r, rank, piv = oracle.rref_c128(np.hstack([a, np.eye(n)]), tol=1e-12)
    assert rank == n and np.array_equal(piv, np.arange(n))
    assert np.allclose(r[:, n:], np.linalg.inv(a), rtol=1e-11, atol=1e-12)
    # a planted pivot of modulus 1e-12 on both sides of the threshold
    d = np.diag([1.0, 1e-12 * np.exp(0.7j), 1.0]).astype(np.complex128)
    d[1, 2] = 1.0                                                                 # the row's scale: the planted entry stays 1e-12
    assert oracle.rref_c128(d, tol=1e-10)[1] == 2
    assert oracle.rref_c128(d, tol=1e-14)[1] == 3
    # degenerate shapes
    assert oracle.rref_c128(np.zeros((3, 4), dtype=np.complex128))[1] == 0
    assert oracle.rref_c128(np.zeros((0, 4), dtype=np.complex128))[1] == 0
