"""Pins for the fp64 oracle (row-scaled partial-pivot Gauss-Jordan solve + backward error)."""
import numpy as np
import pytest

import linac_inputs as gen


def eta_numpy(a, x, b):
    """The acceptance metric written again with numpy (inf-norms), independent of the C routine."""
    x2 = x.reshape(len(x), -1)
    b2 = b.reshape(len(b), -1)
    na = np.abs(a).sum(axis=1).max()
    res = np.abs(a @ x2 - b2).max(axis=0)
    return float((res / (na * np.abs(x2).max(axis=0) + np.abs(b2).max(axis=0))).max())


@pytest.mark.parametrize("n,nrhs", [(1, 1), (2, 3), (17, 4), (64, 8), (200, 5)])
def test_solve_vs_lapack(oracle, n, nrhs):
    a, b = gen.shifted_normal_system(n, nrhs, seed_a=5, seed_b=6)
    rc, info, x = oracle.solve_f64(a, b)
    assert rc == 0 and info == 0
    ref = np.linalg.solve(a, b)
    assert np.allclose(x, ref, rtol=1e-12, atol=1e-13)
    assert oracle.backward_error(a, x, b) <= 1e-14
    assert abs(oracle.backward_error(a, x, b) - eta_numpy(a, x, b)) <= 1e-15   # fp64 vs long-double residual noise
    rc2, _, x2 = oracle.solve_f64(a, b, nthreads=4)
    assert rc2 == 0 and np.array_equal(x, x2)


def test_manufactured_solution_and_exact_cases(oracle):
    n = 50
    a, _ = gen.shifted_normal_system(n, 1, seed_a=9, seed_b=10)
    ones = np.ones((n, 1))
    rc, _, x = oracle.solve_f64(a, a @ ones)
    assert rc == 0 and np.allclose(x, ones, rtol=1e-12)
    # identity and diagonal systems are exact
    b = gen.normal_matrix(n, 3, seed=3)
    rc, _, x = oracle.solve_f64(np.eye(n), b)
    assert rc == 0 and np.array_equal(x, b)
    d = np.diag(2.0 ** np.arange(-5, n - 5, dtype=np.float64))
    rc, _, x = oracle.solve_f64(d, b)
    assert rc == 0 and np.array_equal(x, b / np.diag(d)[:, None])


def test_pivoting_is_needed_and_done(oracle):
    """Tiny leading entry: without row exchange the answer is garbage; with it, exact to rounding."""
    a = np.array([[1e-20, 1.0], [1.0, 1.0]])
    b = np.array([[1.0], [2.0]])
    rc, _, x = oracle.solve_f64(a, b)
    assert rc == 0 and np.allclose(x, np.linalg.solve(a, b), rtol=1e-15)
    # badly row-scaled system: equilibration keeps the pivot choice sane
    a = np.array([[1.0, 1e18], [1.0, 1.0]])
    b = np.array([[1e18], [2.0]])
    rc, _, x = oracle.solve_f64(a, b)
    assert rc == 0 and oracle.backward_error(a, x, b) < 1e-15


def test_singular_detection(oracle):
    n = 12
    a, b = gen.shifted_normal_system(n, 2, seed_a=1, seed_b=2)
    a[7] = a[2]                                    # duplicate row -> exactly singular
    rc, info, x = oracle.solve_f64(a, b)
    assert rc == 1 and 1 <= info <= n and x is None
    z = np.zeros((3, 3)); z[0, 0] = 1.0            # a zero row -> singular at the scaling step
    rc, info, _ = oracle.solve_f64(z, np.ones((3, 1)))
    assert rc == 1 and info >= 1
    # a tolerance the caller controls: eps-perturbed duplicate is singular under tol=1e-6
    a, b = gen.shifted_normal_system(n, 2, seed_a=1, seed_b=2)
    a[7] = a[2] * (1 + 1e-9)
    assert oracle.solve_f64(a, b, tol=1e-6)[0] == 1
    assert oracle.solve_f64(a, b, tol=0.0)[0] == 0


def test_backward_error_definition(oracle):
    rng = np.random.default_rng(3)
    a = rng.standard_normal((30, 30)); x = rng.standard_normal((30, 4)); b = a @ x
    assert oracle.backward_error(a, x, b) < 1e-15
    b2 = b.copy(); b2[3, 1] += 1.0                 # known residual in one column
    expect = 1.0 / (np.abs(a).sum(axis=1).max() * np.abs(x[:, 1]).max() + np.abs(b2[:, 1]).max())
    assert abs(oracle.backward_error(a, x, b2) - expect) < 1e-12
    assert abs(oracle.backward_error(a, x, b2, nthreads=4) - expect) < 1e-12


# ---------------------------------------------------------------- floating-point RREF with a threshold (8(f) rank 3)
def _rref_exact(a_int):
    """Exact rational RREF with sympy (independent black box); returns (float matrix, pivots)."""
    import sympy
    m, piv = sympy.Matrix(a_int.tolist()).rref()
    return np.array(m.tolist(), dtype=np.float64), list(piv)


def test_rref_f64_vs_exact_rational(oracle):
    pytest.importorskip("sympy")
    rng = np.random.default_rng(41)
    for rows, cols, r in [(5, 7, 3), (7, 5, 4), (6, 6, 6), (6, 6, 2), (4, 9, 4), (8, 3, 2)]:
        b = rng.integers(-4, 5, size=(rows, r))
        c = rng.integers(-4, 5, size=(r, cols))
        a = (b @ c).astype(np.int64)
        want, piv = _rref_exact(a)
        got, rank, gp = oracle.rref_f64(a.astype(np.float64), tol=1e-9)
        assert rank == len(piv) and list(gp) == piv
        assert np.allclose(got, want, rtol=0, atol=1e-11)
        assert not got[rank:].any()                                 # flushed zero rows (reading Q19)
        for k, c0 in enumerate(gp):                                 # exact structure: unit pivot columns, zeros on the left
            assert got[k, c0] == 1.0 and np.count_nonzero(got[:, c0]) == 1 and not got[k, :c0].any()
        got4, rank4, gp4 = oracle.rref_f64(a.astype(np.float64), tol=1e-9, nthreads=4)
        assert rank4 == rank and np.array_equal(got4, got)


def test_rref_f64_rank_vs_svd_and_rowspace(oracle):
    for rows, cols, r, seed in [(40, 60, 17, 1), (60, 40, 25, 2), (50, 50, 50, 3)]:
        a = gen.normal_matrix(rows, r, seed) @ gen.normal_matrix(r, cols, seed + 100)
        a *= (10.0 ** gen.normal_matrix(rows, 1, seed + 200))       # badly scaled rows: the rescaling step matters
        got, rank, piv = oracle.rref_f64(a, tol=1e-9)
        s = np.linalg.svd(a / np.abs(a).max(axis=1, keepdims=True), compute_uv=False)
        assert rank == int((s > 1e-9 * s[0]).sum()) == r
        # every row of A lies in the row space of R: a = a[pivots] . R (R is the identity on the pivot columns)
        recon = a[:, piv] @ got[:rank]
        assert np.abs(recon - a).max() <= 1e-9 * np.abs(a).max()
        # idempotence: reducing the result changes nothing beyond rounding
        again, rank2, piv2 = oracle.rref_f64(got, tol=1e-9)
        assert rank2 == rank and np.array_equal(piv2, piv) and np.allclose(again, got, rtol=0, atol=1e-10)


def test_rref_f64_inverse_and_threshold(oracle):
    n = 30
    a, _ = gen.shifted_normal_system(n, 1, seed_a=7, seed_b=8)
    got, rank, piv = oracle.rref_f64(np.hstack([a, np.eye(n)]))
    assert rank == n and list(piv) == list(range(n))
    # the row rescaling multiplies row r of (A | I) by 1/s_r; row operations never mix columns, so the
    # right block is A^-1 regardless
    assert np.allclose(got[:, n:], np.linalg.inv(a), rtol=1e-11, atol=1e-13)
    # threshold semantics: a planted pivot of 1e-12 is a pivot for tol = 1e-15, zero for tol = 1e-9
    m = np.array([[1.0, 2.0, 3.0], [0.0, 1e-12, 1.0], [0.0, 0.0, 1.0]])
    _, rank_lo, piv_lo = oracle.rref_f64(m, tol=1e-15)
    _, rank_hi, piv_hi = oracle.rref_f64(m, tol=1e-9)
    assert (rank_lo, list(piv_lo)) == (3, [0, 1, 2]) and (rank_hi, list(piv_hi)) == (2, [0, 2])
    # degenerate shapes
    z, rank0, _ = oracle.rref_f64(np.zeros((3, 4)))
    assert rank0 == 0 and not z.any()
    e, ranke, _ = oracle.rref_f64(np.zeros((0, 4)))
    assert ranke == 0 and e.shape == (0, 4)
