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
