"""linac_solve_u32 against the oracle: the oracle reduces (A | b) one
right-hand side at a time, the library reduces all of them together -- consistency flags and particular solutions
(free variables zero) must agree exactly, and the in-place result must be the RREF of the augmented matrix."""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import require_cuda, from_device

pytestmark = pytest.mark.gpu
P31 = 2147483647
P29 = 2147483629


@pytest.fixture(autouse=True, scope="module")
def _cuda():
    require_cuda()


def run(oracle, a, b, p):
    import paper_2605_25863_b200 as L
    cols = a.shape[1]
    m = np.ascontiguousarray(np.hstack([a, b]))
    d = torch.from_numpy(m.view(np.int32)).cuda()
    rank_a, piv, cons, x = L.solve_u32(d, cols, p)
    cons_ref, x_ref = oracle.solve_modp(a, b, p, nthreads=oracle.max_threads())
    assert np.array_equal(cons.numpy(), cons_ref)
    assert np.array_equal(from_device(x), x_ref)
    r_ref, rank_ref, piv_ref = oracle.rref_modp(m, p, nthreads=oracle.max_threads())
    assert np.array_equal(from_device(d), r_ref)                       # in place: the RREF of (A | B)
    assert rank_a == int((piv_ref < cols).sum())
    return cons_ref, x_ref


def test_square_full_rank_reads_the_solution_off_the_last_columns(oracle):
    n, nrhs = 300, 5
    a = gen.uniform_matrix(n, n, P31, seed=41)
    y = gen.uniform_matrix(n, nrhs, P31, seed=42)
    b = oracle.matmul_modp(a, y, P31, nthreads=oracle.max_threads())
    cons, x = run(oracle, a, b, P31)
    assert cons.all() and np.array_equal(x, y)                         # eq. 12: (I | x)


@pytest.mark.parametrize("shape", [(200, 260), (260, 200), (150, 150)])
def test_rank_deficient_mixed_consistency(oracle, shape):
    m_, n_ = shape
    a, _, _ = gen.lowrank_factors(m_, min(m_, n_) // 2, n_, P29, seed_b=43, seed_c=44)
    y = gen.uniform_matrix(n_, 3, P29, seed=45)
    good = oracle.matmul_modp(a, y, P29, nthreads=oracle.max_threads())
    bad = gen.uniform_matrix(m_, 2, P29, seed=46)                      # random: outside the column space w.h.p.
    # b3 = bad0 + A.y: not a pivot column of the joint reduction (it lies in span(A, bad0)) yet inconsistent with A alone
    tricky = ((bad[:, :1].astype(np.uint64) + good[:, :1]) % P29).astype(np.uint32)
    b = np.hstack([good[:, :1], bad[:, :1], good[:, 1:2], tricky, bad[:, 1:2], good[:, 2:3]])
    cons, x = run(oracle, a, b, P29)
    assert list(cons) == [True, False, True, False, False, True]
    assert np.array_equal(oracle.matmul_modp(a, x[:, [0, 2, 5]], P29), b[:, [0, 2, 5]])


def test_small_fields_and_degenerate_shapes(oracle):
    rng = np.random.default_rng(47)
    for p, m_, n_, k in [(2, 40, 30, 4), (3, 25, 60, 3), (7, 1, 5, 2), (7, 5, 1, 2), (5, 33, 33, 1)]:
        a = rng.integers(0, p, size=(m_, n_)).astype(np.uint32)
        b = rng.integers(0, p, size=(m_, k)).astype(np.uint32)
        run(oracle, a, b, p)
    # zero matrix: only the zero right-hand side is consistent
    a = np.zeros((20, 10), dtype=np.uint32)
    b = np.zeros((20, 2), dtype=np.uint32)
    b[3, 1] = 5
    cons, x = run(oracle, a, b, P31)
    assert list(cons) == [True, False] and not x.any()


def test_no_right_hand_sides_and_no_unknowns(oracle):
    import paper_2605_25863_b200 as L
    a = gen.uniform_matrix(50, 40, P31, seed=48)
    d = torch.from_numpy(a.view(np.int32)).cuda()
    rank_a, piv, cons, x = L.solve_u32(d, 40, P31)                     # nrhs = 0: plain RREF
    assert rank_a == 40 and cons.numel() == 0 and x.shape == (40, 0)
    b = gen.uniform_matrix(50, 3, P31, seed=49)
    d = torch.from_numpy(b.view(np.int32)).cuda()
    rank_a, piv, cons, x = L.solve_u32(d, 0, P31)                      # cols = 0: consistent iff b = 0
    assert rank_a == 0 and not cons.any() and x.shape == (0, 3)
