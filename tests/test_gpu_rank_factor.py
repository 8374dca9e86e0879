"""linac_rank_factor_u32 (eq. 7) against the oracle: C, R and the pivot
columns bit-exact, the input untouched, and C.R = A checked with the oracle's plain product."""
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


def run(oracle, a, p, ld=None):
    import paper_2605_25863_b200 as L
    rows, cols = a.shape
    ld = cols if ld is None else ld
    buf = np.full((rows, ld), 0xDEADBEEF, dtype=np.uint32)
    buf[:, :cols] = a
    d = torch.from_numpy(buf.view(np.int32)).cuda()
    view = d[:, :cols] if cols else d
    rank, piv, c, r = L.rank_factor_u32(view, p)
    assert np.array_equal(from_device(d), buf), "the input must be left untouched"
    c_ref, r_ref, piv_ref = oracle.rank_factor_modp(a, p, nthreads=oracle.max_threads())
    assert rank == len(piv_ref) and np.array_equal(piv.numpy(), piv_ref)
    assert np.array_equal(from_device(c).reshape(rows, rank), c_ref)
    assert np.array_equal(from_device(r).reshape(rank, cols), r_ref)
    return from_device(c).reshape(rows, rank), from_device(r).reshape(rank, cols)


@pytest.mark.parametrize("shape,k", [((300, 420), 77), ((420, 300), 131), ((513, 513), 512), ((64, 1000), 64),
                                     ((1000, 64), 33)])
def test_low_rank_products(oracle, shape, k):
    a, _, _ = gen.lowrank_factors(shape[0], k, shape[1], P29, seed_b=shape[0], seed_c=shape[1])
    c, r = run(oracle, a, P29)
    assert c.shape[1] == k
    assert np.array_equal(oracle.matmul_modp(c, r, P29, nthreads=oracle.max_threads()), a)


def test_full_rank_square_gives_c_equal_a_and_r_identity(oracle):
    a = gen.uniform_matrix(700, 700, P31, seed=3)
    c, r = run(oracle, a, P31)
    assert np.array_equal(c, a) and np.array_equal(r, np.eye(700, dtype=np.uint32))


def test_sparse_dependent_rows_and_padded_rows(oracle):
    cfg = gen.CONFIGS["c5"]
    a = gen.sparse_dependent_rows(0, 900, 900, 1100, cfg["p"], cfg["seed"], cfg["seed_dep"])
    c, r = run(oracle, a, cfg["p"], ld=1104)
    assert c.shape[1] == 900 - 900 // cfg["period"]
    assert np.array_equal(oracle.matmul_modp(c, r, cfg["p"], nthreads=oracle.max_threads()), a)


def test_entries_ge_p_and_tiny_fields(oracle):
    rng = np.random.default_rng(4)
    for p in (2, 3, 5, 65521):
        a = rng.integers(0, 2**32, size=(150, 170), dtype=np.uint64).astype(np.uint32)
        c, r = run(oracle, a, p)
        assert np.array_equal(oracle.matmul_modp(c, r, p), a % np.uint32(p))


@pytest.mark.parametrize("shape", [(0, 0), (0, 5), (5, 0), (1, 1), (1, 9), (9, 1)])
def test_degenerate_shapes(oracle, shape):
    a = gen.uniform_matrix(shape[0], shape[1], P31, seed=9) if shape[0] and shape[1] else np.zeros(shape, dtype=np.uint32)
    run(oracle, a, P31)


def test_zero_matrix(oracle):
    c, r = run(oracle, np.zeros((40, 50), dtype=np.uint32), P31)
    assert c.shape == (40, 0) and r.shape == (0, 50)
