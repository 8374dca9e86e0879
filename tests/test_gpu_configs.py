"""BASELINE.json's configs at FULL size, in the launch configuration bench.py times (same binding call).

c1 is in test_gpu_fp.py.  Where the oracle cannot finish in seconds the check is a property that holds at any
size (identity RREF of a full-rank square matrix, A.x = b for the augmented system, A.K = 0 on sampled rows,
backward error on the original data)."""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import require_cuda, from_device

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True, scope="module")
def _cuda():
    require_cuda()


def matvec_mod_p(a: np.ndarray, x: np.ndarray, p: int) -> np.ndarray:
    """(a @ x) mod p with numpy uint64, written independently of oracle/ and of the CUDA path."""
    out = np.zeros(a.shape[0], dtype=np.uint64)
    xx = x.astype(np.uint64)
    for c0 in range(0, a.shape[1], 2048):
        blk = a[:, c0:c0 + 2048].astype(np.uint64) * xx[None, c0:c0 + 2048] % np.uint64(p)
        out = (out + blk.sum(axis=1) % np.uint64(p)) % np.uint64(p)
    return out


def test_config_c2_rank_3000_with_null_space(oracle):
    import paper_2605_25863_b200 as L
    c = gen.CONFIGS["c2"]
    p = c["p"]
    a, b, cc = gen.lowrank_factors(c["rows"], c["inner"], c["cols"], p, c["seed_b"], c["seed_c"])
    d = torch.from_numpy(a.view(np.int32)).cuda()
    rank, piv, k = L.nullspace_u32(d, p)
    r = from_device(d)
    kk = from_device(k)
    assert rank == c["inner"] and kk.shape == (c["cols"], c["cols"] - c["inner"])
    # full oracle comparison (threads only split independent rows; bit-identical to 1 thread)
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    assert rank == rank_ref and np.array_equal(piv.numpy(), piv_ref)
    assert np.array_equal(r, r_ref)
    assert np.array_equal(kk, oracle.nullspace_modp(r_ref, p, rank_ref, piv_ref))
    # A.K = 0 mod p (eq. 9) on sampled rows of the ORIGINAL A, plain triple loop
    rows = np.random.default_rng(0).choice(c["rows"], size=48, replace=False)
    assert not oracle.matmul_modp(a[rows], kk, p, nthreads=oracle.max_threads()).any()
    # and for every row, Freivalds style: A.(K.w) = 0
    w = gen.uniform_rows(0, 1, kk.shape[1], p, seed=99)[0]
    assert not matvec_mod_p(a, matvec_mod_p(kk, w, p).astype(np.uint32), p).any()


def test_config_c3_full_rank_10k_and_augmented_solve():
    import paper_2605_25863_b200 as L
    c = gen.CONFIGS["c3"]
    p, n = c["p"], c["rows"]
    a = gen.uniform_matrix(n, n, p, c["seed"])
    d = torch.from_numpy(a.view(np.int32)).cuda()
    rank, piv = L.rref_u32(d, p)
    assert rank == n and np.array_equal(piv.numpy(), np.arange(n))
    eye = torch.eye(n, dtype=torch.int32, device="cuda")
    assert torch.equal(d, eye)                                   # RREF of a full-rank square matrix is I
    del d, eye
    # same size, non-trivial output: (A | B) -> (I | X) with A.X = B mod p (eq. 12)
    nb = 8
    bmat = gen.uniform_matrix(n, nb, p, seed=77)
    aug = torch.from_numpy(np.hstack([a, bmat]).view(np.int32)).cuda()
    rank, piv = L.rref_u32(aug, p)
    assert rank == n
    x = from_device(aug[:, n:].contiguous())
    for q in range(nb):
        assert np.array_equal(matvec_mod_p(a, x[:, q], p), bmat[:, q].astype(np.uint64))


def test_config_c4_fp64_16384(oracle):
    import paper_2605_25863_b200 as L
    c = gen.CONFIGS["c4"]
    a, b = gen.shifted_normal_system(c["n"], c["nrhs"], c["seed_a"], c["seed_b"])
    da = torch.from_numpy(a).cuda()
    db = torch.from_numpy(b).cuda()
    L.solve_f64(da, db)
    x = db.cpu().numpy()
    del da, db
    eta = oracle.backward_error(a, x, b, nthreads=oracle.max_threads())
    assert eta <= 1e-11, eta
