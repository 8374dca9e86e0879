"""Parity of linac_rref_c128 (complex128: PAPER.md:163) against the CPU oracle, through the C ABI.

The GPU reduces the real 2 x 2 block embedding of the matrix with the fp64 kernels; the oracle runs the
paper's loop in complex arithmetic with a largest-modulus pivot.  Compared as for linac_rref_f64: rank and pivot columns
exactly (the inputs keep many orders of magnitude between the smallest true pivot and the threshold), entries within
1e-8 * max(1, max|R|) (different pivot choices and summation orders on the same rescaled rows), the exact structure
(unit pivot columns, flushed zeros) bit for bit, and the reconstruction a = a[:, pivots] . R on the ORIGINAL rows."""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import require_cuda

pytestmark = pytest.mark.gpu
SENT = complex(-7.25e300, 3.5e300)


@pytest.fixture(autouse=True, scope="module")
def _cuda():
    require_cuda()


def complex_normal(rows, cols, seed):
    return gen.normal_matrix(rows, cols, seed=seed) + 1j * gen.normal_matrix(rows, cols, seed=seed + 1000)


def gpu_rref_c128(a, tol=-1.0, ld=None):
    import paper_2605_25863_b200 as L
    rows, cols = a.shape
    ld = cols if ld is None else ld
    buf = np.full((rows, ld), SENT, dtype=np.complex128)
    buf[:, :cols] = a
    t = torch.from_numpy(buf).cuda()
    view = t[:, :cols] if cols else t
    rank, piv = L.rref_c128(view, tol)
    out = t.cpu().numpy()
    if ld > cols:
        assert (out[:, cols:] == SENT).all(), "padding columns were written"
    return out[:, :cols].copy(), rank, piv.numpy().copy()


def check(oracle, a, tol=1e-9, ld=None, recon_tol=1e-10):
    r_ref, rank_ref, piv_ref = oracle.rref_c128(a, tol=tol, nthreads=oracle.max_threads())
    r, rank, piv = gpu_rref_c128(a, tol, ld)
    assert rank == rank_ref and np.array_equal(piv, piv_ref)
    scale = max(1.0, float(np.abs(r_ref).max()) if r_ref.size else 1.0)
    assert np.abs(r - r_ref).max(initial=0.0) <= 1e-8 * scale
    assert not r[rank:].any()
    for k, c0 in enumerate(piv):
        assert r[k, c0] == 1.0 and np.count_nonzero(r[:, c0]) == 1 and not r[k, :c0].any()
    if rank:
        recon = a[:, piv] @ r[:rank]
        assert np.abs(recon - a).max() <= recon_tol * max(1.0, np.abs(a).max()) * max(1.0, np.abs(r).max())
    return r, rank, piv


@pytest.mark.parametrize("rows,cols,r", [(1, 1, 1), (5, 7, 3), (7, 5, 4), (33, 31, 20), (31, 33, 31), (64, 96, 64),
                                         (100, 257, 60), (257, 100, 100), (130, 130, 1)])
def test_gaussian_integer_lowrank_products(oracle, rows, cols, r):
    rng = np.random.default_rng(rows * 1000 + cols)
    b = rng.integers(-4, 5, size=(rows, r)) + 1j * rng.integers(-4, 5, size=(rows, r))
    c = rng.integers(-4, 5, size=(r, cols)) + 1j * rng.integers(-4, 5, size=(r, cols))
    _, rank, _ = check(oracle, (b @ c).astype(np.complex128))
    assert rank <= r


@pytest.mark.parametrize("rows,cols,r,seed", [(200, 300, 77, 1), (300, 200, 150, 2), (400, 400, 400, 3), (500, 700, 333, 4)])
def test_normal_lowrank_badly_scaled_rows_and_phases(oracle, rows, cols, r, seed):
    a = complex_normal(rows, r, seed) @ complex_normal(r, cols, seed + 100)
    a *= 10.0 ** (3.0 * gen.normal_matrix(rows, 1, seed + 200))                 # row scales over ~12 decades
    a *= np.exp(2j * np.pi * gen.normal_matrix(rows, 1, seed + 300))            # and arbitrary row phases
    _, rank, _ = check(oracle, a)
    assert rank == r


def test_full_rank_square_is_identity_and_inverse(oracle):
    n = 150
    a = complex_normal(n, n, 7) + 4 * np.sqrt(n) * np.eye(n)
    r, rank, piv = gpu_rref_c128(a)
    assert rank == n and np.array_equal(r, np.eye(n))
    r, rank, piv = gpu_rref_c128(np.hstack([a, np.eye(n)]))
    assert rank == n and np.array_equal(piv, np.arange(n))
    assert np.allclose(r[:, n:], np.linalg.inv(a), rtol=1e-10, atol=1e-12)


def test_padded_rows_real_input_and_degenerate_shapes(oracle):
    a = complex_normal(70, 30, 11) @ complex_normal(30, 90, 12)
    check(oracle, a, ld=97)
    # a real matrix through the complex entry point reduces like linac_rref_f64's oracle
    b = gen.normal_matrix(50, 20, seed=13) @ gen.normal_matrix(20, 60, seed=14)
    r, rank, piv = gpu_rref_c128(b.astype(np.complex128), 1e-9)
    r_re, rank_re, piv_re = oracle.rref_f64(b, tol=1e-9)
    assert rank == rank_re and np.array_equal(piv, piv_re)
    assert np.abs(r.imag).max() <= 1e-9 and np.abs(r.real - r_re).max() <= 1e-8 * max(1.0, np.abs(r_re).max())
    # all-zero and empty inputs
    z, rank, piv = gpu_rref_c128(np.zeros((9, 5), dtype=np.complex128))
    assert rank == 0 and not z.any()
    import paper_2605_25863_b200 as L
    assert L.rref_c128(torch.zeros((0, 6), dtype=torch.complex128, device="cuda"))[0] == 0


def test_threshold_semantics(oracle):
    d = np.diag([1.0, 1e-12 * np.exp(0.7j), 1.0]).astype(np.complex128)
    d[1, 2] = 1.0                                   # the row's scale: the planted entry stays 1e-12 after rescaling
    assert gpu_rref_c128(d, 1e-10)[1] == 2 == oracle.rref_c128(d, tol=1e-10)[1]
    assert gpu_rref_c128(d, 1e-14)[1] == 3 == oracle.rref_c128(d, tol=1e-14)[1]
