"""Parity of linac_rref_f64 (floating-point row reduction with a threshold, PAPER.md:65,
231-251) against the CPU oracle, through the C ABI.

What is compared ("fp64 RREF tolerance"): rank and pivot columns exactly (the inputs keep a gap of many
orders of magnitude between the smallest true pivot and the threshold); the entries of R element by element within
1e-8 * max(1, max|R|) (both sides run Gauss-Jordan with partial pivoting, in different summation orders: the oracle
column by column, the GPU 32 pivots at a time through the inverse of the pivot block); the exact structure (unit pivot
columns, flushed zeros) bit for bit; and the reconstruction a = a[pivots] . R on the ORIGINAL rows to 1e-10."""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import require_cuda

pytestmark = pytest.mark.gpu
SENT = -7.25e300


@pytest.fixture(autouse=True, scope="module")
def _cuda():
    require_cuda()


def gpu_rref_f64(a, tol=-1.0, ld=None):
    import paper_2605_25863_b200 as L
    rows, cols = a.shape
    ld = cols if ld is None else ld
    buf = np.full((rows, ld), SENT, dtype=np.float64)
    buf[:, :cols] = a
    t = torch.from_numpy(buf).cuda()
    view = t[:, :cols] if cols else t
    rank, piv = L.rref_f64(view, tol)
    out = t.cpu().numpy()
    if ld > cols:
        assert (out[:, cols:] == SENT).all(), "padding columns were written"
    return out[:, :cols].copy(), rank, piv.numpy().copy()


def check(oracle, a, tol=1e-9, ld=None, recon_tol=1e-10):
    r_ref, rank_ref, piv_ref = oracle.rref_f64(a, tol=tol, nthreads=oracle.max_threads())
    r, rank, piv = gpu_rref_f64(a, tol, ld)
    assert rank == rank_ref and np.array_equal(piv, piv_ref)
    scale = max(1.0, float(np.abs(r_ref).max()) if r_ref.size else 1.0)
    assert np.abs(r - r_ref).max(initial=0.0) <= 1e-8 * scale
    # exact structure
    assert not r[rank:].any()
    for k, c0 in enumerate(piv):
        assert r[k, c0] == 1.0 and np.count_nonzero(r[:, c0]) == 1 and not r[k, :c0].any()
    # reconstruction on the original data: every row of a is a[pivots] . R
    if rank:
        recon = a[:, piv] @ r[:rank]
        assert np.abs(recon - a).max() <= recon_tol * max(1.0, np.abs(a).max()) * max(1.0, np.abs(r).max())
    else:
        assert np.abs(a).max(initial=0.0) <= tol * max(1.0, np.abs(a).max(initial=0.0))
    return r, rank, piv


@pytest.mark.parametrize("rows,cols,r", [(5, 7, 3), (7, 5, 4), (40, 40, 40), (33, 31, 20), (31, 33, 31), (64, 96, 64),
                                         (100, 257, 60), (257, 100, 100), (300, 400, 120), (130, 130, 1)])
def test_integer_lowrank_products(oracle, rows, cols, r):
    rng = np.random.default_rng(rows * 1000 + cols)
    a = (rng.integers(-4, 5, size=(rows, r)) @ rng.integers(-4, 5, size=(r, cols))).astype(np.float64)
    _, rank, _ = check(oracle, a)
    assert rank <= r


@pytest.mark.parametrize("rows,cols,r,seed", [(200, 300, 77, 1), (300, 200, 150, 2), (500, 500, 500, 3), (600, 800, 333, 4)])
def test_normal_lowrank_badly_scaled_rows(oracle, rows, cols, r, seed):
    a = gen.normal_matrix(rows, r, seed) @ gen.normal_matrix(r, cols, seed + 100)
    a *= 10.0 ** (3.0 * gen.normal_matrix(rows, 1, seed + 200))          # row scales over ~12 decades
    _, rank, _ = check(oracle, a)
    assert rank == r


def test_full_rank_square_is_identity_and_inverse(oracle):
    n = 200
    a, _ = gen.shifted_normal_system(n, 1, seed_a=7, seed_b=8)
    r, rank, piv = gpu_rref_f64(a)
    assert rank == n and np.array_equal(r, np.eye(n))
    aug = np.hstack([a, np.eye(n)])
    r, rank, piv = check(oracle, aug, tol=-1.0)
    assert rank == n and np.allclose(r[:, n:], np.linalg.inv(a), rtol=1e-10, atol=1e-12)


def test_free_columns_in_the_middle_and_pivots_far_down(oracle):
    a = gen.normal_matrix(300, 260, 9)
    a[:, 5] = 0
    a[:, 40:75] = 0
    a[:, 130] = a[:, 3]
    a[:, 131] = 5.0 * a[:, 4] - a[:, 6]
    a[:150, :60] = 0
    a[10:20, :] = 0
    check(oracle, a)


def test_threshold_semantics_and_degenerate_shapes(oracle):
    import paper_2605_25863_b200 as L
    m = np.array([[1.0, 2.0, 3.0], [0.0, 1e-12, 1.0], [0.0, 0.0, 1.0]])
    _, rank_lo, piv_lo = gpu_rref_f64(m, tol=1e-15)
    _, rank_hi, piv_hi = gpu_rref_f64(m, tol=1e-9)
    assert (rank_lo, list(piv_lo)) == (3, [0, 1, 2]) and (rank_hi, list(piv_hi)) == (2, [0, 2])
    z, rank0, _ = gpu_rref_f64(np.zeros((70, 90)))
    assert rank0 == 0 and not z.any()
    for shape in [(0, 5), (5, 0), (0, 0)]:
        t = torch.zeros(shape, dtype=torch.float64, device="cuda")
        rank, piv = L.rref_f64(t)
        assert rank == 0 and piv.numel() == 0
    check(oracle, np.array([[0.0, 0.0, 2.0]]))
    check(oracle, np.array([[0.0], [3.0], [0.0]]))


@pytest.mark.parametrize("shape,ld", [((50, 37), 41), ((129, 65), 67)])
def test_odd_leading_dimension(oracle, shape, ld):
    a = gen.normal_matrix(shape[0], 20, 5) @ gen.normal_matrix(20, shape[1], 6)
    check(oracle, a, ld=ld)


def test_tags_and_grid_barrier_agree(oracle):
    """The tagged-record panel (one 128-bit scalar operation per record) and the grid-barrier panel give the same bits."""
    import paper_2605_25863_b200 as L
    a = gen.normal_matrix(700, 60, 11) @ gen.normal_matrix(60, 500, 12)
    try:
        L.set_option("f64_panel_tags", 0)
        r0, rank0, piv0 = gpu_rref_f64(a, 1e-9)
    finally:
        L.set_option("f64_panel_tags", 1)
    for _ in range(3):
        r1, rank1, piv1 = gpu_rref_f64(a, 1e-9)
        assert rank1 == rank0 == 60 and np.array_equal(piv1, piv0) and np.array_equal(r1, r0)


def test_large_rank_deficient(oracle):
    """Many panels, several row tiles per CTA of the pivot search, K = 32 DMMA updates over a ragged shape."""
    a = gen.normal_matrix(2100, 700, 21) @ gen.normal_matrix(700, 2500, 22)
    _, rank, _ = check(oracle, a, recon_tol=1e-9)
    assert rank == 700


@pytest.mark.parametrize("strip", [32, 64, 96, 128])
def test_strip_widths_against_the_oracle(oracle, strip):
    """Strips of 32 (every panel updates everything), 64, 96 and 128 columns: the deferred K = strip update right of the
    strip, the catch-up product on the pivot rows and the exchanged rows of the L stack, on shapes with ragged last
    strips, free columns inside strips (rank-deficient products) and row exchanges in every panel."""
    import paper_2605_25863_b200 as L
    cases = [gen.normal_matrix(520, 130, 31) @ gen.normal_matrix(130, 777, 32),       # free columns from column ~130 on
             gen.normal_matrix(300, 300, 33),                                         # full rank: the RREF is the identity
             gen.normal_matrix(450, 449, 34) @ gen.normal_matrix(449, 600, 35)]       # nearly every column a pivot
    # free columns in the middle of strips: duplicate / zero some columns of a full-rank matrix
    b = gen.normal_matrix(400, 400, 36)
    b[:, 5::7] = 0.0
    b[:, 130:170] = b[:, 10:50] * 3.0
    cases.append(b)
    try:
        L.set_option("f64_rref_strip", strip)
        for a in cases:
            check(oracle, a, recon_tol=1e-9)
    finally:
        L.set_option("f64_rref_strip", 128)
