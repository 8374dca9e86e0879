"""Parity cases the small-shape tests cannot reach (VERDICT r1 "Parity / untested configs"):

  * oracle BYTES on a rank-deficient matrix that spans about 40 strips with free columns spread over every strip
    (a flat-sweep or back-elimination bug that needs many strips with free columns would show here);
  * p = 2 and p = 3 at sizes that reach the flat sweep, the general (non-fast) panel path on every panel together
    with the tensor-core update, and the non-Montgomery tensor epilogue (p = 2);
  * a c3-scale NON-TRIVIAL output (10^4 x 11 000, rank-deficient), certified by properties that hold at any size:
    structure scan, Freivalds row-space containment A.v = A[:, piv].(R.v) for every row, A.K = 0 through A.(K.z).
"""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import gpu_rref, require_cuda, to_device_padded, from_device

pytestmark = pytest.mark.gpu
P31 = 2147483647
P29 = 2147483629


@pytest.fixture(autouse=True, scope="module")
def _cuda():
    require_cuda()


def test_forty_strips_with_free_columns_everywhere_oracle_bytes(oracle):
    p = P29
    rows, cols, r = 4608, 5248, 4000
    b = gen.uniform_matrix(rows, r, p, seed=21)
    c = gen.uniform_matrix(r, cols, p, seed=22)
    # every 7th column of C a combination of the two columns before it: free columns in every strip of A = B.C
    for j in range(6, cols, 7):
        c[:, j] = ((c[:, j - 1].astype(np.uint64) * 3 + c[:, j - 2].astype(np.uint64) * 5) % p).astype(np.uint32)
    a = np.empty((rows, cols), dtype=np.uint32)
    for r0 in range(0, rows, 512):
        a[r0:r0 + 512] = gen.gen._matmul_mod_p_exact(b[r0:r0 + 512], c, p)
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    out, rank, piv, st = gpu_rref(a, p)
    assert rank == rank_ref and np.array_equal(piv, piv_ref)
    assert np.array_equal(out, r_ref)
    assert rank < r + 1 and st["tc_launches"] > 30      # rank-deficient strips (K = 110 < 128) still take the tensor update


@pytest.mark.parametrize("p", [2, 3])
@pytest.mark.parametrize("shape", [(1200, 1200), (1000, 2000)])
def test_tiny_fields_at_flat_sweep_sizes(oracle, p, shape):
    import paper_2605_25863_b200 as L
    a = gen.uniform_matrix(shape[0], shape[1], p, seed=31 + p)
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    k_ref = oracle.nullspace_modp(r_ref, p, rank_ref, piv_ref)
    d = to_device_padded(a)
    rank, piv, k = L.nullspace_u32(d, p)
    st = L.last_stats()
    assert rank == rank_ref and np.array_equal(piv.numpy(), piv_ref)
    assert np.array_equal(from_device(d), r_ref)
    assert np.array_equal(from_device(k), k_ref)
    assert st["tc_launches"] > 0            # the tensor update ran (p = 2: the non-Montgomery epilogue)


@pytest.mark.parametrize("p", [2, 3])
def test_tensor_gemm_tiny_fields(oracle, p):
    import paper_2605_25863_b200 as L
    for m, n, k in [(1000, 900, 256), (640, 576, 700)]:
        a = gen.uniform_matrix(m, k, p, seed=1)
        b = gen.uniform_matrix(k, n, p, seed=2)
        c = gen.uniform_matrix(m, n, p, seed=3)
        dc, da, db = (torch.from_numpy(x.view(np.int32)).cuda() for x in (c, a, b))
        L.gemm_sub_u32(dc, da, db, p, 2)
        prod = oracle.matmul_modp(a, b, p, nthreads=oracle.max_threads())
        assert np.array_equal(from_device(dc), ((c.astype(np.int64) - prod.astype(np.int64)) % p).astype(np.uint32))


def _matvec(blk, x, p):
    return torch.stack([(blk * x[None, :, j] % p).sum(dim=1) % p for j in range(x.shape[1])], dim=1)


@pytest.mark.timeout(900)
def test_c3_scale_rank_deficient_wide_certificates(oracle):
    """10^4 x 11 000 over F_{2^31-1}: rows of c3's generator, every 40th row a combination of two others (rank 9750),
    1 000 extra columns -- a non-identity RREF at the paper's N = 10^4 size."""
    import paper_2605_25863_b200 as L
    p, rows, cols = P31, 10000, 11000
    dev = torch.device("cuda")
    a = gen.uniform_matrix(rows, cols, p, seed=4)
    dep = np.arange(39, rows, 40)
    a[dep] = ((a[dep - 1].astype(np.uint64) * 7 + a[dep - 2].astype(np.uint64) * 11) % p).astype(np.uint32)
    r_true = rows - dep.size
    d = torch.from_numpy(a.view(np.int32)).to(dev)
    rank, piv, k = L.nullspace_u32(d, p)
    assert rank == r_true
    pivn = piv.numpy()
    assert np.array_equal(pivn, np.arange(r_true)), "pivots 0..r-1 w.h.p. for dense uniform rows"
    assert k.shape == (cols, cols - rank)
    # structure
    R = d.to(torch.int64)
    assert int(R.min()) >= 0 and int(R.max()) < p
    assert torch.equal(R[:rank, :rank], torch.eye(rank, dtype=torch.int64, device=dev))
    assert not R[rank:].any()
    # Freivalds: A.v == A[:, :r].(R.v) for every row, three vectors; A.(K.z) == 0
    A = torch.from_numpy(a.astype(np.int64)).to(dev)
    v = torch.from_numpy(np.stack([gen.uniform_rows(0, 1, cols, p, seed=900 + j)[0] for j in range(3)], axis=1)
                         .astype(np.int64)).to(dev)
    z = torch.from_numpy(gen.uniform_rows(0, 1, cols - rank, p, seed=950)[0].astype(np.int64)).to(dev)[:, None]
    bad = 0
    Rv = torch.cat([_matvec(R[r0:min(r0 + 500, rank), :], v, p) for r0 in range(0, rank, 500)])
    K64 = k.to(torch.int64)
    Kz = torch.cat([_matvec(K64[r0:r0 + 500], z, p) for r0 in range(0, cols, 500)])
    for r0 in range(0, rows, 500):
        blk = A[r0:r0 + 500]
        lhs = _matvec(blk, v, p)
        rhs = _matvec(blk[:, :rank], Rv, p)
        bad += int((lhs != rhs).sum()) + int(_matvec(blk, Kz, p).count_nonzero())
    assert bad == 0
    # exact, sampled: rows of A against the oracle's plain product with sampled columns of R
    rng = np.random.default_rng(6)
    rows_s = np.sort(rng.choice(rows, size=6, replace=False))
    rows_s[0] = 39
    cols_s = np.sort(np.concatenate([rng.choice(rank, 100, replace=False), rank + rng.choice(cols - rank, 400, replace=False)]))
    r_cols = from_device(d[:rank][:, torch.from_numpy(cols_s).to(dev)].contiguous())
    got = oracle.matmul_modp(np.ascontiguousarray(a[rows_s][:, :rank]), np.ascontiguousarray(r_cols), p,
                             nthreads=oracle.max_threads())
    assert np.array_equal(got, a[rows_s][:, cols_s])


@pytest.mark.parametrize("lookahead", [1, 0])
def test_lookahead_with_row_exchanges_in_every_strip(oracle, lookahead):
    """The look-ahead schedule defers a strip's row exchanges on all columns but its own while the previous strip's bulk
    update still owns those rows.  Here every strip must fetch pivots from far below its candidate rows (the block
    under the diagonal is zero), some rows are dependent, and a band of columns is free: exchanges, the general panel
    path and free columns occur in every strip, with look-ahead on and off; both must give the oracle's bytes."""
    import paper_2605_25863_b200 as L
    p, n, m = P31, 3072, 2816
    a = gen.uniform_matrix(n, m, p, seed=41)
    for s in range(0, m, 128):
        a[s:s + 96, s:s + 128] = 0                      # the candidate rows of every strip are zero in its columns
    a[500:520] = ((a[100:120].astype(np.uint64) * 3 + a[900:920].astype(np.uint64)) % p).astype(np.uint32)   # dependent rows
    a[:, 1500:1530] = 0                                 # free columns
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    try:
        L.set_option("lookahead", lookahead)
        L.set_option("la_ctas", 40)                     # force the fork (the cost model would not fork at this size)
        out, rank, piv, st = gpu_rref(a, p)
    finally:
        L.set_option("lookahead", 1)
        L.set_option("la_ctas", 0)
    assert rank == rank_ref and np.array_equal(piv, piv_ref)
    assert np.array_equal(out, r_ref)
    assert st["row_swaps"] > 1000
    assert (st["lookahead_strips"] > 5) == (lookahead == 1)
