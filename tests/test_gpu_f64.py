"""fp64 path through the C ABI: backward error <= 1e-11 on the original data (BASELINE.json), agreement with
the oracle's solution to rounding, singular detection, exact special cases."""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import require_cuda

pytestmark = pytest.mark.gpu
ETA_MAX = 1e-11        # north_star: ||Ax-b|| / (||A|| ||x|| + ||b||) <= 1e-11


@pytest.fixture(autouse=True, scope="module")
def _cuda():
    require_cuda()


def gpu_solve(a, b, tol=-1.0, lda=None, ldb=None):
    import paper_2605_25863_b200 as L
    n, nrhs = b.shape
    lda = n if lda is None else lda
    ldb = nrhs if ldb is None else ldb
    da = torch.full((n, lda), float("nan"), dtype=torch.float64, device="cuda")
    db = torch.full((n, ldb), float("nan"), dtype=torch.float64, device="cuda")
    da[:, :n] = torch.from_numpy(a).cuda()
    db[:, :nrhs] = torch.from_numpy(b).cuda()
    L.solve_f64(da[:, :n], db[:, :nrhs], tol)
    if ldb > nrhs:
        assert torch.isnan(db[:, nrhs:]).all()
    return db[:, :nrhs].cpu().numpy()


@pytest.mark.parametrize("n,nrhs", [(1, 1), (2, 2), (31, 3), (32, 1), (33, 5), (64, 64), (100, 7), (257, 9), (1000, 64)])
def test_solve_backward_error_and_oracle_agreement(oracle, n, nrhs):
    a, b = gen.shifted_normal_system(n, nrhs, seed_a=5, seed_b=6)
    x = gpu_solve(a, b)
    eta = oracle.backward_error(a, x, b, nthreads=oracle.max_threads())
    assert eta <= ETA_MAX
    rc, info, x_ref = oracle.solve_f64(a, b, nthreads=oracle.max_threads())
    assert rc == 0
    assert np.allclose(x, x_ref, rtol=1e-9, atol=1e-12)          # several x are "correct": loose agreement only


def test_unshifted_gaussian_needs_pivoting(oracle):
    """Plain N(0,1) matrix (no diagonal shift): without partial pivoting the error would be huge."""
    n = 500
    a = gen.normal_matrix(n, n, seed=21)
    b = gen.normal_matrix(n, 4, seed=22)
    x = gpu_solve(a, b)
    assert oracle.backward_error(a, x, b, nthreads=oracle.max_threads()) <= ETA_MAX


def test_row_scaling_and_leading_dimensions(oracle):
    n, nrhs = 150, 6
    a, b = gen.shifted_normal_system(n, nrhs, seed_a=7, seed_b=8)
    scale = 10.0 ** np.linspace(-8, 8, n)
    a2, b2 = a * scale[:, None], b * scale[:, None]          # badly row-scaled, same solution
    x = gpu_solve(a2, b2, lda=n + 3, ldb=nrhs + 2)
    assert oracle.backward_error(a, x, b) <= ETA_MAX
    assert oracle.backward_error(a2, x, b2) <= ETA_MAX


def test_exact_cases_and_manufactured_solution():
    n = 96
    b = gen.normal_matrix(n, 3, seed=3)
    assert np.array_equal(gpu_solve(np.eye(n), b), b)
    d = 2.0 ** np.arange(-10, n - 10, dtype=np.float64)
    assert np.array_equal(gpu_solve(np.diag(d), b), b / d[:, None])
    perm = np.random.default_rng(1).permutation(n)
    pm = np.eye(n)[perm]
    assert np.array_equal(gpu_solve(pm, b), pm.T @ b)
    a, _ = gen.shifted_normal_system(n, 1, seed_a=9, seed_b=10)
    ones = np.ones((n, 2))
    assert np.allclose(gpu_solve(a, a @ ones), ones, rtol=1e-12)


def test_singular_is_reported():
    import paper_2605_25863_b200 as L
    n = 80
    a, b = gen.shifted_normal_system(n, 2, seed_a=1, seed_b=2)
    a[50] = a[20]
    with pytest.raises(L.LinacError) as e:
        gpu_solve(a, b)
    assert e.value.status == L.linac.ERR_SINGULAR and 1 <= e.value.info <= n
    z, _ = gen.shifted_normal_system(n, 2, seed_a=1, seed_b=2)
    z[7] = 0.0
    with pytest.raises(L.LinacError) as e:
        gpu_solve(z, b)
    assert e.value.status == L.linac.ERR_SINGULAR
    # caller-controlled threshold
    a, b = gen.shifted_normal_system(n, 2, seed_a=1, seed_b=2)
    a[50] = a[20] * (1 + 1e-9)
    with pytest.raises(L.LinacError):
        gpu_solve(a, b, tol=1e-6)
    gpu_solve(a, b, tol=0.0)


def test_medium_size_several_panels_and_recursion_levels(oracle):
    n, nrhs = 3000, 64
    a, b = gen.shifted_normal_system(n, nrhs, seed_a=5, seed_b=6)
    x = gpu_solve(a, b)
    assert oracle.backward_error(a, x, b, nthreads=oracle.max_threads()) <= ETA_MAX
    ref = np.linalg.solve(a, b)
    assert np.allclose(x, ref, rtol=1e-9, atol=1e-12)


@pytest.mark.parametrize("opts", [
    {"f64_strip": 0}, {"f64_strip": 256}, {"f64_rhs_inv": 0}, {"f64_mma": 0},
    {"f64_panel_threads": 256}, {"f64_panel_threads": 1024}, {"f64_panel_tags": 0},
    {"f64_panel_cluster": 16, "f64_cluster_rows": 4096}, {"f64_panel_cluster": 8, "f64_cluster_rows": 100},
])
def test_schedule_options_solve_the_same_system(oracle, opts):
    """Every schedule (pure recursion / flat strips, recursive / inverse-block substitution, DFMA / DMMA update, the
    panel kernel's block sizes, the cluster + DSMEM panel kernel) on a matrix that needs row exchanges, with a
    ragged size and more than 64 right-hand sides."""
    import paper_2605_25863_b200 as L
    defaults = {"f64_strip": 512, "f64_rhs_inv": 1, "f64_mma": 1, "f64_panel_threads": 512, "f64_panel_cluster": 0,
                "f64_cluster_rows": 128, "f64_panel_tags": 1}
    n, nrhs = 1337, 70
    a, b = gen.normal_matrix(n, n, seed=21), gen.normal_matrix(n, nrhs, seed=22)
    try:
        for k, v in opts.items():
            L.set_option(k, v)
        x = gpu_solve(a, b)
    finally:
        for k, v in defaults.items():
            L.set_option(k, v)
    assert oracle.backward_error(a, x, b, nthreads=oracle.max_threads()) <= ETA_MAX
    assert np.allclose(x, np.linalg.solve(a, b), rtol=1e-7, atol=1e-10)


def test_tagged_records_match_the_grid_barrier_bitwise_and_repeat():
    """The panel kernel's per-column exchange through self-validating {value, tag} 16-byte words (option
    f64_panel_tags, default) must pick the same pivots and produce the same bits as the grid-barrier version, run
    after run: a torn or stale read would show up as a different pivot row somewhere in 2500 columns."""
    import paper_2605_25863_b200 as L
    n, nrhs = 2500, 9
    a0 = torch.from_numpy(gen.normal_matrix(n, n, seed=31)).cuda()
    b0 = torch.from_numpy(gen.normal_matrix(n, nrhs, seed=32)).cuda()

    def solve():
        a, b = a0.clone(), b0.clone()
        L.solve_f64(a, b)
        return a, b

    try:
        L.set_option("f64_panel_tags", 0)
        lu_ref, x_ref = solve()
    finally:
        L.set_option("f64_panel_tags", 1)
    for _ in range(12):
        lu, x = solve()
        assert torch.equal(lu, lu_ref) and torch.equal(x, x_ref)
