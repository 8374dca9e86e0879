"""Parity of the CUDA F_p path against the CPU oracle, element by element (bit-exact), through the C ABI."""
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


def check_against_oracle(oracle, a, p, ld=None):
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    r, rank, piv, st = gpu_rref(a, p, ld)
    assert rank == rank_ref
    assert np.array_equal(piv, piv_ref)
    assert np.array_equal(r, r_ref)
    assert st["residual_nonzero"] == 0
    return st


@pytest.mark.parametrize("shape", [(1, 1), (1, 7), (7, 1), (5, 5), (31, 33), (33, 31), (32, 32), (64, 64), (65, 63),
                                   (100, 257), (257, 100), (130, 130), (300, 300)])
@pytest.mark.parametrize("p", [P31, 7, 2])
def test_small_dense_shapes(oracle, shape, p):
    a = gen.uniform_matrix(shape[0], shape[1], p, seed=100 + shape[0] + shape[1])
    check_against_oracle(oracle, a, p)


@pytest.mark.parametrize("shape,ld", [((50, 37), 41), ((129, 65), 67), ((64, 100), 101)])
def test_odd_leading_dimension_and_padding_untouched(oracle, shape, ld):
    a = gen.uniform_matrix(shape[0], shape[1], P29, seed=3)
    check_against_oracle(oracle, a, P29, ld=ld)


def test_empty_shapes():
    import paper_2605_25863_b200 as L
    for shape in [(0, 5), (5, 0), (0, 0)]:
        t = torch.zeros(shape, dtype=torch.int32, device="cuda")
        rank, piv = L.rref_u32(t, P31)
        assert rank == 0 and piv.numel() == 0


def test_all_zero_and_identity_and_permutation(oracle):
    z = np.zeros((70, 90), dtype=np.uint32)
    r, rank, piv, _ = gpu_rref(z, P31)
    assert rank == 0 and not r.any()
    rng = np.random.default_rng(1)
    n = 150
    pm = np.zeros((n, n), dtype=np.uint32)
    pm[np.arange(n), rng.permutation(n)] = 1
    st = check_against_oracle(oracle, pm, P31)
    assert st["row_swaps"] > 0


@pytest.mark.parametrize("m,r,n", [(120, 40, 150), (200, 33, 90), (96, 64, 96), (400, 100, 300)])
def test_rank_deficient_products(oracle, m, r, n):
    a, _, _ = gen.lowrank_factors(m, r, n, P29, seed_b=2, seed_c=3)
    check_against_oracle(oracle, a, P29)


def test_zero_columns_and_free_columns_in_the_middle(oracle):
    a = gen.uniform_matrix(200, 260, P31, seed=9)
    a[:, 5] = 0
    a[:, 40:75] = 0
    a[:, 130] = a[:, 3]                 # dependent column -> free column with non-trivial RREF entries
    a[:, 131] = (a[:, 4].astype(np.uint64) * 5 % P31).astype(np.uint32)
    check_against_oracle(oracle, a, P31)


def test_pivots_far_down_need_row_swaps(oracle):
    """First rows are zero in the leading columns, so pivots come from later chunks of the scan."""
    a = gen.uniform_matrix(300, 120, P31, seed=10)
    a[:150, :60] = 0
    a[10:20, :] = 0
    st = check_against_oracle(oracle, a, P31)
    assert st["row_swaps"] > 0


def test_sparse_rank_deficient_recipe(oracle):
    """Config c5's generator at an oracle-sized shape (90% zeros, 2% dependent rows)."""
    n = 600
    a = gen.sparse_dependent_rows(0, n, n, n, P31, seed=7, seed_dep=8)
    st = check_against_oracle(oracle, a, P31)
    assert st["row_swaps"] > 0


@pytest.mark.parametrize("shape", [(500, 1500), (1500, 500)])
def test_wide_and_tall(oracle, shape):
    a = gen.uniform_matrix(shape[0], shape[1], P31, seed=11)
    check_against_oracle(oracle, a, P31)


@pytest.mark.parametrize("shape", [(90, 110), (96, 112), (70, 259)])
def test_entries_ge_p_are_reduced(oracle, shape):
    """Scalar ingest (rows not 16-byte aligned), the 128-bit ingest, and both on one matrix (cols % 4 != 0 with
    an aligned leading dimension is exercised through the padded variant below)."""
    rng = np.random.default_rng(4)
    a = rng.integers(0, 2**32, size=shape, dtype=np.uint64).astype(np.uint32)
    check_against_oracle(oracle, a, P29)
    if shape[1] % 4:
        check_against_oracle(oracle, a, P29, ld=(shape[1] + 7) // 4 * 4)


def test_augmented_solve_nontrivial_output(oracle):
    """(A | B) with 64 extra columns: the RREF is (I | A^-1 B), a non-identity output at c1's size."""
    a = gen.uniform_matrix(512, 512 + 64, P31, seed=12)
    check_against_oracle(oracle, a, P31)


def test_config_c1(oracle):
    c = gen.CONFIGS["c1"]
    a = gen.uniform_matrix(c["rows"], c["cols"], c["p"], c["seed"])
    check_against_oracle(oracle, a, c["p"])


def test_bad_arguments():
    import paper_2605_25863_b200 as L
    t = torch.zeros((4, 4), dtype=torch.int32, device="cuda")
    for bad_p in (0, 1, 4, 2147483649 % (1 << 32), 2147483647 * 0 + 15):
        with pytest.raises(L.LinacError) as e:
            L.rref_u32(t, bad_p)
        assert e.value.status == L.linac.ERR_BAD_MODULUS


# ------------------------------------------------------------------ null space
@pytest.mark.parametrize("m,r,n", [(60, 20, 75), (150, 150, 200), (128, 40, 128)])
def test_nullspace_matches_oracle(oracle, m, r, n):
    import paper_2605_25863_b200 as L
    a, _, _ = gen.lowrank_factors(m, min(r, m, n), n, P29, seed_b=5, seed_c=6)
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, P29)
    k_ref = oracle.nullspace_modp(r_ref, P29, rank_ref, piv_ref)
    buf = to_device_padded(a)
    rank, piv, k = L.nullspace_u32(buf, P29)
    assert rank == rank_ref and np.array_equal(piv.numpy(), piv_ref)
    assert np.array_equal(from_device(buf), r_ref)
    assert np.array_equal(from_device(k), k_ref)
    # caller-provided buffer, exact capacity and too small
    buf2 = to_device_padded(a)
    kbuf = torch.zeros((n, n - rank_ref + 3), dtype=torch.int32, device="cuda")
    rank2, _, k2 = L.nullspace_u32(buf2, P29, kbuf)
    assert np.array_equal(from_device(k2), k_ref)
    if n - rank_ref > 1:
        buf3 = to_device_padded(a)
        small = torch.zeros((n, n - rank_ref - 1), dtype=torch.int32, device="cuda")
        with pytest.raises(L.LinacError) as e:
            L.nullspace_u32(buf3, P29, small)
        assert e.value.status == L.linac.ERR_BUFFER_TOO_SMALL
        assert np.array_equal(from_device(buf3), r_ref)      # documented: dA already holds the RREF


# ------------------------------------------------------------------ schedule variants
@pytest.mark.parametrize("opts", [
    {"strip_width": 32}, {"strip_width": 64}, {"strip_width": 256}, {"strip_width": 96, "flat_group": 2},
    {"flat_cols": 0}, {"flat_cols": 256, "flat_group": 4}, {"tc_panel": 0}, {"gemm_path": 1},
    {"tc_min_k": 32, "tc_min_mn": 128, "strip_width": 32},
])
def test_schedule_options_do_not_change_the_result(oracle, opts):
    """Every tunable only changes the schedule (strip width, flat sweep vs recursion, which GEMM kernel): the RREF
    is unique, so the bytes must not move.  One rank-deficient and one full-rank wide matrix."""
    import paper_2605_25863_b200 as L
    defaults = {"strip_width": 128, "flat_group": 1, "flat_cols": 16384, "tc_panel": 1, "gemm_path": 0,
                "tc_min_k": 48, "tc_min_mn": 128}
    a1, _, _ = gen.lowrank_factors(700, 333, 900, P29, seed_b=21, seed_c=22)
    a2 = gen.uniform_matrix(600, 1100, P31, seed=23)
    try:
        for k, v in opts.items():
            L.set_option(k, v)
        check_against_oracle(oracle, a1, P29)
        check_against_oracle(oracle, a2, P31)
    finally:
        for k, v in defaults.items():
            L.set_option(k, v)


# ------------------------------------------------------------------ mid-size stress (several strips, all paths)
@pytest.mark.parametrize("case", ["tall", "wide", "p3", "zero_blocks", "sparse2000", "lowrank_swaps"])
def test_mid_size_stress(oracle, case):
    """Shapes spanning many strips where the general panel path, row exchanges, free columns and rank exhaustion
    all occur, still small enough for the oracle."""
    if case == "tall":
        a, p = gen.uniform_matrix(3000, 700, P31, seed=31), P31
    elif case == "wide":
        a, p = gen.uniform_matrix(700, 3000, P29, seed=32), P29
    elif case == "p3":
        a, p = gen.uniform_matrix(1200, 1200, 3, seed=33), 3              # a third of all entries are zero
    elif case == "zero_blocks":
        a, p = gen.uniform_matrix(1500, 1500, 65521, seed=34), 65521
        a[:, 100:230] = 0
        a[:, 700:701] = 0
        a[300:420, :] = 0
        a[:, 1000:1100] = a[:, 0:100]                                     # dependent columns
    elif case == "sparse2000":
        a, p = gen.sparse_dependent_rows(0, 2000, 2000, 2000, P31, seed=7, seed_dep=8), P31
    else:
        a, _, _ = gen.lowrank_factors(1800, 900, 1600, P31, seed_b=35, seed_c=36)
        a, p = a[::-1].copy(), P31                                        # reversed rows: same row space
        a[:64, :] = 0                                                     # pivots must come from further down
    check_against_oracle(oracle, a, p)
