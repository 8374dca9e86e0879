"""Row-block solve of a regular strip as one tensor-core product with the strip's explicit operator W
(`strip_winv_kernel` + `trsm_winv_kernel`, paper_2605_25863_b200/csrc/fp_trsm_inv.cuh; S4 of SURVEY.md 8(a)).

The path is taken inside the look-ahead sweep (at least 1536 rows and columns) for strips whose four base panels found
32 pivots each; every case here is compared with the oracle's bytes, with the option on and off:

  * ragged widths: cols - 128 k is never a multiple of 32, so every solve ends in a partial tile;
  * a leading dimension that breaks the 16-byte alignment of the rows (scalar stores in the epilogue);
  * p = 2^31 - 1, a second 31-bit prime, and the tiny fields 3 and 2 (p = 2: general panel path, non-Montgomery tensor
    epilogue in the update that consumes the limb planes this kernel writes);
  * regular strips that exchange rows (zero blocks under the diagonal): the deferred exchanges of a look-ahead strip
    must reach the columns right of it before the product reads them.
"""
import numpy as np
import pytest

import linac_inputs as gen
from gpu_util import gpu_rref, require_cuda

pytestmark = pytest.mark.gpu
P31 = 2147483647
P29 = 2147483629


@pytest.fixture(autouse=True, scope="module")
def _cuda():
    require_cuda()


def _run(a, p, ld=None, **opts):
    import paper_2605_25863_b200 as L
    try:
        for k, v in opts.items():
            L.set_option(k, v)
        return gpu_rref(a, p, ld)
    finally:
        for k in opts:
            L.set_option(k, {"trsm_winv": 1, "la_ctas": 0, "lookahead": 1, "trsm_split": 1, "pdl": 1, "tc_panel_deep": 1}[k])


@pytest.mark.parametrize("p", [P31, P29, 3, 2])
def test_ragged_full_rank_wide_matches_oracle_with_and_without_w(oracle, p):
    rows, cols = 2000, 2077
    a = gen.uniform_matrix(rows, cols, p, seed=70 + (p % 13))
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    for winv in (1, 0):
        out, rank, piv, st = _run(a, p, trsm_winv=winv)
        assert rank == rank_ref and np.array_equal(piv, piv_ref)
        assert np.array_equal(out, r_ref)
        if winv == 0:
            assert st["winv_solves"] == 0
        else:
            assert st["winv_solves"] >= 10


def test_unaligned_rows(oracle):
    p, rows, cols = P31, 1700, 1903
    a = gen.uniform_matrix(rows, cols, p, seed=81)
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    out, rank, piv, st = _run(a, p, ld=cols + 3)
    assert rank == rank_ref and np.array_equal(piv, piv_ref)
    assert np.array_equal(out, r_ref)
    assert st["winv_solves"] >= 10


@pytest.mark.parametrize("p,la_ctas", [(P31, 0), (P31, 40), (3, 40)])
def test_regular_strips_that_exchange_rows(oracle, p, la_ctas):
    """The first 40 candidate rows of every strip are zero in the strip's columns, so its panels fetch their pivots from
    further down (row exchanges, the general panel path) while every panel still finds its 32 pivots; with a forced
    partition every strip after the first is a look-ahead strip whose exchanges on the other columns are deferred.  Over
    F_3 a third of all candidate entries is zero anyway."""
    rows, cols = 2304, 2500
    a = gen.uniform_matrix(rows, cols, p, seed=83)
    for s0 in range(0, rows, 128):
        a[s0:s0 + 40, s0:s0 + 128] = 0
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    assert rank_ref == rows
    out, rank, piv, st = _run(a, p, la_ctas=la_ctas)
    assert rank == rank_ref and np.array_equal(piv, piv_ref)
    assert np.array_equal(out, r_ref)
    assert st["row_swaps"] > 100
    assert st["winv_solves"] >= 10
    assert (st["lookahead_strips"] > 5) == (la_ctas == 40)


@pytest.fixture(scope="module")
def forked_case(oracle):
    """2304 x 2500 dense over F_{2^31-1}, its oracle RREF computed once for the option sweep below."""
    a = gen.uniform_matrix(2304, 2500, P31, seed=91)
    return a, oracle.rref_modp(a, P31, nthreads=oracle.max_threads())


@pytest.mark.parametrize("opts", [{"trsm_split": 0}, {"pdl": 0}, {"tc_panel_deep": 0}, {"trsm_split": 0, "pdl": 0, "tc_panel_deep": 0},
                                  {"lookahead": 0}])
def test_schedule_options_of_the_forked_sweep_keep_the_bytes(forked_case, opts):
    """The split of the W product over two streams, the programmatic dependent launch of the updates behind it and the
    deep C-tile ring of the K = 128 update only change the schedule; with a forced partition every strip is forked."""
    a, (r_ref, rank_ref, piv_ref) = forked_case
    out, rank, piv, st = _run(a, P31, la_ctas=40, **opts)
    assert rank == rank_ref and np.array_equal(piv, piv_ref)
    assert np.array_equal(out, r_ref)
    assert (st["lookahead_strips"] > 5) == (opts.get("lookahead", 1) == 1)
