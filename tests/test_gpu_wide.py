"""Parity of the wide-modulus CUDA path (uint32 storage with 2^31 <= p < 2^32, and the
uint64 backend) against the CPU oracle, element by element (bit-exact), through the C ABI."""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import gpu_rref, require_cuda, SENTINEL

pytestmark = pytest.mark.gpu

P32 = 4294967291          # 2^32 - 5
P32B = 2147483659         # first prime above 2^31
P61 = (1 << 61) - 1
P63 = 9223372036854775783 # 2^63 - 25
P40 = 1099511627791


@pytest.fixture(autouse=True, scope="module")
def _cuda():
    require_cuda()


def gpu_rref64(a: np.ndarray, p: int, ld: int | None = None):
    import paper_2605_25863_b200 as L
    rows, cols = a.shape
    ld = cols if ld is None else ld
    buf = np.full((rows, ld), SENTINEL, dtype=np.uint64)
    buf[:, :cols] = a
    t = torch.from_numpy(buf.view(np.int64)).cuda()
    view = t[:, :cols] if cols else t
    rank, piv = L.rref_u64(view, p)
    out = t.cpu().numpy().view(np.uint64)
    if ld > cols:
        assert (out[:, cols:] == SENTINEL).all(), "padding columns were written"
    return out[:, :cols].copy(), rank, piv.numpy().copy()


def check32(oracle, a, p, ld=None):
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    r, rank, piv, _ = gpu_rref(a, p, ld)
    assert rank == rank_ref and np.array_equal(piv, piv_ref)
    assert np.array_equal(r, r_ref)


def check64(oracle, a, p, ld=None):
    r_ref, rank_ref, piv_ref = oracle.rref_modp64(a, p, nthreads=oracle.max_threads())
    r, rank, piv = gpu_rref64(a, p, ld)
    assert rank == rank_ref and np.array_equal(piv, piv_ref)
    assert np.array_equal(r, r_ref)


SHAPES = [(1, 1), (1, 7), (7, 1), (5, 5), (31, 33), (33, 31), (32, 32), (64, 64), (65, 63), (100, 257), (257, 100),
          (300, 300)]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("p", [P32, P32B])
def test_u32_wide_small_dense(oracle, shape, p):
    a = gen.uniform_matrix(shape[0], shape[1], p, seed=200 + shape[0] + shape[1])
    if a.size > 3:
        a.flat[0] = p - 1
        a.flat[a.size // 2] = 0xFFFFFFFF        # >= p: reduced on entry (reading Q5)
    check32(oracle, a, p)


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("p", [P61, P63, P40, 7])
def test_u64_small_dense(oracle, shape, p):
    a = gen.uniform_matrix_u64(shape[0], shape[1], p, seed=300 + shape[0] + shape[1])
    if a.size > 3:
        a.flat[0] = p - 1
        a.flat[a.size // 2] = np.uint64(0xFFFFFFFFFFFFFFFF)
    check64(oracle, a, p)


@pytest.mark.parametrize("which", ["u32", "u64"])
def test_rank_deficient_free_columns_pivots_far_down(oracle, which):
    p = P32 if which == "u32" else P61
    mk = gen.uniform_matrix if which == "u32" else gen.uniform_matrix_u64
    dt = np.uint32 if which == "u32" else np.uint64
    chk = check32 if which == "u32" else check64
    # product of factors: exact rank 37, non-trivial free block
    b, c = mk(150, 37, p, 2), mk(37, 190, p, 3)
    a = np.array((b.astype(object) @ c.astype(object)) % p, dtype=dt)
    chk(oracle, a, p)
    # zero / dependent columns in the middle, pivots that only appear in later chunks of the scan
    a = mk(300, 140, p, 9)
    a[:, 5] = 0
    a[:, 40:75] = 0
    a[:, 130] = a[:, 3]
    a[:150, :60] = 0
    a[10:20, :] = 0
    chk(oracle, a, p)
    # all-zero, identity, a permutation matrix
    chk(oracle, np.zeros((70, 90), dtype=dt), p)
    pm = np.zeros((150, 150), dtype=dt)
    pm[np.arange(150), np.random.default_rng(1).permutation(150)] = 1
    chk(oracle, pm, p)


@pytest.mark.parametrize("shape,ld", [((50, 37), 41), ((129, 65), 67)])
def test_odd_leading_dimension(oracle, shape, ld):
    check32(oracle, gen.uniform_matrix(shape[0], shape[1], P32, seed=3), P32, ld=ld)
    check64(oracle, gen.uniform_matrix_u64(shape[0], shape[1], P63, seed=3), P63, ld=ld)


def test_medium_sizes_span_many_panels(oracle):
    """Several column tiles of every kernel, a ragged tail, wide and tall shapes."""
    check32(oracle, gen.uniform_matrix(700, 1000, P32, seed=11), P32)
    check32(oracle, gen.uniform_matrix(1000, 700, P32B, seed=12), P32B)
    check64(oracle, gen.uniform_matrix_u64(500, 777, P63, seed=13), P63)
    check64(oracle, gen.uniform_matrix_u64(777, 500, P61, seed=14), P61)


def test_nullspace_and_solve_with_wide_p(oracle):
    """The consumers of the RREF work unchanged on top of the wide path (A.K = 0 by the oracle's plain product)."""
    import paper_2605_25863_b200 as L
    from gpu_util import to_device_padded, from_device
    p = P32
    b, c = gen.uniform_matrix(120, 50, p, 2), gen.uniform_matrix(50, 160, p, 3)
    a = ((b.astype(object) @ c.astype(object)) % p).astype(np.uint32)
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p)
    k_ref = oracle.nullspace_modp(r_ref, p, rank_ref, piv_ref)
    d = to_device_padded(a)
    rank, piv, k = L.nullspace_u32(d, p)
    assert rank == rank_ref == 50 and np.array_equal(from_device(k), k_ref)
    assert not oracle.matmul_modp(a, from_device(k), p).any()


def test_bad_moduli():
    import paper_2605_25863_b200 as L
    t = torch.zeros((4, 4), dtype=torch.int64, device="cuda")
    for bad in [2, 4, 1 << 63, (1 << 61) + 1, 0xFFFFFFFF * 3]:
        with pytest.raises(L.LinacError) as e:
            L.rref_u64(t, bad)
        assert e.value.status == L.linac.ERR_BAD_MODULUS
    t32 = torch.zeros((4, 4), dtype=torch.int32, device="cuda")
    with pytest.raises(L.LinacError):
        L.rref_u32(t32, 4294967295)      # 2^32 - 1 = 3 * 5 * 17 * 257 * 65537
