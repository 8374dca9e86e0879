"""S5 primitive C <- C - A.B mod p: CUDA-core kernel and tensor-core (tcgen05 int8 limb) kernel, each
element by element against the oracle's plain triple loop."""
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


def run_gemm(c, a, b, p, path):
    import paper_2605_25863_b200 as L
    dc = torch.from_numpy(c.view(np.int32)).cuda()
    da = torch.from_numpy(a.view(np.int32)).cuda()
    db = torch.from_numpy(b.view(np.int32)).cuda()
    L.gemm_sub_u32(dc, da, db, p, path)
    return from_device(dc), L.last_stats()


def expected(oracle, c, a, b, p):
    prod = oracle.matmul_modp(a, b, p, nthreads=oracle.max_threads())
    return ((c.astype(np.int64) - prod.astype(np.int64)) % p).astype(np.uint32)


SHAPES = [(1, 1, 1), (5, 7, 3), (128, 64, 16), (129, 65, 17), (200, 300, 100), (257, 130, 33)]
TC_SHAPES = [(128, 64, 128), (128, 64, 32), (256, 128, 256), (300, 200, 150), (512, 512, 512), (1000, 900, 700),
             (640, 576, 4224), (130, 70, 1),
             (256, 192, 9000),      # K > 8192: two chunks per call (the s32 accumulators hold K <= 8256)
             # K <= 256: the persistent A-stationary panel kernel (several items per CTA, ragged M and N tiles)
             (1000, 2100, 256), (3000, 1500, 128), (5000, 40, 200), (20000, 100, 256)]


@pytest.mark.parametrize("m,n,k", SHAPES + TC_SHAPES)
@pytest.mark.parametrize("p", [P31, P29, 7])
def test_simt_kernel(oracle, m, n, k, p):
    if (m, n, k) == (640, 576, 4224) and p != P31:
        pytest.skip("one modulus is enough at the largest shape")
    a = gen.uniform_matrix(m, k, p, seed=1)
    b = gen.uniform_matrix(k, n, p, seed=2)
    c = gen.uniform_matrix(m, n, p, seed=3)
    out, _ = run_gemm(c, a, b, p, path=1)
    assert np.array_equal(out, expected(oracle, c, a, b, p))


@pytest.mark.parametrize("m,n,k", TC_SHAPES)
@pytest.mark.parametrize("p", [P31, P29, 7])
def test_tensor_core_kernel(oracle, m, n, k, p):
    if (m, n, k) in ((640, 576, 4224), (256, 192, 9000)) and p != P31:
        pytest.skip("one modulus is enough at the largest shapes")
    a = gen.uniform_matrix(m, k, p, seed=1)
    b = gen.uniform_matrix(k, n, p, seed=2)
    c = gen.uniform_matrix(m, n, p, seed=3)
    out, st = run_gemm(c, a, b, p, path=2)
    assert st["tc_launches"] >= 1
    assert np.array_equal(out, expected(oracle, c, a, b, p))


def test_tensor_core_worst_case_operands(oracle):
    """All entries p-1: every limb product at its maximum, K = 8192 in one launch (s32 accumulator headroom)."""
    m, n, k = 128, 64, 8192
    a = np.full((m, k), P31 - 1, dtype=np.uint32)
    b = np.full((k, n), P31 - 1, dtype=np.uint32)
    c = np.zeros((m, n), dtype=np.uint32)
    out, st = run_gemm(c, a, b, P31, path=2)
    assert st["tc_launches"] == 1
    want = (-(k * pow(P31 - 1, 2, P31))) % P31
    assert (out == want).all()
    out1, _ = run_gemm(c, a, b, P31, path=1)
    assert (out1 == want).all()


@pytest.mark.parametrize("k", [128, 256])
def test_panel_kernel_worst_case_operands(k):
    """All entries p-1 at the panel kernel's largest K: every limb product at its maximum."""
    m, n = 300, 100
    a = np.full((m, k), P31 - 1, dtype=np.uint32)
    b = np.full((k, n), P31 - 1, dtype=np.uint32)
    c = np.zeros((m, n), dtype=np.uint32)
    out, st = run_gemm(c, a, b, P31, path=2)
    assert st["tc_launches"] == 1
    assert (out == (-(k * pow(P31 - 1, 2, P31))) % P31).all()
