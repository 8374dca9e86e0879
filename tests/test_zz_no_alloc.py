"""linac_gemm_sub_u32_static: the entry point that allocates no device memory (scratch in the library's static
32 MiB device array) against the existing linac_gemm_sub_u32, bit for bit -- integer work, so the tolerance is
equality, as in tests/test_gpu_gemm.py -- on calls in a row that share the array.  This file sorts last on purpose."""
import gc

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


def _dev(x):
    return torch.from_numpy(x.view(np.int32)).cuda()


def _operands(m, n, k, p, seed):
    return (gen.uniform_matrix(m, n, p, seed), gen.uniform_matrix(m, k, p, seed + 1), gen.uniform_matrix(k, n, p, seed + 2))


def test_two_calls_in_a_row_match_the_existing_path_without_allocating():
    import paper_2605_25863_b200 as L
    # second call: smaller, ragged, K padded up to the next multiple of 128 -- it reads limb planes whose padding the
    # first call left full of its own data unless the second call rewrites it; third call: another modulus
    cases = [(1024, 1536, 512, P31, 11), (333, 517, 200, P31, 21), (700, 260, 1000, P29, 31), (96, 40, 7, P29, 41)]
    ref, dev = [], []
    for (m, n, k, p, seed) in cases:
        c, a, b = _operands(m, n, k, p, seed)
        d_ref = _dev(c)
        L.gemm_sub_u32(d_ref, _dev(a), _dev(b), p, 0)                  # the existing path (workspace from the library)
        ref.append(from_device(d_ref))
        del d_ref
        dev.append((_dev(c), _dev(a), _dev(b), p))
    tiny = torch.zeros((8, 8), dtype=torch.int32, device="cuda")
    L.gemm_sub_u32_static(tiny, tiny.clone(), tiny.clone(), P31)      # set-up: the module with the array is loaded here
    torch.cuda.synchronize()
    gc.collect()                                                       # tensors of earlier tests still waiting in reference cycles go now,
    torch.cuda.synchronize()                                           # not in the middle of the measurement below
    before = torch.cuda.memory_allocated()
    free_before, _ = torch.cuda.mem_get_info()
    for t in dev:                                                      # back to back on one stream, no sync between
        L.gemm_sub_u32_static(*t)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_allocated() <= before                     # the binding made no tensor (a collection may still free one)
    assert free_after >= free_before, "device memory was allocated inside the no-allocation entry point"
    for t, want in zip(dev, ref):
        assert np.array_equal(from_device(t[0]), want)
    # and the first case again, after the others have overwritten the array
    m, n, k, p, seed = cases[0]
    c, a, b = _operands(m, n, k, p, seed)
    dc = _dev(c)
    L.gemm_sub_u32_static(dc, _dev(a), _dev(b), p)
    assert np.array_equal(from_device(dc), ref[0])


def test_the_limit_is_enforced_before_anything_runs():
    import paper_2605_25863_b200 as L
    from paper_2605_25863_b200 import linac
    # 4 (M + N) Kc + 4096 with M = N = 4096: Kc = 1024 fits exactly below 32 MiB?  No: 4 * 8192 * 1024 = 32 MiB, plus
    # 4096 -> just over.  K = 896 fits; K = 1024 is rejected and C stays as it was.
    m = n = 4096
    c = torch.full((m, n), 5, dtype=torch.int32, device="cuda")
    a = torch.ones((m, 1024), dtype=torch.int32, device="cuda")
    b = torch.ones((1024, n), dtype=torch.int32, device="cuda")
    with pytest.raises(L.LinacError) as ei:
        L.gemm_sub_u32_static(c, a, b, P31)
    assert ei.value.status == linac.ERR_TOO_LARGE and "static scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert int(c.min()) == 5 and int(c.max()) == 5
    L.gemm_sub_u32_static(c, a[:, :896], b[:896], P31)                 # largest K that fits at this M, N
    torch.cuda.synchronize()
    want = (5 - 896) % P31
    assert int(c.min()) == want and int(c.max()) == want
    with pytest.raises(L.LinacError) as ei:
        L.gemm_sub_u32_static(c, a, b, 2147483645)                     # 5 x 429496729: rejected as everywhere else
    assert ei.value.status == linac.ERR_BAD_MODULUS
