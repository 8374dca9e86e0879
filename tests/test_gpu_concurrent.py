""""re-entrant across streams when each call has its own workspace".  Two host threads reduce different
matrices over different primes at the same time, each on its own stream with its own workspace; both results must be
the oracle's bytes, repeatedly."""
import ctypes as C
import threading

import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import require_cuda

pytestmark = pytest.mark.gpu


def _raw_rref(lib, t, p, stream, ws):
    """linac_rref_u32 through the C ABI on an explicit stream with an explicit workspace (the thread's own)."""
    rows, cols = t.shape
    rc = lib.linac_set_workspace(ws.data_ptr(), ws.numel())
    assert rc == 0
    rank = C.c_int64(0)
    piv = np.zeros(max(1, min(rows, cols)), dtype=np.int32)
    rc = lib.linac_rref_u32(t.data_ptr(), rows, cols, t.stride(0), p, C.c_void_p(stream.cuda_stream), C.byref(rank),
                            piv.ctypes.data_as(C.c_void_p))
    assert rc == 0, rc
    return int(rank.value), piv[: rank.value].copy()


def test_two_threads_two_streams_two_primes(oracle):
    require_cuda()
    from paper_2605_25863_b200 import linac
    lib = linac._lib()
    cases = [(gen.lowrank_factors(900, 500, 1100, 2147483629, 2, 3)[0], 2147483629),
             (gen.uniform_matrix(1000, 1000, 2147483647, 5), 2147483647)]
    cases[1][0][:, 300:340] = 0                          # free columns in the middle of the second matrix
    refs = [oracle.rref_modp(a, p, nthreads=oracle.max_threads()) for a, p in cases]
    results = [None, None]
    errors = []

    def worker(i):
        try:
            a, p = cases[i]
            torch.cuda.set_device(0)
            stream = torch.cuda.Stream()
            need = C.c_size_t(0)
            lib.linac_rref_u32_workspace(a.shape[0], a.shape[1], C.byref(need))
            ws = torch.empty(need.value, dtype=torch.uint8, device="cuda")
            out = []
            for _ in range(6):
                with torch.cuda.stream(stream):
                    t = torch.from_numpy(a.view(np.int32)).cuda()
                    stream.synchronize()
                    rank, piv = _raw_rref(lib, t, p, stream, ws)
                    out.append((rank, piv, t.cpu().numpy().view(np.uint32)))
            lib.linac_set_workspace(None, 0)
            results[i] = out
        except Exception as e:      # noqa: BLE001
            errors.append(e)

    th = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errors, errors
    for i in range(2):
        r_ref, rank_ref, piv_ref = refs[i]
        for rank, piv, r in results[i]:
            assert rank == rank_ref and np.array_equal(piv, piv_ref) and np.array_equal(r, r_ref)
