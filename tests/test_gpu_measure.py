"""The measurement plumbing bench.py relies on: linac_measure_peak returns pipe rates in the documented units, and the
production-schedule timing mode (timing = 2) accounts for the step without changing the result."""
import numpy as np
import pytest
import torch

import linac_inputs as gen
from gpu_util import require_cuda, gpu_rref

pytestmark = pytest.mark.gpu


def test_measure_peak_units_and_ranges():
    require_cuda()
    import paper_2605_25863_b200 as L
    v, mhz = L.measure_peak("tc_i8_n256", 2.0)
    assert 1500.0 < v < 6000.0 and 800.0 < mhz < 2500.0          # TOP/s: nominal 4.5 P dense int8
    v128, _ = L.measure_peak("tc_i8_n128", 2.0)
    assert 1000.0 < v128 < 6000.0
    v, mhz = L.measure_peak("dmma", 2.0)
    assert 15.0 < v < 45.0                                       # TFLOP/s: 148 SMs x 64 FMA/clk x 2 x 1.965 GHz = 37.2
    v, mhz = L.measure_peak("imad_wide", 2.0)
    assert 4.0 < v < 12.0                                        # T/s: the wide multiply takes two passes of the FMA pipe (148 x 32 lanes x 1.965 GHz = 9.3)
    scratch = torch.empty(1 << 30, dtype=torch.uint8, device="cuda")
    copy, _ = L.measure_peak("hbm_copy", 0, scratch)
    read, _ = L.measure_peak("hbm_read", 0, scratch)
    assert 3000.0 < copy < 8500.0 and 3000.0 < read < 8500.0     # GB/s: 7.7 TB/s nominal
    with pytest.raises(L.LinacError):
        L.measure_peak("no_such_pipe", 1.0)


def test_timing_mode_2_keeps_the_result_and_accounts_for_the_step(oracle):
    require_cuda()
    import paper_2605_25863_b200 as L
    p = 2147483647
    a = gen.uniform_matrix(1500, 1700, p, seed=77)
    r_ref, rank_ref, piv_ref = oracle.rref_modp(a, p, nthreads=oracle.max_threads())
    try:
        L.set_option("timing", 2)
        r, rank, piv, st = gpu_rref(a, p)
    finally:
        L.set_option("timing", 0)
    assert rank == rank_ref and np.array_equal(piv, piv_ref) and np.array_equal(r, r_ref)
    parts = st["ms_update"] + st["ms_strip"] + st["ms_trsm"]
    assert st["ms_update"] > 0 and st["ms_strip"] > 0 and st["ms_trsm"] > 0
    assert parts <= st["ms_total"] * 1.02 + 0.05                  # the classes are disjoint launches of one stream
    assert st["top_k"] > 0 and st["ms_update_top"] > 0


def test_marks_of_a_timed_call_cover_its_launches_and_show_the_overlap():
    """linac_get_last_marks: with timing = 2 every strip / update / solve launch of the call has an interval inside the call,
    and under look-ahead some strip kernel runs while an update on the second stream is in flight."""
    require_cuda()
    import paper_2605_25863_b200 as L
    import linac_inputs as gen
    p = 2147483647
    a = torch.from_numpy(gen.uniform_matrix(2304, 2304, p, seed=5).view(np.int32)).cuda()
    try:
        L.set_option("timing", 2)
        L.set_option("la_ctas", 40)
        rank, _ = L.rref_u32(a, p)
    finally:
        L.set_option("timing", 0)
        L.set_option("la_ctas", 0)
    st, marks = L.last_stats(), L.last_marks()
    assert rank == 2304 and st["lookahead_strips"] > 5
    assert len(marks) >= 4 * 18 - 8 and {m["cls"] for m in marks} == {0, 1, 2}
    assert all(0.0 <= m["t0_ms"] <= m["t1_ms"] <= st["ms_total"] + 1e-3 for m in marks)
    strips = [m for m in marks if m["cls"] == 1]
    bulk = [m for m in marks if m["cls"] == 0 and m["stream"] == 1]
    assert bulk and any(min(s["t1_ms"], b["t1_ms"]) > max(s["t0_ms"], b["t0_ms"]) for s in strips for b in bulk)
    L.set_option("timing", 0)
    L.rref_u32(torch.from_numpy(gen.uniform_matrix(64, 64, p, seed=6).view(np.int32)).cuda(), p)
