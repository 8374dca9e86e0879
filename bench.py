#!/usr/bin/env python
"""bench.py -- one JSON line for the Linac hot path on B200 (contract: see DESIGN.md "Measurement").

A "step" is one pass of the whole hot path (S0 ingest .. S7 finalise) over one seeded synthetic
matrix.  The HEADLINE workload is config c3, the paper's N = 10^4 point (dense uniform over F_{2^31-1}, PAPER.md:59,
308): `value`, `ms_per_step`, `e2e`, `roofline`, `clocks` describe it.  The default run (1 GPU, no --workload) also
carries one leg per remaining config and per widened row, each with its own timing, clocks and roofline:

  legs.c1, legs.c2   the small F_p configs (c2 with the null space), latency chains: us per pivot
  legs.c5            N = 10^5 (40 GB, generated on the device): 1 warm-up + 2 timed calls
  legs.fp64_solve    config c4 through linac_solve_f64: ms per solve, GFLOP/s, backward error
  legs.rref_f64      SURVEY.md 8(f)#3: linac_rref_f64 on a rank-deficient float64 matrix
  legs.rref_c128     the same for complex128 (linac_rref_c128: the fp64 reduction of the 2 x 2 real block embedding)
  legs.wide_u32/u64  SURVEY.md 8(f)#4: linac_rref_u32 with p = 2^32 - 5 and linac_rref_u64 with p = 2^61 - 1

  value      : whole-job Gmulmod/s = (2 N^3 / 3) / t, matrix already resident in HBM, t = CUDA-event time of the C-ABI
               call (max over ranks); N > 1 runs independent replicas (weak scaling, no collective on the data path).
  e2e        : same metric with HOST buffers: pinned H2D of the matrix + call + D2H of the RREF every step, double
               buffered; the strictly serial figure is kept beside it as e2e.serial_ms_per_step.
  roofline   : the Schur-update kernels (dominant class): executed u8 multiply-accumulates / their CUDA-event time in
               the PRODUCTION schedule (option timing = 2: an event pair around every launch, no host syncs), against
               the int8 tensor peak linac_measure_peak measures live in this run (tcgen05.mma kind::i8 from on-chip
               operands): the 2 ms burst figure when the step held the maximum clock, the 400 ms power-capped one
               otherwise.  roofline.whole_step_frac puts the whole step against the same peak.
  cpu_baseline: the CPU oracle timed on this box's host cores on bounded samples, with labelled cubic extrapolations.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import linac_inputs as gen  # noqa: E402

WORKLOAD_KIND = {"uniform": "dense uniform", "lowrank": "product of uniform factors (exact rank)",
                 "sparse_dep": "90% zeros, every 50th row dependent"}
BASELINE_CONTEXT = ("paper, A100: 3.6 s at N=1e4 (PAPER.md:59) = 185 Gmulmod/s, 45 min at N=1e5 (PAPER.md:61) = 247 "
                    "Gmulmod/s; another machine, context only (BASELINE.json publishes no number for this metric)")
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r02_traffic.json.txt")      # written from an ncu --set full capture of HEAD


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=d["hbm_gbs"], bf16_burst=d["bf16_tflops"], bf16_sustained=d["bf16_tflops_sustained"],
                    sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="MEASURED_PEAKS.json")
    return dict(hbm_gbs=6650.0, bf16_burst=1590.0, bf16_sustained=1400.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except OSError:
            self.proc = None
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in self.rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i] == "Active"})
        busy = [x for x in sm if x > 0.6 * (max(mx) if mx else 1)] or sm
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm), "power_w_max": max(pw) if pw else None}


def make_workload(name: str, rank_seed: int = 0):
    """Returns (host uint32 matrix, p, config).  rank_seed shifts the seed for replicas."""
    c = dict(gen.CONFIGS[name])
    if c["kind"] == "uniform":
        a = gen.uniform_matrix(c["rows"], c["cols"], c["p"], c["seed"] + 1000 * rank_seed)  # == replicas.replica_seed
    elif c["kind"] == "lowrank":
        a, _, _ = gen.lowrank_factors(c["rows"], c["inner"], c["cols"], c["p"], c["seed_b"] + 1000 * rank_seed, c["seed_c"])
    else:
        raise SystemExit(f"workload {name} has no host generator here")
    return a, c["p"], c


# ------------------------------------------------------------------------------------------------ CPU oracle legs
def oracle_time_fp(n: int, p: int, threads: int):
    """Seconds the CPU oracle (as it stands) takes on an n x n dense uniform matrix over F_p."""
    import oracle
    a = gen.uniform_matrix(n, n, p, seed=4)
    t0 = time.perf_counter()
    _, rank, _ = oracle.rref_modp(a, p, nthreads=threads)
    dt = time.perf_counter() - t0
    assert rank == n
    return dt


def oracle_time_f64(n: int, nrhs: int, threads: int):
    import oracle
    a, b = gen.shifted_normal_system(n, nrhs, seed_a=5, seed_b=6)
    t0 = time.perf_counter()
    rc, _, _ = oracle.solve_f64(a, b, nthreads=threads)
    dt = time.perf_counter() - t0
    assert rc == 0
    return dt


def cpu_baseline_plan(p: int, full: bool):
    """SURVEY.md 8(d) "Oracle timed beside it", bounded to ~20-30 s of CPU work by default: the oracle single-threaded at
    c1 and at a 1024^2 sample, the OpenMP build of the same loop on all host cores at c1 and at 1536^2 / 2048^2 samples,
    cubic extrapolations (labelled) to c2, c3 and c5, and the fp64 oracle at 1024 / 2048 extrapolated to c4.  The
    oracle's Gauss-Jordan loop executes N^3/2 multiply-subtracts on an N x N full-rank matrix; the rate below is in
    the metric's unit (2N^3/3 per solve).  --cpu-baseline full runs c2 and c3 themselves (minutes)."""
    import oracle
    threads = oracle.max_threads()
    gm = lambda n, t: (2 * n ** 3 / 3) / t / 1e9          # noqa: E731
    out = {"cores": threads, "kind": "oracle", "unit": "Gmulmod/s"}
    t_c1_1 = oracle_time_fp(512, p, 1)
    t_c1_n = oracle_time_fp(512, p, threads)
    t_1024_1 = oracle_time_fp(1024, p, 1)
    t_1536_n = oracle_time_fp(1536, p, threads)
    t_2048_n = oracle_time_fp(2048, p, threads)
    out["measured"] = {
        "c1_single_thread": {"n": 512, "threads": 1, "seconds": t_c1_1, "value": gm(512, t_c1_1)},
        "c1_openmp": {"n": 512, "threads": threads, "seconds": t_c1_n, "value": gm(512, t_c1_n)},
        "sample_1024_single_thread": {"n": 1024, "threads": 1, "seconds": t_1024_1, "value": gm(1024, t_1024_1)},
        "sample_1536_openmp": {"n": 1536, "threads": threads, "seconds": t_1536_n, "value": gm(1536, t_1536_n)},
        "sample_2048_openmp": {"n": 2048, "threads": threads, "seconds": t_2048_n, "value": gm(2048, t_2048_n)},
    }
    # cubic extrapolation t(N) = t(N0) (N/N0)^3 from the largest measured sample; c2's loop runs rows*cols*rank
    # multiply-subtracts (4096*4096*3000), c5's about rows*cols*rank too (dense after fill-in)
    k1, kn = t_1024_1 / 1024 ** 3, t_2048_n / 2048 ** 3
    out["extrapolated"] = {
        "c2_single_thread_s": k1 * 4096 * 4096 * 3000, "c2_openmp_s": kn * 4096 * 4096 * 3000,
        "c3_single_thread_s": k1 * 1e12, "c3_openmp_s": kn * 1e12,
        "c5_single_thread_s": k1 * 1e5 * 1e5 * 98000, "c5_openmp_s": kn * 1e5 * 1e5 * 98000,
        "label": "EXTRAPOLATED: t = t(N0) * work / N0^3 with work = rows * cols * rank, N0 = 1024 (1 thread) / 2048 "
                 f"({threads} threads); not measured"}
    tf1, tf2 = oracle_time_f64(1024, 64, threads), oracle_time_f64(2048, 64, threads)
    flop = lambda n: 2.0 * n ** 3 / 3.0 + 2.0 * n * n * 64          # noqa: E731
    out["fp64"] = {"measured": {"n1024_openmp_s": tf1, "n2048_openmp_s": tf2, "n2048_gflops": flop(2048) / tf2 / 1e9},
                   "extrapolated": {"c4_openmp_s": tf2 * (16384 / 2048) ** 3,
                                    "label": "EXTRAPOLATED cubically from N = 2048 (the oracle is Gauss-Jordan on (A B): "
                                             "about N^3 multiply-adds)"},
                   "unit": "GFLOP/s in the metric's count (2N^3/3 + 2N^2 nrhs)"}
    if full:
        a2, p2, _ = make_workload("c2")
        t0 = time.perf_counter(); oracle.rref_modp(a2, p2, nthreads=1); t_c2_1 = time.perf_counter() - t0
        t0 = time.perf_counter(); oracle.rref_modp(a2, p2, nthreads=threads); t_c2_n = time.perf_counter() - t0
        a3, p3, _ = make_workload("c3")
        t0 = time.perf_counter(); oracle.rref_modp(a3, p3, nthreads=threads); t_c3_n = time.perf_counter() - t0
        out["measured"].update({"c2_single_thread": {"seconds": t_c2_1, "threads": 1},
                                "c2_openmp": {"seconds": t_c2_n, "threads": threads},
                                "c3_openmp": {"seconds": t_c3_n, "threads": threads, "value": gm(10000, t_c3_n)}})
    # the contract's top-level fields: the OpenMP sample closest to the headline workload
    out["value"] = gm(2048, t_2048_n)
    out["seconds"] = t_2048_n
    out["sample"] = (f"2048x2048 dense uniform F_p (same recipe as c3), oracle Gauss-Jordan, {threads} OpenMP threads; "
                     "see .measured / .extrapolated for the rest of the plan")
    return out


def run_reference(args):
    """--impl reference: the oracle on the host cores, a bounded sample of the same workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    threads = oracle.max_threads()
    n = args.ref_n
    wl = "c3" if args.workload == "all" else args.workload
    p = gen.CONFIGS[wl].get("p", 2147483647)
    for _ in range(args.warmup):
        oracle_time_fp(min(n, 512), p, threads)
    times = [oracle_time_fp(n, p, threads) for _ in range(args.steps)]
    t = float(np.mean(times))
    val = (2 * n ** 3 / 3) / t / 1e9
    sample = f"{n}x{n} dense uniform F_p sample of workload {wl}, CPU oracle Gauss-Jordan"
    print(json.dumps({
        "impl": "reference", "metric": "rref_gmulmod_per_s", "value": val, "unit": "Gmulmod/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": wl, "sample": sample},
        "cpu_baseline": {"value": val, "unit": "Gmulmod/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "Gmulmod/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ------------------------------------------------------------------------------------------------ GPU legs
class Bench:
    def __init__(self, torch, L, dev, local, world, rank, opts):
        self.torch, self.L, self.dev, self.local, self.world, self.rank, self.opts = torch, L, dev, local, world, rank, opts
        self.peaks_file = load_peaks()
        self._peak_cache = {}

    def barrier(self):
        self.torch.cuda.synchronize(self.dev)
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
            self.torch.cuda.synchronize(self.dev)

    def peak(self, what, ms):
        key = (what, ms)
        if key not in self._peak_cache:
            self._peak_cache[key] = self.L.measure_peak(what, ms)
        return self._peak_cache[key]

    def tensor_peak(self, clocks, hot=False):
        """The int8 tensor peak for a run with these clocks: the 2 ms burst figure if the run sat near the maximum clock
        with no power cap, else a power-capped one (both measured live, random operand bytes).  hot=True: the leg has just
        run under the power cap, so the sustained figure is taken NOW, in the same thermal / power state, over one second
        (the pipe itself delivers 3.2-3.4 PTOP/s right after a long dense run against 3.8-3.9 from an idle board)."""
        burst, mhz_b = self.peak("tc_i8_n256", 2.0)
        capped = "sw_power_cap" in (clocks.get("reasons") or []) or (
            clocks.get("sm_mhz") and clocks.get("sm_max_mhz") and clocks["sm_mhz"] < 0.93 * clocks["sm_max_mhz"])
        if capped and hot:
            sust, mhz_s = self.L.measure_peak("tc_i8_n256", 1000.0)
            self._peak_cache[("tc_i8_n256 (hot, right after the leg)", 1000.0)] = (sust, mhz_s)
            skind = "sustained (1 s, measured right after the leg in the same power state)"
        else:
            sust, mhz_s = self.peak("tc_i8_n256", 400.0)
            skind = "sustained (400 ms)"
        use, mhz, kind = (sust, mhz_s, skind) if capped else (burst, mhz_b, "burst (2 ms)")
        return {"peak": use, "peak_kind": kind, "peak_sm_mhz": mhz,
                "peak_source": "measured live by linac_measure_peak('tc_i8_n256'): tcgen05.mma kind::i8 128x256x32 from "
                               "on-chip pseudo-random operands",
                "peak_burst": burst, "peak_burst_sm_mhz": mhz_b, "peak_sustained": sust, "peak_sustained_sm_mhz": mhz_s,
                "peak_2x_bf16_for_comparison": {"burst": 2 * self.peaks_file["bf16_burst"],
                                                "sustained": 2 * self.peaks_file["bf16_sustained"],
                                                "source": self.peaks_file["source"] + " x nominal int8:bf16 ratio 2"}}

    def fp_leg(self, name, steps, warmup, with_e2e=False, nullspace=False):
        """One F_p config through linac_rref_u32 (or linac_nullspace_u32): device-resident timing, clocks, production-
        schedule class split and the update roofline."""
        torch, L, dev = self.torch, self.L, self.dev
        from paper_2605_25863_b200 import replicas
        cfg = dict(gen.CONFIGS[name])
        on_device = cfg["kind"] == "sparse_dep"
        if on_device:
            from linac_inputs import gen_torch
            cfg["seed"] += 1000 * self.rank
            p, rows, cols = cfg["p"], cfg["rows"], cfg["cols"]
            d_work = torch.empty((rows, cols), dtype=torch.int32, device=dev)
            nbytes = rows * cols * 4
            pinned = d_in = out_host = None
            restore = lambda: gen_torch.fill_c5(d_work, cfg)            # noqa: E731  (NOT part of the step)
        else:
            a_host, p, cfg = make_workload(name, rank_seed=self.rank)
            rows, cols = a_host.shape
            nbytes = a_host.nbytes
            pinned = torch.from_numpy(a_host.view(np.int32)).pin_memory()
            d_in = pinned.to(dev, non_blocking=False)
            d_work = torch.empty_like(d_in)
            out_host = torch.empty_like(pinned).pin_memory() if with_e2e else None
            restore = lambda: d_work.copy_(d_in)                        # noqa: E731  (NOT part of the step)
        nominal = 2.0 * rows * cols * min(rows, cols) / 3.0
        stream = torch.cuda.current_stream(dev)

        def call(buf):
            if nullspace:
                rk, _, _ = L.nullspace_u32(buf, p)
                return rk
            return L.rref_u32(buf, p)[0]

        def step_resident():
            restore()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            rk = call(d_work)
            e1.record(stream)
            e1.synchronize()
            return e0.elapsed_time(e1), rk

        L.set_option("timing", 0)
        for _ in range(warmup):
            step_resident()
        sampler = ClockSampler(self.local).start()
        self.barrier()
        times, ranks = [], []
        for _ in range(steps):
            ms, rk = step_resident()
            times.append(ms)
            ranks.append(rk)
        self.barrier()
        clocks = sampler.stop()
        stats = L.last_stats()
        peak_info = self.tensor_peak(clocks, hot=True)          # right after the timed steps (same power state)
        total_ms = replicas.max_over_ranks(float(sum(times)), dev)
        ms_per_step = total_ms / steps
        value = replicas.aggregate_throughput(nominal, ms_per_step * 1e-3, self.world) / 1e9
        leg = {"workload": f"{name}: {rows}x{cols} uint32 {WORKLOAD_KIND[cfg['kind']]}, p={p}" +
                           (" + null space" if nullspace else ""),
               "ms_per_step": ms_per_step, "ms_min": float(min(times)), "value": value, "unit": "Gmulmod/s", "steps": steps,
               "warmup": warmup, "rank": int(ranks[-1]), "clocks": clocks, "gpu_launches_per_step": int(stats["kernel_launches"]),
               "us_per_pivot": ms_per_step * 1e3 / max(1, int(ranks[-1])),
               "l2": "input (%d MB) larger than L2" % (nbytes // 2 ** 20) if nbytes > 126 * 2 ** 20 else
                     "input fits L2; restored by a device copy before each step, outside the timed region",
               "stats": {k: stats[k] for k in ("kernel_launches", "host_syncs", "panels", "row_swaps", "update_macs")}}

        # production-schedule class split (timing = 2: event pairs, no host syncs) and the update roofline
        # (event pairs are enqueued by the host right around each launch: when the host falls behind the device an
        # interval also holds the idle gap, so the least perturbed of a few calls -- the shortest -- is kept)
        L.set_option("timing", 2)
        step_resident()
        ms_t, st_t = None, None
        for _ in range(1 if on_device else 5):
            ms_i, _ = step_resident()
            if ms_t is None or ms_i < ms_t:
                ms_t, st_t = ms_i, L.last_stats()
        # the update kernels on their own: the same code with look-ahead off (under look-ahead the bulk update shares the
        # GPU with the next strip kernel, so its launches are slower although the step is faster)
        st_alone = st_t
        if st_t.get("lookahead_strips", 0) > 0:
            L.set_option("lookahead", 0)
            ms_a = None
            for _ in range(1 if on_device else 3):
                ms_i, _ = step_resident()
                if ms_a is None or ms_i < ms_a:
                    ms_a, st_alone = ms_i, L.last_stats()
            L.set_option("lookahead", 1)
        L.set_option("timing", 0)
        macs, ms_upd = st_alone["update_macs"], st_alone["ms_update"]
        roof = {"bound": "tensor", "unit": "TOP/s (int8, 2 ops per u8 multiply-accumulate, 16 per field multiply-accumulate)",
                "kernel": "Schur-update GEMMs on tcgen05 kind::i8 (gemm_tc_panel_kernel for K <= 256, gemm_tc_kernel above; "
                          "the CUDA-core kernel only for shapes below 128)"}
        roof.update(peak_info)
        if st_t.get("tc_launches", 0) and ms_upd > 0:
            ach = macs * 32.0 / (ms_upd * 1e-3) / 1e12
            roof.update({"achieved": ach, "frac": ach / roof["peak"]})
        else:
            roof.update({"achieved": None, "frac": None})
        whole = nominal / 2.0 * 32.0 / (ms_per_step * 1e-3) / 1e12          # 2N^3/3 counts multiply AND add: N^3/3 field MACs
        roof["whole_step_achieved"] = whole
        roof["whole_step_frac"] = whole / roof["peak"]
        roof["update_share_of_step"] = ms_upd / st_alone["ms_total"] if st_alone["ms_total"] else None
        if st_alone is not st_t:
            roof["kernels_timed_alone"] = {"schedule": "look-ahead off (option lookahead = 0): every kernel has the whole GPU; trsm here is the chain kernel (the sequential sweep enqueues the solve before the host has the strip's records, so it cannot pick the tensor-core W product)",
                                           "update": st_alone["ms_update"], "strip": st_alone.get("ms_strip"),
                                           "trsm": st_alone.get("ms_trsm"), "call_with_event_marks": st_alone["ms_total"]}
            la_ach = st_t["update_macs"] * 32.0 / (st_t["ms_update"] * 1e-3) / 1e12 if st_t["ms_update"] > 0 else None
            roof["update_under_lookahead"] = {"achieved": la_ach, "frac": la_ach / roof["peak"] if la_ach else None,
                                              "note": "the same launches in the production schedule, sharing the SMs with the strip kernel"}
        roof["timed_split_ms"] = {"update": st_t["ms_update"], "strip": st_t.get("ms_strip"), "trsm": st_t.get("ms_trsm"),
                                  "call_with_event_marks": ms_t, "strip_and_update_in_flight_together": st_t.get("ms_overlap"),
                                  "lookahead_strips": st_t.get("lookahead_strips"),
                                  "schedule": "production (fused, look-ahead: the strip kernel of s+1 runs on a partition of the SMs beside "
                                              "the bulk update of s, so the classes overlap and their sum exceeds the call), event "
                                              "pairs, no host syncs"}
        roof["note"] = ("achieved = executed update field-MACs x 32 / summed CUDA-event time of the update launches (event pairs, no "
                        "host syncs; with look-ahead off, so that each launch has the whole GPU: kernels_timed_alone); frac = "
                        "achieved / peak; whole_step_* = (N^3/3 field MACs x 32) / ms_per_step of the production schedule (look-ahead "
                        "on) against the same peak")
        tm_, tn_, tk_ = st_alone.get("top_m", 0), st_alone.get("top_n", 0), st_alone.get("top_k", 0)
        if st_alone.get("ms_update_top", 0) > 0:
            kp_ = -(-tk_ // 128) * 128
            top = {"M": tm_, "N": tn_, "K": tk_, "ms": st_alone["ms_update_top"],
                   "achieved": 32.0 * tm_ * tn_ * tk_ / (st_alone["ms_update_top"] * 1e-3) / 1e12,
                   "algorithmic_bytes": 8 * tm_ * tn_ + 4 * kp_ * (tm_ + tn_),
                   "algorithmic_bytes_note": "C read + C written (8 B per element) + both u8 limb-plane operands read once"}
            top["frac"] = top["achieved"] / roof["peak"]
            top["hbm_gbs_at_algorithmic_bytes"] = top["algorithmic_bytes"] / (top["ms"] * 1e-3) / 1e9
            roof["top_launch"] = top
        roof["traffic"] = None
        if os.path.exists(TRAFFIC_FILE):
            tr = json.load(open(TRAFFIC_FILE)).get(name)
            if tr:
                roof["traffic"] = tr["dram_bytes"]
                roof["traffic_source"] = tr["source"]
        leg["roofline"] = roof

        if with_e2e and not on_device:
            def step_e2e():
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                d_work.copy_(pinned, non_blocking=True)
                rk = call(d_work)
                out_host.copy_(d_work, non_blocking=True)
                e1.record(stream)
                e1.synchronize()
                return e0.elapsed_time(e1), rk

            def run_pipelined(k_steps):
                """K end-to-end steps, pipelined: while the call of step k runs, the pinned H2D of step k+1 and the
                D2H of step k-1 are in flight on their own streams; every step's copies are inside the timed region."""
                s_c, s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev), torch.cuda.Stream(dev)
                # three device buffers: with two, the D2H of step k-1 and the H2D of step k+1 use the same buffer one after
                # the other and their sum (14 ms at c3), not the call (13.5 ms), sets the period
                NB = 3
                bufs = [d_work] + [torch.empty_like(d_work) for _ in range(NB - 1)]
                outs = [out_host, torch.empty_like(out_host).pin_memory()]
                ev_in = [torch.cuda.Event() for _ in range(NB)]
                ev_done = [torch.cuda.Event() for _ in range(NB)]
                ev_out = [torch.cuda.Event() for _ in range(NB)]
                t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize(dev)
                t0.record(s_in)
                with torch.cuda.stream(s_in):
                    bufs[0].copy_(pinned, non_blocking=True)
                    ev_in[0].record(s_in)
                rk = None
                for k in range(k_steps):
                    b = k % NB
                    if k + 1 < k_steps:
                        nb = (k + 1) % NB
                        if k + 1 >= NB:
                            s_in.wait_event(ev_out[nb])                 # the D2H of step k + 1 - NB has left this buffer
                        with torch.cuda.stream(s_in):
                            bufs[nb].copy_(pinned, non_blocking=True)
                            ev_in[nb].record(s_in)
                    s_c.wait_event(ev_in[b])
                    with torch.cuda.stream(s_c):
                        rk = call(bufs[b])
                        ev_done[b].record(s_c)
                    s_out.wait_event(ev_done[b])
                    with torch.cuda.stream(s_out):
                        outs[k % 2].copy_(bufs[b], non_blocking=True)
                        ev_out[b].record(s_out)
                t1.record(s_out)
                t1.synchronize()
                torch.cuda.synchronize(dev)
                return t0.elapsed_time(t1) / k_steps, rk

            step_e2e()
            self.barrier()
            serial = [step_e2e()[0] for _ in range(max(2, min(steps, 3)))]
            self.barrier()
            serial_ms = replicas.max_over_ranks(float(np.mean(serial)), dev)
            run_pipelined(2)
            self.barrier()
            e2e_ms, rk_p = run_pipelined(max(12, steps))
            assert rk_p == ranks[-1]
            self.barrier()
            e2e_ms = replicas.max_over_ranks(float(e2e_ms), dev)
            leg["e2e"] = {"value": replicas.aggregate_throughput(nominal, e2e_ms * 1e-3, self.world) / 1e9, "unit": "Gmulmod/s",
                          "ms_per_step": e2e_ms, "h2d_bytes_per_step": int(nbytes), "d2h_bytes_per_step": int(nbytes),
                          "mode": "pipelined over three device buffers: the pinned H2D of step k+1 and the D2H of step k-1 overlap "
                                  "the call of step k; every step's copies are inside the timed region",
                          "serial_ms_per_step": serial_ms,
                          "serial_value": replicas.aggregate_throughput(nominal, serial_ms * 1e-3, self.world) / 1e9}
        else:
            leg["e2e"] = {"value": None, "unit": "Gmulmod/s", "ms_per_step": None, "h2d_bytes_per_step": 0,
                          "d2h_bytes_per_step": 0,
                          "note": "not measured: generated on the device (40 GB)" if on_device else "not measured for this leg"}
        del d_work
        torch.cuda.empty_cache()
        return leg

    def f64_solve_leg(self, n=16384, nrhs=64, reps=3):
        """Config c4 through linac_solve_f64: A = G + 4 sqrt(N) I, G i.i.d. N(0,1), 64 N(0,1) right-hand sides, drawn on the
        device from a seeded torch generator (same distribution as linac_inputs' c4 recipe, whose numpy generator takes
        half a minute on the host).  Backward error in the infinity norm on the ORIGINAL data with torch fp64 products
        (cuBLAS; a bench-side check only -- the parity tests use the oracle's long-double residual)."""
        torch, L, dev = self.torch, self.L, self.dev
        g = torch.Generator(device=dev)
        g.manual_seed(5)
        a0 = torch.randn((n, n), dtype=torch.float64, device=dev, generator=g)
        a0.diagonal().add_(4.0 * n ** 0.5)
        b0 = torch.randn((n, nrhs), dtype=torch.float64, device=dev, generator=g)
        a, b = torch.empty_like(a0), torch.empty_like(b0)
        stream = torch.cuda.current_stream(dev)
        times = []
        sampler = None
        for i in range(reps + 1):
            a.copy_(a0)
            b.copy_(b0)
            if i == 1:
                sampler = ClockSampler(self.local).start()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            L.solve_f64(a, b)
            e1.record(stream)
            e1.synchronize()
            if i:
                times.append(e0.elapsed_time(e1))
        clocks = sampler.stop()
        launches = L.last_stats()["kernel_launches"]
        resid = (a0 @ b - b0).abs().amax(dim=0)
        eta = float((resid / (a0.abs().sum(dim=1).max() * b.abs().amax(dim=0) + b0.abs().amax(dim=0))).max())
        ms = float(np.mean(times))
        flop = 2.0 * n ** 3 / 3.0 + 2.0 * n * n * nrhs
        peak, mhz = self.peak("dmma", 20.0)
        del a0, b0, a, b
        torch.cuda.empty_cache()
        return {"workload": f"c4: {n}x{n} float64 N(0,1) + 4 sqrt(N) I, {nrhs} right-hand sides (torch generator on the device, "
                            "seed 5; eta checked with torch fp64 products)",
                "ms_per_solve": ms, "gflops": flop / ms / 1e6, "backward_error": eta, "backward_error_bound": 1e-11,
                "clocks": clocks, "gpu_launches_per_solve": int(launches),
                "roofline": {"bound": "tensor", "achieved": flop / ms / 1e9, "peak": peak, "unit": "TFLOP/s (fp64 DMMA)",
                             "frac": flop / ms / 1e9 / peak, "peak_sm_mhz": mhz,
                             "peak_source": "measured live by linac_measure_peak('dmma'): mma.sync m8n8k4 f64 from registers",
                             "note": "whole solve (panel chain, exchanges and substitutions included) against the FP64 tensor pipe"},
                "note": "flop = 2N^3/3 + 2N^2 nrhs"}

    def rref_f64_leg(self, rows=8192, cols=8192, r=6144, reps=2):
        """linac_rref_f64 on a rank-deficient product (rows x r).(r x cols) of N(0,1) factors with rows
        rescaled over several decades; flop count of the blocked Gauss-Jordan that runs: 2 rows cols rank / ... stated."""
        torch, L, dev = self.torch, self.L, self.dev
        g = torch.Generator(device=dev)
        g.manual_seed(9)
        a0 = torch.randn((rows, r), dtype=torch.float64, device=dev, generator=g) @ \
            torch.randn((r, cols), dtype=torch.float64, device=dev, generator=g)
        a0 *= 10.0 ** (2.0 * torch.randn((rows, 1), dtype=torch.float64, device=dev, generator=g))
        a = torch.empty_like(a0)
        stream = torch.cuda.current_stream(dev)
        times, rk = [], None
        for i in range(reps + 1):
            a.copy_(a0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            rk, piv = L.rref_f64(a, 1e-9)
            e1.record(stream)
            e1.synchronize()
            if i:
                times.append(e0.elapsed_time(e1))
        launches = L.last_stats()["kernel_launches"]
        pv = piv.to(dev).long()
        recon = a0[:, pv] @ a[:rk]
        err = float(((recon - a0).abs().amax(dim=1) / a0.abs().amax(dim=1)).max())
        ms = float(np.mean(times))
        # executed: every panel updates all rows on the columns from the panel on: sum_j 2 rows (cols - j) 32 ~ rows cols^2
        flop = float(sum(2.0 * rows * (cols - j0) * 32 for j0 in range(0, cols, 32) if j0 < rk + 32))
        peak, mhz = self.peak("dmma", 20.0)
        del a0, a
        torch.cuda.empty_cache()
        return {"workload": f"rref_f64: {rows}x{cols} float64, rank {r} product of N(0,1) factors, rows rescaled by 10^(2 N(0,1)), "
                            "tol 1e-9", "ms_per_call": ms, "rank": int(rk), "gflops_executed": flop / ms / 1e6,
                "row_space_residual": err, "gpu_launches_per_call": int(launches),
                "roofline": {"bound": "tensor", "achieved": flop / ms / 1e9, "peak": peak, "unit": "TFLOP/s (fp64 DMMA)",
                             "frac": flop / ms / 1e9 / peak, "peak_sm_mhz": mhz,
                             "note": "executed flops of the DMMA updates (2 rows (cols - j0) 32 per panel: K = 32 inside the panel's 128-column strip, K = 128 right of it) / whole call"}}

    def rref_c128_leg(self, rows=4096, cols=4096, r=3072, reps=2):
        """SURVEY.md 8(f)#3, complex128: linac_rref_c128 on a rank-deficient complex product with rows rescaled over several
        decades and rotated by arbitrary phases.  The GPU reduces the 2 rows x 2 cols real embedding, so the flops that run
        are those of linac_rref_f64 at that shape: twice what a native complex elimination needs (stated in the note)."""
        torch, L, dev = self.torch, self.L, self.dev
        g = torch.Generator(device=dev)
        g.manual_seed(10)
        def cn(m, n):
            return torch.complex(torch.randn((m, n), dtype=torch.float64, device=dev, generator=g),
                                 torch.randn((m, n), dtype=torch.float64, device=dev, generator=g))
        a0 = cn(rows, r) @ cn(r, cols)
        a0 *= 10.0 ** (2.0 * torch.randn((rows, 1), dtype=torch.float64, device=dev, generator=g))
        a0 *= torch.exp(2j * np.pi * torch.rand((rows, 1), dtype=torch.float64, device=dev, generator=g))
        a = torch.empty_like(a0)
        stream = torch.cuda.current_stream(dev)
        times, rk = [], None
        for i in range(reps + 1):
            a.copy_(a0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            rk, piv = L.rref_c128(a, 1e-9)
            e1.record(stream)
            e1.synchronize()
            if i:
                times.append(e0.elapsed_time(e1))
        launches = L.last_stats()["kernel_launches"]
        pv = piv.to(dev).long()
        recon = a0[:, pv] @ a[:rk]
        err = float(((recon - a0).abs().amax(dim=1) / a0.abs().amax(dim=1)).max())
        ms = float(np.mean(times))
        R, Cc, rk2 = 2 * rows, 2 * cols, 2 * rk
        flop = float(sum(2.0 * R * (Cc - j0) * 32 for j0 in range(0, Cc, 32) if j0 < rk2 + 32))
        peak, mhz = self.peak("dmma", 20.0)
        del a0, a
        torch.cuda.empty_cache()
        return {"workload": f"rref_c128: {rows}x{cols} complex128, rank {r} product of complex N(0,1) factors, rows rescaled by "
                            "10^(2 N(0,1)) and rotated by random phases, tol 1e-9", "ms_per_call": ms, "rank": int(rk),
                "gflops_executed": flop / ms / 1e6, "row_space_residual": err, "gpu_launches_per_call": int(launches),
                "roofline": {"bound": "tensor", "achieved": flop / ms / 1e9, "peak": peak, "unit": "TFLOP/s (fp64 DMMA)",
                             "frac": flop / ms / 1e9 / peak, "peak_sm_mhz": mhz,
                             "note": "executed real flops of the DMMA updates on the 2 rows x 2 cols embedding (2x the real "
                                     "flops of a native complex elimination, which needs 4 real multiply-adds per complex one "
                                     "where the embedding spends 8) / whole call incl. the expand and contract kernels"}}

    def wide_leg(self, which, n=4096, reps=2):
        """dense uniform n x n over F_p with p = 2^32 - 5 (uint32 storage) or 2^61 - 1 (uint64)."""
        torch, L, dev = self.torch, self.L, self.dev
        if which == "u32":
            p = 4294967291
            a0 = torch.from_numpy(gen.uniform_matrix(n, n, p, seed=4).view(np.int32)).to(dev)
            fn = L.rref_u32
        else:
            p = (1 << 61) - 1
            a0 = torch.from_numpy(gen.uniform_matrix_u64(n, n, p, seed=4).view(np.int64)).to(dev)
            fn = L.rref_u64
        a = torch.empty_like(a0)
        stream = torch.cuda.current_stream(dev)
        times, rk = [], None
        for i in range(reps + 1):
            a.copy_(a0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            rk, _ = fn(a, p)
            e1.record(stream)
            e1.synchronize()
            if i:
                times.append(e0.elapsed_time(e1))
        st = L.last_stats()
        ms = float(np.mean(times))
        imad, mhz = self.peak("imad_wide", 20.0)
        macs = float(st["update_macs"])
        # 32 x 32 -> 64-bit multiplies per field multiply-accumulate of the lazily reduced update (cuobjdump of
        # wide_update_kernel's inner loop): u32: one IMAD.WIDE (+ the carry additions the peak kernel also pays);
        # u64: the 128-bit product = 5 IMAD.WIDE + 2 IMAD (counted as half a wide multiply each)
        per_mac = 1.0 if which == "u32" else 6.0
        del a0, a
        torch.cuda.empty_cache()
        return {"workload": f"wide_{which}: {n}x{n} dense uniform, p={p}", "ms_per_call": ms, "rank": int(rk),
                "value": (2.0 * n ** 3 / 3.0) / (ms * 1e-3) / 1e9, "unit": "Gmulmod/s (2N^3/3)",
                "executed_tmacs_per_s": macs / (ms * 1e-3) / 1e12, "gpu_launches_per_call": int(st["kernel_launches"]),
                "roofline": {"bound": "alu", "achieved": macs * per_mac / (ms * 1e-3) / 1e12, "peak": imad,
                             "unit": "T 32x32->64-bit multiply-adds/s (thread level)", "peak_sm_mhz": mhz,
                             "frac": macs * per_mac / (ms * 1e-3) / 1e12 / imad,
                             "peak_source": "measured live by linac_measure_peak('imad_wide')",
                             "note": f"achieved = executed field MACs (rows x cols-from-panel x 32 per panel, Gauss-Jordan over all "
                                     f"rows) x {per_mac:g} wide multiplies per multiply-accumulate (raw products summed in a 96 / 192-bit "
                                     f"accumulator, one Montgomery reduction per output and panel) / whole call"}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="all", choices=["all", "c1", "c2", "c3", "c5"],
                    help="all (default): headline c3 + one leg per other config; or a single F_p config as the headline")
    ap.add_argument("--legs", default="c1,c2,c5,fp64_solve,rref_f64,rref_c128,wide_u32,wide_u64",
                    help="comma list of the extra legs of the default run")
    ap.add_argument("--ref-n", type=int, default=1280, help="sample size for --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--cpu-baseline", default="bounded", choices=["bounded", "full"])
    ap.add_argument("--no-f64", action="store_true", help="skip the fp64 legs")
    ap.add_argument("--fp64-only", action="store_true", help="run only legs.fp64_solve and print {\"fp64\": ...}")
    ap.add_argument("--only-leg", default="", choices=["", "rref_f64", "rref_c128", "wide_u32", "wide_u64"],
                    help="run only this leg of the widened rows (SURVEY.md 8(f)) and print {name: ...}; for profiles")
    ap.add_argument("--gemm", default=None, metavar="M,N,K[,path]",
                    help="time the S5 primitive linac_gemm_sub_u32 alone (C -= A.B mod 2^31-1, path 2 = tensor cores by default) "
                         "and print {\"gemm\": ...}; the command of the GEMM ncu captures under profiles/")
    ap.add_argument("--load-matrix", default=None, metavar="ROWS,COLS,D",
                    help="time linac_load_matrix_u32 alone (SURVEY.md 8(f)#2) and print {\"load_matrix\": ...}")
    ap.add_argument("--timeline", default=None, metavar="N",
                    help="one linac_rref_u32 call on an N x N dense matrix with option timing = 2 and print its per-launch intervals "
                         "(linac_get_last_marks) as a table: which strip kernel ran beside which update (profiles/r02_lookahead.md)")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="library tunable for A/B runs (linac_set_option), e.g. --opt strip_width=256")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2605_25863_b200 as L

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    for kv in args.opt:
        name, _, val = kv.partition("=")
        L.set_option(name, int(val))
    B = Bench(torch, L, dev, local, world, rank, args.opt)
    if args.timeline:
        n = int(args.timeline)
        p = 2147483647
        from linac_inputs import gen_torch
        a0 = gen_torch.uniform_rows(0, n, n, p, 3, dev)
        L.set_option("timing", 2)
        for _ in range(3):                                   # the last call's marks are the ones printed
            a = a0.clone()
            rk, _ = L.rref_u32(a, p)
        L.set_option("timing", 0)
        marks = sorted(L.last_marks(), key=lambda mk: mk["t0_ms"])
        names = {0: "update", 1: "strip", 2: "solve"}
        print(f"# linac_rref_u32 {n} x {n}, p = {p}, rank {rk}: {len(marks)} launches, call {L.last_stats()['ms_total']:.3f} ms (with the event marks)")
        print("# start_us end_us dur_us class stream shape(update: M N K)")
        for mk in marks:
            shape = f"{mk['m']} {mk['n']} {mk['k']}" if mk["cls"] == 0 else ""
            print(f"{mk['t0_ms'] * 1e3:9.1f} {mk['t1_ms'] * 1e3:9.1f} {(mk['t1_ms'] - mk['t0_ms']) * 1e3:7.1f} {names[mk['cls']]:6s} "
                  f"{'second' if mk['stream'] else 'call'  :6s} {shape}")
        return
    if args.gemm:
        parts = [int(x) for x in args.gemm.split(",")]
        m, n, k = parts[:3]
        path = parts[3] if len(parts) > 3 else 2
        p = 2147483647
        from linac_inputs import gen_torch
        a = gen_torch.uniform_rows(0, m, k, p, 1, dev)
        b = gen_torch.uniform_rows(0, k, n, p, 2, dev)
        c = gen_torch.uniform_rows(0, m, n, p, 3, dev)
        times = []
        for i in range(args.warmup + min(args.steps, 5)):
            L.gemm_sub_u32(c, a, b, p, path)
            if i >= args.warmup:
                times.append(L.last_stats()["ms_total"])
        ms = float(np.mean(times))
        clk = {"sm_mhz": None, "reasons": []}
        peak = B.tensor_peak(clk)
        ach = 32.0 * m * n * k / (ms * 1e-3) / 1e12
        print(json.dumps({"gemm": {"M": m, "N": n, "K": k, "path": path, "ms": ms, "achieved_tops": ach,
                                   "field_tmacs_per_s": ach / 32.0, "frac_of_burst_peak": ach / peak["peak_burst"],
                                   "peak_burst": peak["peak_burst"], "peak_sustained": peak["peak_sustained"],
                                   "note": "event time of the whole call incl. the limb-split pre-passes"}}))
        return
    if args.load_matrix:
        rows, cols, d = (int(x) for x in args.load_matrix.split(","))
        p, nb = 2147483647, 64
        from linac_inputs import gen_torch
        bases = gen_torch.uniform_rows(0, rows, nb, p, 11, dev)
        lind = (gen_torch.uniform_rows(0, cols, d, nb, 12, dev)).to(torch.int32).contiguous()
        out_t = torch.empty((rows, cols), dtype=torch.int32, device=dev)
        stream = torch.cuda.current_stream(dev)
        times = []
        for i in range(args.warmup + min(args.steps, 5)):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            L.load_matrix_u32(bases, lind, p, out=out_t)
            e1.record(stream)
            e1.synchronize()
            if i >= args.warmup:
                times.append(e0.elapsed_time(e1))
        ms = float(np.mean(times))
        imad, mhz = B.peak("imad_wide", 20.0)
        print(json.dumps({"load_matrix": {"rows": rows, "cols": cols, "d": d, "n_basis": nb, "ms": ms,
                                          "gb_per_s_written": rows * cols * 4 / (ms * 1e-3) / 1e9,
                                          "field_products_per_s_T": rows * cols * d / (ms * 1e-3) / 1e12,
                                          "imad_wide_peak_T": imad, "hbm_peak_gbs": B.peaks_file["hbm_gbs"],
                                          "note": "d Montgomery products (IMAD.WIDE + IMAD + IMAD.WIDE each) per 4-byte element: "
                                                  "ALU-bound, not HBM-bound, for d >= 2"}}))
        return
    if args.fp64_only:
        if rank == 0:
            print(json.dumps({"fp64": B.f64_solve_leg(reps=max(1, min(args.steps, 5)))}))
        return
    if args.only_leg:
        if rank == 0:
            reps = max(1, min(args.steps, 3))
            leg = {"rref_f64": lambda: B.rref_f64_leg(reps=reps), "rref_c128": lambda: B.rref_c128_leg(reps=reps), "wide_u32": lambda: B.wide_leg("u32", reps=reps),
                   "wide_u64": lambda: B.wide_leg("u64", reps=reps)}[args.only_leg]()
            print(json.dumps({args.only_leg: leg}))
        return

    headline = "c3" if args.workload == "all" else args.workload
    if headline == "c5":
        h = B.fp_leg("c5", steps=min(args.steps, 2), warmup=min(args.warmup, 1))
        args.steps, args.warmup = h["steps"], h["warmup"]
    else:
        h = B.fp_leg(headline, steps=args.steps, warmup=args.warmup, with_e2e=not args.no_e2e, nullspace=(headline == "c2"))
    out = {
        "metric": "rref_gmulmod_per_s", "value": h["value"], "unit": "Gmulmod/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": h["ms_per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": h["workload"], "rank": h["rank"], "parallelism": "replicas" if world > 1 else "single",
                   "l2": h["l2"], "options": args.opt},
        "e2e": h["e2e"], "gpu_launches": h["gpu_launches_per_step"] * args.steps, "clocks": h["clocks"],
        "roofline": h["roofline"], "stats": h["stats"], "us_per_pivot": h["us_per_pivot"],
        "baseline_context": BASELINE_CONTEXT,
    }
    if rank == 0 and world == 1 and args.workload == "all":
        legs = {}
        want = [x for x in args.legs.split(",") if x]
        for name in want:
            try:
                if name == "c1":
                    legs[name] = B.fp_leg("c1", steps=20, warmup=3, with_e2e=True)
                elif name == "c2":
                    legs[name] = B.fp_leg("c2", steps=10, warmup=3, with_e2e=True, nullspace=True)
                elif name == "c5":
                    free_b, _ = torch.cuda.mem_get_info()
                    if free_b < 60e9:
                        legs[name] = {"skipped": "needs about 60 GB of free device memory"}
                    else:
                        legs[name] = B.fp_leg("c5", steps=2, warmup=1)
                elif name == "fp64_solve" and not args.no_f64:
                    legs[name] = B.f64_solve_leg()
                elif name == "rref_f64" and not args.no_f64:
                    legs[name] = B.rref_f64_leg()
                elif name == "rref_c128" and not args.no_f64:
                    legs[name] = B.rref_c128_leg()
                elif name == "wide_u32":
                    legs[name] = B.wide_leg("u32")
                elif name == "wide_u64":
                    legs[name] = B.wide_leg("u64")
            except Exception as e:                       # a failed leg must not lose the headline line
                legs[name] = {"error": f"{type(e).__name__}: {e}"}
        out["legs"] = legs
        if "fp64_solve" in legs:
            out["fp64"] = legs["fp64_solve"]
        out["measured_peaks_live"] = {f"{k[0]}@{k[1]:g}ms": {"value": v[0], "sm_mhz": v[1]} for k, v in B._peak_cache.items()}
    if rank == 0 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline_plan(gen.CONFIGS[headline]["p"], full=(args.cpu_baseline == "full"))
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
