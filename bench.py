#!/usr/bin/env python
"""bench.py -- one JSON line for the Linac hot path on B200 (contract: see DESIGN.md "Measurement").

A "step" is one pass of the whole hot path (S0 ingest .. S7 finalise) over one
seeded synthetic matrix of the workload BASELINE.json's metric is quoted on: config c3, the
paper's N = 10^4 point (dense uniform over F_{2^31-1}).  `--workload c2|c5|...`
selects another config; the default finishes in well under a minute.

  value      : whole-job Gmulmod/s = (2 N^3 / 3) / t, matrix already resident in HBM, t = CUDA-event
               time of the C-ABI call (max over ranks); N > 1 runs independent replicas (weak).
  e2e        : same metric with HOST buffers: pinned H2D of the matrix + call + D2H of the RREF every step, double
               buffered (the copies of neighbouring steps overlap the call); the strictly serial figure is kept
               beside it as e2e.serial_ms_per_step.
  roofline   : the Schur-update kernel (dominant): executed field MACs / its event-timed duration.
  cpu_baseline: the CPU oracle timed on a bounded sample on this box's host cores.
  fp64       : (default workload only) linac_solve_f64 on config c4: ms per solve, GFLOP/s, backward error.
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

#: ncu --set full, gemm_tc_panel_kernel, second launch of a c3 call (profiles/r01_v9_launches_c3.md)
NCU_TOP_LAUNCH_DRAM_BYTES_C3 = 396063488 + 324826368

PAPER_A100_GMULMOD = {"c3": (2 * 1e4 ** 3 / 3) / 3.6 / 1e9,            # PAPER.md:59  (3.6 s at N = 10^4)
                      "c5": (2 * 1e5 ** 3 / 3) / (45 * 60) / 1e9}       # PAPER.md:61  (45 min at N = 10^5)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm_gbs=d["hbm_gbs"], bf16_burst=d["bf16_tflops"], bf16_sustained=d["bf16_tflops_sustained"],
                    sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="measured")
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

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i] == "Active"})
        busy = [x for x in sm if x > 0.6 * (max(mx) if mx else 1)] or sm
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def make_workload(name: str, rank_seed: int = 0):
    """Returns (host uint32 matrix, p, description).  rank_seed shifts the seed for replicas."""
    c = dict(gen.CONFIGS[name])
    if c["kind"] == "uniform":
        a = gen.uniform_matrix(c["rows"], c["cols"], c["p"], c["seed"] + 1000 * rank_seed)  # == replicas.replica_seed
    elif c["kind"] == "lowrank":
        a, _, _ = gen.lowrank_factors(c["rows"], c["inner"], c["cols"], c["p"], c["seed_b"] + 1000 * rank_seed, c["seed_c"])
    elif c["kind"] == "sparse_dep":
        raise SystemExit("workload c5 is generated on the device: use --workload c5 (handled separately)")
    else:
        raise SystemExit(f"workload {name} is not an F_p RREF config")
    return a, c["p"], c


def oracle_sample_gmulmod(n: int, p: int, threads: int):
    """Times the CPU oracle (as it stands) on an n x n dense uniform matrix; returns (Gmulmod/s, seconds)."""
    import oracle
    a = gen.uniform_matrix(n, n, p, seed=4)
    t0 = time.perf_counter()
    _, rank, _ = oracle.rref_modp(a, p, nthreads=threads)
    dt = time.perf_counter() - t0
    assert rank == n
    return (2 * n ** 3 / 3) / dt / 1e9, dt


def f64_leg(torch, L, dev, n=16384, nrhs=64, reps=3):
    """The metric's second half ("fp64 GFLOP/s"): linac_solve_f64 on config c4's shape and distribution
    (A = G + 4 sqrt(N) I with G i.i.d. N(0,1), 64 N(0,1) right-hand sides), drawn on the device from a seeded torch
    generator (the numpy recipe of linac_inputs takes half a minute on the host); the solve works in place, so every
    repetition restores A and B by a device copy outside the timed region.  Backward error in the infinity norm on
    the ORIGINAL data, computed with torch fp64 on the device."""
    g = torch.Generator(device=dev)
    g.manual_seed(5)
    a0 = torch.randn((n, n), dtype=torch.float64, device=dev, generator=g)
    a0.diagonal().add_(4.0 * n ** 0.5)
    b0 = torch.randn((n, nrhs), dtype=torch.float64, device=dev, generator=g)
    a, b = torch.empty_like(a0), torch.empty_like(b0)
    stream = torch.cuda.current_stream(dev)
    times = []
    for i in range(reps + 1):
        a.copy_(a0)
        b.copy_(b0)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        L.solve_f64(a, b)
        e1.record(stream)
        e1.synchronize()
        if i:
            times.append(e0.elapsed_time(e1))
    resid = (a0 @ b - b0).abs().amax(dim=0)
    eta = float((resid / (a0.abs().sum(dim=1).max() * b.abs().amax(dim=0) + b0.abs().amax(dim=0))).max())
    ms = float(np.mean(times))
    flop = 2.0 * n ** 3 / 3.0 + 2.0 * n * n * nrhs
    return {"workload": f"c4: {n}x{n} float64 N(0,1) + 4 sqrt(N) I, {nrhs} right-hand sides (torch generator, seed 5)",
            "ms_per_solve": ms, "gflops": flop / ms / 1e6, "backward_error": eta, "backward_error_bound": 1e-11,
            "roofline": {"bound": "tensor", "achieved": flop / ms / 1e9, "peak": 36.9, "unit": "TFLOP/s (fp64 DMMA)",
                         "frac": flop / ms / 1e9 / 36.9,
                         "note": "whole solve (panel chain and solves included) against the FP64 tensor pipe: 148 SMs x 64 "
                                 "FMA/clk x 2 x 1.95 GHz, consistent with ncu (78 % sub-pipe utilisation at 28.8 TFLOP/s on "
                                 "the largest update, profiles/r01_v13_dmma_top_ncu.md) and with cuBLAS DGEMM measured at "
                                 "36.0 TFLOP/s on this pool"},
            "note": "flop = 2N^3/3 + 2N^2 nrhs; trailing update on the FP64 tensor pipe (DMMA m8n8k4), substitution with "
                    "inverted 128 x 128 diagonal blocks"}


def run_reference(args):
    """--impl reference: the oracle on the host cores, a bounded sample of the same workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    threads = oracle.max_threads()
    n = args.ref_n
    p = gen.CONFIGS[args.workload].get("p", 2147483647)
    for _ in range(args.warmup):
        oracle_sample_gmulmod(min(n, 512), p, threads)
    times = []
    for _ in range(args.steps):
        _, dt = oracle_sample_gmulmod(n, p, threads)
        times.append(dt)
    t = float(np.mean(times))
    val = (2 * n ** 3 / 3) / t / 1e9
    sample = f"{n}x{n} dense uniform F_p sample of workload {args.workload}, CPU oracle Gauss-Jordan"
    print(json.dumps({
        "impl": "reference", "metric": "rref_gmulmod_per_s", "value": val, "unit": "Gmulmod/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": args.workload, "sample": sample},
        "cpu_baseline": {"value": val, "unit": "Gmulmod/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "Gmulmod/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3", choices=["c1", "c2", "c3", "c5"])
    ap.add_argument("--ref-n", type=int, default=1280, help="sample size for the oracle legs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-f64", action="store_true", help="skip the fp64 leg (config c4) of the default run")
    ap.add_argument("--fp64-only", action="store_true",
                    help="run only the fp64 leg (config c4) and print {\"fp64\": ...}; the command of the fp64 launch list")
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
    if args.fp64_only:
        for kv in args.opt:
            name, _, val = kv.partition("=")
            L.set_option(name, int(val))
        if rank == 0:
            print(json.dumps({"fp64": f64_leg(torch, L, dev, reps=max(1, min(args.steps, 5)))}))
        return

    from paper_2605_25863_b200 import replicas
    on_device = gen.CONFIGS[args.workload]["kind"] == "sparse_dep"     # c5: 40 GB, generated straight into HBM
    if on_device:
        from linac_inputs import gen_torch
        cfg = dict(gen.CONFIGS[args.workload])
        cfg["seed"] += 1000 * rank
        p, rows, cols = cfg["p"], cfg["rows"], cfg["cols"]
        a_host = pinned = out_host = d_in = None
        d_work = torch.empty((rows, cols), dtype=torch.int32, device=dev)
        nbytes = rows * cols * 4
    else:
        a_host, p, cfg = make_workload(args.workload, rank_seed=rank)      # replicas: one matrix per rank
        rows, cols = a_host.shape
        nbytes = a_host.nbytes
        pinned = torch.from_numpy(a_host.view(np.int32)).pin_memory()
        d_in = pinned.to(dev, non_blocking=False)
        d_work = torch.empty_like(d_in)
        out_host = torch.empty_like(pinned).pin_memory()
    n_nominal = 2.0 * rows * cols * min(rows, cols) / 3.0              # 2N^3/3 for square N
    stream = torch.cuda.current_stream(dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize(dev)

    def step_resident():
        if on_device:
            gen_torch.fill_c5(d_work, cfg)        # regenerate the input: NOT part of the step
        else:
            d_work.copy_(d_in)                    # restore the input: NOT part of the step
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        rank_, _ = L.rref_u32(d_work, p)
        e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1), rank_

    def step_e2e():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        d_work.copy_(pinned, non_blocking=True)   # H2D of this step's input
        rank_, piv = L.rref_u32(d_work, p)
        out_host.copy_(d_work, non_blocking=True)  # D2H of the RREF
        e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1), rank_

    def run_e2e_pipelined(k_steps):
        """K end-to-end steps, double buffered: while the call of step k runs, the pinned H2D of step k+1 and the
        D2H of step k-1 are in flight on their own streams.  Every step still copies its input from pinned host
        memory and reads its RREF back; all of it inside the timed region (events across the three streams)."""
        s_c, s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        bufs = [d_work, torch.empty_like(d_work)]
        outs = [out_host, torch.empty_like(out_host).pin_memory()]
        ev_in = [torch.cuda.Event(), torch.cuda.Event()]
        ev_done = [torch.cuda.Event(), torch.cuda.Event()]
        ev_out = [torch.cuda.Event(), torch.cuda.Event()]
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        t0.record(s_in)
        with torch.cuda.stream(s_in):
            bufs[0].copy_(pinned, non_blocking=True)
            ev_in[0].record(s_in)
        rk = None
        for k in range(k_steps):
            b = k % 2
            if k + 1 < k_steps:
                nb = (k + 1) % 2
                if k >= 1:
                    s_in.wait_event(ev_out[nb])          # buffer nb is free once step k-1's result has left it
                with torch.cuda.stream(s_in):
                    bufs[nb].copy_(pinned, non_blocking=True)
                    ev_in[nb].record(s_in)
            s_c.wait_event(ev_in[b])
            with torch.cuda.stream(s_c):
                rk, _ = L.rref_u32(bufs[b], p)           # returns when the RREF is complete on s_c
                ev_done[b].record(s_c)
            s_out.wait_event(ev_done[b])
            with torch.cuda.stream(s_out):
                outs[b].copy_(bufs[b], non_blocking=True)
                ev_out[b].record(s_out)
        t1.record(s_out)
        t1.synchronize()
        torch.cuda.synchronize(dev)
        return t0.elapsed_time(t1) / k_steps, rk

    L.set_option("timing", 0)
    for kv in args.opt:
        name, val = kv.split("=")
        L.set_option(name, int(val))
    for _ in range(args.warmup):
        step_resident()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    times, ranks = [], []
    for _ in range(args.steps):
        ms, rk = step_resident()
        times.append(ms)
        ranks.append(rk)
    barrier()
    clocks = sampler.stop()
    stats = L.last_stats()
    total_ms = float(sum(times))
    total_ms = replicas.max_over_ranks(total_ms, dev)
    ms_per_step = total_ms / args.steps
    value = replicas.aggregate_throughput(n_nominal, ms_per_step * 1e-3, world) / 1e9

    # end-to-end leg (host buffers; not run for the device-generated 40 GB config)
    e2e_ms = e2e_value = None
    if not on_device:
        step_e2e()
        barrier()
        e2e_times = [step_e2e()[0] for _ in range(max(2, min(args.steps, 3)))]
        barrier()
        e2e_serial_ms = replicas.max_over_ranks(float(np.mean(e2e_times)), dev)
        run_e2e_pipelined(2)
        barrier()
        e2e_ms, rk_p = run_e2e_pipelined(max(12, args.steps))
        assert rk_p == ranks[-1]
        barrier()
        e2e_ms = replicas.max_over_ranks(float(e2e_ms), dev)
        e2e_value = replicas.aggregate_throughput(n_nominal, e2e_ms * 1e-3, world) / 1e9

    # roofline of the dominant kernel family (Schur update), event-timed launch by launch
    L.set_option("timing", 1)
    step_resident()
    step_resident()
    st_t = L.last_stats()
    L.set_option("timing", 0)
    peaks = load_peaks()
    macs, ms_upd = st_t["update_macs"], st_t["ms_update"]
    path = st_t.get("gemm_path_used", None)
    achieved_tmacs = macs / (ms_upd * 1e-3) / 1e12 if ms_upd > 0 else None
    tensor_used = bool(st_t.get("tc_launches", 0))
    if tensor_used:
        # 16 u8xu8 MACs per field MAC on the int8 tensor pipe; int8 dense peak = 2 x measured bf16 (nominal ratio)
        peak = peaks["bf16_sustained"] * 2.0
        ach = achieved_tmacs * 16 * 2 if achieved_tmacs else None
        roof = {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TOP/s (int8, 2 ops per MAC)",
                "frac": ach / peak if ach else None, "traffic": None,
                "kernel": "Schur-update GEMMs on tcgen05 kind::i8 (gemm_tc_panel_kernel for K <= 256, gemm_tc_kernel above), "
                          "limb-split pre-passes included in the time",
                "note": f"achieved = executed update field-MACs x 16 u8 MACs x 2 ops / summed CUDA-event time of those "
                        f"launches on the call's stream; peak = 2 x {peaks['source']} sustained bf16 (guide's nominal "
                        f"int8:bf16 ratio); traffic: see profiles/ (ncu --set full capture of the top launch)"}
    else:
        # CUDA-core path: one IMAD.WIDE.U32 per field MAC; nominal issue peak 148 SM x 64 lanes x f_max
        peak = 148 * 64 * peaks["sm_max_mhz"] * 1e6 / 1e12
        roof = {"bound": "alu", "achieved": achieved_tmacs, "peak": peak, "unit": "T field-MAC/s",
                "frac": achieved_tmacs / peak if achieved_tmacs else None, "traffic": None,
                "note": "peak = 148 SM x 64 IMAD lanes x max SM clock (DESIGN.md); "
                        "achieved = executed update MACs / summed event time of the update kernels"}
    # the largest single launch, per launch: algorithmic bytes (C read + C written + both limb-plane sets read) and,
    # for the default workload, the DRAM traffic ncu measured for the same launch (profiles/r01_v9_launches_c3.md)
    tm_, tn_, tk_ = st_t.get("top_m", 0), st_t.get("top_n", 0), st_t.get("top_k", 0)
    if tensor_used and st_t.get("ms_update_top", 0) > 0:
        kp_ = -(-tk_ // 128) * 128
        roof["top_launch"] = {
            "M": tm_, "N": tn_, "K": tk_, "ms": st_t["ms_update_top"],
            "achieved": 32.0 * tm_ * tn_ * tk_ / (st_t["ms_update_top"] * 1e-3) / 1e12,
            "algorithmic_bytes": 8 * tm_ * tn_ + 4 * kp_ * (tm_ + tn_),
            "note": "event-timed, limb split included"}
        if args.workload == "c3" and not args.opt:
            roof["traffic"] = NCU_TOP_LAUNCH_DRAM_BYTES_C3
            roof["top_launch"]["traffic_note"] = ("roofline.traffic = dram__bytes_read.sum + dram__bytes_write.sum of the "
                                                  "M = N = 9744, K = 128 launch in the ncu --set full capture")
    roof["update_share_of_step"] = ms_upd / st_t["ms_total"] if st_t["ms_total"] else None
    roof["timed_split_ms"] = {"update": ms_upd, "strip": st_t.get("ms_strip"), "trsm": st_t.get("ms_trsm"),
                              "total_with_timing_syncs": st_t["ms_total"]}

    out = {
        "metric": "rref_gmulmod_per_s", "value": value, "unit": "Gmulmod/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": (value / world / PAPER_A100_GMULMOD[args.workload]) if args.workload in PAPER_A100_GMULMOD else None,
        "dtype": "u32", "data": "synthetic",
        "config": {"workload": f"{args.workload}: {rows}x{cols} uint32 {WORKLOAD_KIND[cfg['kind']]}, p={p}", "rank": int(ranks[-1]),
                   "parallelism": "replicas" if world > 1 else "single", "l2": "input (%d MB) larger than L2" %
                   (nbytes // 2 ** 20) if nbytes > 126 * 2 ** 20 else "input fits L2; restored by a device copy each step",
                   "options": args.opt},
        "e2e": {"value": e2e_value, "unit": "Gmulmod/s", "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": 0 if on_device else int(nbytes), "d2h_bytes_per_step": 0 if on_device else int(nbytes),
                **({"note": "not measured: this config is generated on the device (40 GB)"} if on_device else
                   {"mode": "double-buffered: the pinned H2D of step k+1 and the D2H of step k-1 overlap the call of step k; "
                            "every step's copies are inside the timed region",
                    "serial_ms_per_step": e2e_serial_ms,
                    "serial_value": replicas.aggregate_throughput(n_nominal, e2e_serial_ms * 1e-3, world) / 1e9})},
        "gpu_launches": int(stats["kernel_launches"]) * args.steps,
        "clocks": clocks, "roofline": roof,
        "stats": {k: stats[k] for k in ("kernel_launches", "host_syncs", "panels", "row_swaps", "update_macs")},
        "baseline_context": "paper, A100: 3.6 s at N=1e4 (PAPER.md:59) = 185 Gmulmod/s, 45 min at N=1e5 (PAPER.md:61) = 247 "
                            "Gmulmod/s; another machine, context only",
    }
    if rank == 0 and world == 1 and args.workload == "c3" and not args.no_f64:
        out["fp64"] = f64_leg(torch, L, dev)
    if rank == 0 and not args.no_cpu_baseline:
        import oracle
        threads = oracle.max_threads()
        v, dt = oracle_sample_gmulmod(args.ref_n, p, threads)
        out["cpu_baseline"] = {"value": v, "unit": "Gmulmod/s", "cores": threads, "kind": "oracle", "seconds": dt,
                               "sample": f"{args.ref_n}x{args.ref_n} dense uniform F_p (same recipe as the workload), "
                                         f"oracle Gauss-Jordan, {threads} OpenMP threads"}
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
