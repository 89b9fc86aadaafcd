#!/usr/bin/env python
"""bench.py -- superiorized feasibility-seeking iterations/s of the FREDopt hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]

A STEP is one superiorized iteration (forward pass at x, transposed pass ->
gradient, forward pass on g + accept test, residual / violation epilogue, transposed back-projection + update +
clamp) on the synthetic plan BASELINE.json configs[I] describes.  `value` = iterations/s with the plan resident in
HBM, timed with CUDA events on the plan's stream around one `fredopt_iterate(K)` call.  `e2e` is the same metric
through the C-ABI with HOST buffers: every step uploads the spot weights from pinned host memory
(fredopt_set_weights), runs fredopt_iterate(1) and reads the weights and the proximity / violation count back.
`roofline` is for the dominant kernel: its algorithmic bytes per launch (fredopt_get_pass_bytes; DESIGN.md
"Bytes") / its mean launch duration measured with CUDA events inside the library (FREDOPT_OPT_TIME_PASSES).
`cpu_baseline` is the fp64 oracle (oracle/), as it stands, timed on the host cores on a bounded sample.

N > 1 (torchrun): the path's units here are independent plans; every rank optimises its own copy of the plan
(weak scaling, no data-path collective), value = all ranks' iterations / max time.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "superiorization iterations/sec"
STATE_BYTES = 176           # sizeof(DevState): what fredopt_get_stats copies back
UNIT = "iterations/s"
DEFAULT_CONFIG = 3          # BASELINE.json configs[3]: the clinical-size plan the metric is quoted on (fits one B200)
DEFAULT_STEPS = {0: 50, 1: 200, 2: 100, 3: 50}
NOMINAL_HBM_GBS = 8000.0    # north_star's "~8 TB/s peak" (context; the roofline denominator is the measured copy figure)
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r02_traffic.csv")   # DRAM bytes per launch from the committed ncu capture
KERNEL_SOURCES = ("fredopt_kernels.cuh", "kernels_iter.cuh")       # the capture is valid for these sources only (hash)
CPU_BUDGET_S = 25.0         # bound of the all-cores oracle leg of the default run


def kernel_source_hash():
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        h.update(open(os.path.join(ROOT, "paper_2509_20012_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def captured_traffic(config, pass_name):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `pass_name` from the committed `ncu --set full` capture, or None
    when there is none for this configuration or the kernel sources have changed since (rows: config,pass,dram_bytes,hash)."""
    try:
        cur = kernel_source_hash()
        for line in open(TRAFFIC_FILE):
            c = [t.strip() for t in line.split(",")]
            if len(c) >= 4 and c[0] == str(config) and c[1] == pass_name and c[3] == cur:
                return int(c[2])
    except Exception:
        pass
    return None


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
            t0 = time.time()
            while not self.rows and time.time() - t0 < 3.0:      # first sample before the timed region starts
                time.sleep(0.01)
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for n, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def _dist_init():
    ws = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    lr = int(os.environ.get("LOCAL_RANK", "0"))
    return ws, rank, lr


# ------------------------------------------------------------------------------------------------ the workload, as both arms state it
L2_RESIDENT_BYTES = 256 * 1024 * 1024      # 2 x the B200's 126 MB L2: below this a pass's matrix bytes can stay in L2


def workload_config(args, spec, plan, ws=1, sharded=False):
    """`config` of the JSON line: what is computed, from the plan and the flags alone (no library call), so that `--impl reference`
    states the same object.  How OUR arm stores the plan (block rows, index width, bytes) is in its `plan` key."""
    lab = plan.labels > 0
    nnz_lab = int((plan.row_ptr[1:] - plan.row_ptr[:-1])[lab].sum())
    resident = 2 * 4 * nnz_lab < L2_RESIDENT_BYTES               # D and L values of the labelled rows, one pass
    return {"workload": f"configs[{args.config}] {spec.name}", "n_voxels": plan.n_rows, "n_spots": plan.n_cols,
            "nnz_per_matrix": plan.nnz, "n_labelled_voxels": int(lab.sum()), "nnz_labelled_per_matrix": nnz_lab,
            "lambda": spec.lam, "beta0": 0.0 if args.ams else spec.beta0, "a": spec.a,
            "value_bits": 16 if args.value_bits == 16 else 32,
            "ams_form": "block-sequential (Fig. 2 loop nest, R23)" if args.block_sequential else "simultaneous (R1)",
            "form": "pure feasibility-seeking (beta0 = 0)" if args.ams else "superiorized",
            "l2": ("L2-resident working set (labelled values of one pass %.1f MB < 256 MB): the GPU arm flushes L2 once before the timed "
                   "region; HBM fraction not meaningful" % (8 * nnz_lab / 1e6)) if resident else
                  "inputs larger than L2 (labelled values of one pass: %.2f GB)" % (8 * nnz_lab / 1e9),
            "parallelism": ("one plan sharded over %d GPUs by voxel range (x replicated, 3 all-reduces of <= n_spots + 3 doubles per "
                            "iteration)" % ws) if sharded else "1 plan per GPU"}


# ------------------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """The oracle, as it stands, on the host cores (its OpenMP timing build: the same source, row loops on all cores): the same
    window as our arm -- W warm-up iterations from x0, then K timed iterations of the full plan."""
    ws, rank, _ = _dist_init()
    if rank != 0:
        return
    from oracle import oracle
    from paper_2509_20012_b200 import plangen as pg
    spec = pg.config_spec(args.config)
    plan = pg.build_plan(spec, device="cuda" if torch.cuda.is_available() else "cpu")
    if args.value_bits == 16:            # the plan of the matrices rounded to half (round to nearest even), as fredopt_create_options.value_bits = 16 defines it
        plan.val_D = plan.val_D.half().float()
        plan.val_L = plan.val_L.half().float()
    cores = oracle.omp_threads()
    orc = oracle.from_plan(plan, omp=True)
    if args.block_sequential:
        orc.set_option(oracle.OPT_BLOCK_SEQUENTIAL, 1)
    orc.set_x(plan.x0)
    K, W = args.steps, args.warmup
    beta0 = 0.0 if args.ams else spec.beta0
    orc.iterate(W, spec.lam, beta0, spec.a)
    t0 = time.perf_counter()
    orc.iterate(K, spec.lam, beta0, spec.a)
    dt = time.perf_counter() - t0
    v = K / dt
    sample = (f"iterations {W}..{W + K - 1} from x0 of configs[{args.config}] ({spec.name}), full plan: the window of our arm; fp64 oracle, "
              f"OpenMP timing build, {cores} threads")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": K, "warmup": W,
        "ms_per_step": 1e3 * dt / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(args, spec, plan, ws=args.gpus, sharded=bool(args.shard) and args.gpus > 1),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def max_over_ranks(values, dist, device):
    """Element-wise MAX of a list of per-rank timings over all ranks (one all-reduce); identity at world size 1."""
    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_rate(units_per_rank, world_size, seconds):
    """Weak scaling over independent plans: every rank processed `units_per_rank` iterations of its own plan in at most
    `seconds` (the max over ranks) => whole-job iterations/s."""
    return world_size * units_per_rank / seconds


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    ws, rank, lr = _dist_init()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(lr)
    dist = None
    if ws > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", lr))
    from paper_2509_20012_b200 import fredopt, plangen as pg

    spec = pg.config_spec(args.config)
    t0 = time.perf_counter()
    plan = pg.build_plan(spec, device="cuda")
    torch.cuda.synchronize()
    t_gen = time.perf_counter() - t0
    torch.cuda.synchronize()
    stream = torch.cuda.Stream()          # the plan's stream: every kernel and every timing event of this run is on it
    torch.cuda.set_stream(stream)
    t0 = time.perf_counter()
    copt = {}
    if args.block_rows:
        copt["block_rows"] = args.block_rows
    if args.index_width:
        copt["index_width"] = args.index_width
    if args.value_bits:
        copt["value_bits"] = args.value_bits
    sharded = bool(args.shard) and ws > 1
    if sharded:                          # ONE plan on all ranks: voxel ranges, x replicated, sums completed by an NCCL all-reduce
        copt.update(shard_rank=rank, shard_world=ws)
    gp = fredopt.from_plan(plan, stream=stream.cuda_stream, **copt)
    if sharded:
        views = {}

        def allreduce(ptr, n, cuda_stream):
            t = views.get((ptr, n))
            if t is None:
                t = views[(ptr, n)] = torch.as_tensor(fredopt.DeviceDoubles(ptr, n), device="cuda")
            with torch.cuda.stream(stream):                 # the plan's stream: NCCL orders the collective after the work queued on it
                dist.all_reduce(t)
        gp.set_reduce(allreduce)
    torch.cuda.synchronize()
    t_create = time.perf_counter() - t0
    if args.block_sequential:
        gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, 1)
    if args.work_queue is not None:
        gp.set_option(fredopt.OPT_WORK_QUEUE, args.work_queue)
    if args.no_pdl:
        gp.set_option(fredopt.OPT_USE_PDL, 0)
    if args.skip_satisfied:
        gp.set_option(fredopt.OPT_SKIP_SATISFIED, 1)
    st0 = gp.stats()
    K, W = args.steps, args.warmup
    lam, beta0, a = spec.lam, (0.0 if args.ams else spec.beta0), spec.a
    pass_bytes = gp.pass_bytes()
    iter_bytes = st0["alg_bytes_iter"]
    if args.ams:      # forward over the constraint rows + back-projection; the vector kernels are noise at this size
        iter_bytes = pass_bytes["transpose_b"] * 2
    l2_bytes = torch.cuda.get_device_properties(lr).L2_cache_size
    config = workload_config(args, spec, plan, ws=ws, sharded=sharded)
    flush = None
    if config["l2"].startswith("L2-resident"):
        flush = torch.empty(int(1.5 * l2_bytes), dtype=torch.uint8, device="cuda")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up iterations, then K iterations in one fredopt_iterate call
    sampler = ClockSampler(lr)
    sampler.start()
    gp.set_weights(plan.x0)
    gp.iterate(W, lam, beta0, a)
    if flush is not None:
        flush.zero_()
    barrier()
    l0 = gp.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    gp.iterate(K, lam, beta0, a)
    e1.record(stream)
    barrier()
    launches = gp.launch_count() - l0
    ms = e0.elapsed_time(e1)
    # ---- end to end: host buffers, copies inside the timed region, every step
    xh = torch.from_numpy(plan.x0.copy()).pin_memory()
    xo = torch.empty_like(xh).pin_memory()
    gp.set_option(fredopt.OPT_RESET, 1)
    for _ in range(W):
        gp.iterate_host(1, lam, beta0, a, xh, xo); xh.copy_(xo)
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        # one C-ABI call per step (fredopt_iterate_host): H2D of S floats from pinned host memory, the iteration, D2H of S floats
        # and of the step's metrics (proximity, chi^2, violation count, k, s, beta), one synchronisation
        st_e = gp.iterate_host(1, lam, beta0, a, xh, xo)
        xh.copy_(xo)
    prox, nviol = st_e["prox"], st_e["n_violated"]
    barrier()
    e2e_s = time.perf_counter() - t0
    clocks = sampler.stop()
    # ---- per-kernel durations (CUDA events inside the library, on the plan's stream)
    gp.set_option(fredopt.OPT_RESET, 1)
    gp.set_weights(plan.x0)
    gp.iterate(W, lam, beta0, a)
    gp.set_option(fredopt.OPT_TIME_PASSES, 1)
    gp.iterate(min(K, 50), lam, beta0, a)
    pt = gp.pass_times()
    pass_bytes_static = pass_bytes
    pass_bytes = gp.pass_bytes_timed()     # as the timed launches needed them: the back-projection reads the values of rows with a coefficient only
    gp.set_option(fredopt.OPT_TIME_PASSES, 0)
    # ---- practical ceiling of a 100%-read pass: the library's streaming-read kernel over a buffer larger than L2
    nb = 1 << 31
    buf = torch.empty(nb, dtype=torch.uint8, device="cuda")
    buf.zero_()
    gp.stream_read(buf, nb, 3)
    r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    r0.record(stream); gp.stream_read(buf, nb, 10); r1.record(stream)
    torch.cuda.synchronize()
    read_gbs = 10 * nb / (r0.elapsed_time(r1) * 1e-3) / 1e9
    del buf
    PASS_KERNELS = {"forward_x": "k_forward<EPI_STORE_PQ> (k_forward<EPI_RESID> with --ams)", "transpose_g": "k_transpose + k_combine<GRAD>",
                    "forward_g": "k_forward<EPI_CPART>", "select": "k_select", "residual": "k_residual",
                    "transpose_b": "k_transpose + k_combine<UPDATE>"}
    top = max(pt, key=lambda n: pt[n][0])
    top_ms = pt[top][0] / max(pt[top][1], 1)
    peak, peak_src = _peaks()
    achieved = pass_bytes[top] / (top_ms * 1e-3) / 1e9
    passes = {n: {"ms": pt[n][0] / max(pt[n][1], 1), "alg_bytes": pass_bytes[n], "alg_bytes_all_rows": pass_bytes_static[n],
                  "gbs": pass_bytes[n] / max(pt[n][0] / max(pt[n][1], 1), 1e-9) / 1e6} for n in pt if pt[n][1] > 0}
    stats = gp.stats()
    # bytes one iteration needs, with the back-projection as the timed launches needed it (rows with a non-zero coefficient)
    iter_bytes_all_rows = iter_bytes
    iter_bytes = sum(pass_bytes[n] for n in (("forward_x", "transpose_b") if args.ams else PASS_KERNELS) if n in pass_bytes)
    spmv = ("forward_x", "transpose_b") if args.ams else ("forward_x", "transpose_g", "forward_g", "transpose_b")
    four_gbs = sum(pass_bytes[n] for n in spmv if n in passes) / max(sum(passes[n]["ms"] for n in spmv if n in passes), 1e-9) / 1e6

    ms, e2e_s = max_over_ranks([ms, e2e_s], dist, "cuda")
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    value = whole_job_rate(K, 1 if sharded else ws, ms * 1e-3)      # sharded: the ranks advance ONE plan together
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": ws, "steps": K, "warmup": W, "ms_per_step": ms / K,
        "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": config,
        "plan": {"nnz_active": stats["nnz_active"], "n_active_rows": stats["n_active_rows"], "n_sets": stats["n_sets"],
                 "block_rows": stats["block_rows"], "entries_active": stats["entries_active"],
                 "fill_in": stats["entries_active"] * stats["block_rows"] / max(stats["nnz_active"], 1),
                 "storage": ("matrix values ROUNDED TO IEEE HALF and stored in 16 bits (--value-bits 16: a different input, not the headline "
                             "configuration)" if args.value_bits == 16 else "fp32 matrix values") +
                            ", 16-bit indices where exact (else int32), fp64 vectors and accumulators",
                 "passes_per_iteration": 2 if args.ams else 4, "alg_bytes_per_iteration": iter_bytes,
                 "alg_bytes_per_iteration_all_rows": iter_bytes_all_rows,
                 "back_projection": "values of rows with a non-zero coefficient only (--skip-satisfied)" if args.skip_satisfied else
                                    "every value"},
        "iter_gbs": iter_bytes * K / (ms * 1e-3) / 1e9,
        "e2e": {"value": whole_job_rate(K, 1 if sharded else ws, e2e_s), "unit": UNIT, "h2d_bytes_per_step": plan.n_cols * 4,
                "d2h_bytes_per_step": plan.n_cols * 4 + STATE_BYTES, "call": "fredopt_iterate_host (pinned host buffers, one call per step)"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": top, "kernel_names": PASS_KERNELS.get(top, top), "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": captured_traffic(args.config, top),
                     "traffic_source": "profiles/r02_traffic.csv (ncu --set full capture; null when the kernel sources changed since)",
                     "peak_source": peak_src,
                     "alg_bytes_per_launch": pass_bytes[top], "ms_per_launch": top_ms,
                     "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS, "read_ceiling_gbs": read_gbs,
                     "frac_of_read_ceiling": achieved / read_gbs,
                     "four_spmv_passes_gbs": four_gbs, "four_spmv_passes_frac": four_gbs / peak},
        "passes": passes,
        "setup": {"generate_s": t_gen, "create_s": t_create},
        "final": {"prox": prox, "n_violated": nviol, "trials": stats["trials"]},
    }
    if ws == 1 and not args.no_forms and not args.ams:
        out["forms"] = compare_forms(gp, fredopt, plan, K, W, lam, beta0, a, stream)
    if ws == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(plan, spec, args, lam, beta0, a)
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def compare_forms(gp, fredopt, plan, K, W, lam, beta0, a, stream):
    """What an iteration buys in each feasibility-seeking form (iterations/s alone favours the form that moves x
    least).  For the simultaneous step (reading R1, the form `value` times) and the block-sequential sweep (R23, Fig. 2's own loop
    nest): iterations/s over the same window, proximity and violated sets (fredopt_proximity) after W + K iterations from x0, and
    the time either form needs to bring the proximity down to what the block-sequential form reaches in that window."""
    res = {}

    def run(block, n, timed):
        gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, block)
        gp.set_option(fredopt.OPT_RESET, 1)
        gp.set_weights(plan.x0)
        gp.iterate(W, lam, beta0, a)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream); gp.iterate(n, lam, beta0, a); e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3

    for name, block in (("simultaneous", 0), ("block_sequential", 1)):
        dt = run(block, K, True)
        p, nv = gp.proximity(None)
        res[name] = {"iterations_per_s": K / dt, "prox_after": p, "n_violated_after": nv, "iterations": W + K}
    target = res["block_sequential"]["prox_after"]
    for name, block in (("simultaneous", 0), ("block_sequential", 1)):
        gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, block); gp.set_option(fredopt.OPT_RESET, 1); gp.set_weights(plan.x0)
        done, secs, hit, step, cap = 0, 0.0, None, 25, 2000
        while done < cap:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); gp.iterate(step, lam, beta0, a); e1.record(stream)
            torch.cuda.synchronize()
            secs += e0.elapsed_time(e1) * 1e-3; done += step
            if gp.proximity(None)[0] <= target:
                hit = done
                break
        res[name]["to_target"] = {"prox_target": target, "iterations": hit, "seconds": secs if hit else None,
                                  "note": None if hit else f"not reached within {cap} iterations ({secs:.2f} s)"}
    gp.set_option(fredopt.OPT_BLOCK_SEQUENTIAL, 0); gp.set_option(fredopt.OPT_RESET, 1)
    return res


def cpu_baseline(plan, spec, args, lam, beta0, a):
    """The oracle as it stands on the host cores, over the window our arm times: W warm-up iterations from x0, then K timed.
    All cores = the OpenMP timing build of the same source; the leg is bounded (CPU_BUDGET_S): if the K iterations would not fit,
    fewer are timed and `sample` says so.  One thread = the plain build, continued from the all-cores oracle's state after the
    warm-up (same x, k, s, beta), over the first iterations of the same window."""
    from oracle import oracle
    K, W = args.steps, args.warmup
    cores = oracle.omp_threads()
    orc = oracle.from_plan(plan, omp=True)
    orc.set_x(plan.x0)
    t0 = time.perf_counter()
    orc.iterate(W, lam, beta0, a)
    t_warm = time.perf_counter() - t0
    x_w, st_w = orc.get_x(), orc.get_state()
    per = t_warm / max(W, 1)
    k_all = int(max(1, min(K, CPU_BUDGET_S / max(per, 1e-9))))
    t0 = time.perf_counter()
    orc.iterate(k_all, lam, beta0, a)
    dt = time.perf_counter() - t0
    one = oracle.from_plan(plan)
    one.set_x(x_w); one.set_state(st_w)
    k_one = int(max(1, min(k_all, 0.5 * CPU_BUDGET_S / max(dt / k_all * cores * 0.5, 1e-9))))
    t0 = time.perf_counter()
    one.iterate(k_one, lam, beta0, a)
    dt1 = time.perf_counter() - t0
    what = "superiorized" if beta0 else "pure feasibility-seeking"
    return {"value": k_all / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{what} iterations {W}..{W + k_all - 1} from x0 of the same plan (our arm times {W}..{W + K - 1}), fp64 oracle, "
                      f"OpenMP timing build, {cores} threads",
            "one_thread": {"value": k_one / dt1, "unit": UNIT, "cores": 1,
                           "sample": f"iterations {W}..{W + k_one - 1} of the same window, plain build, continued from the same state"}}


# ------------------------------------------------------------------------------------------------ configs[4]: pass sweep
def run_sweep(args):
    """BASELINE.json configs[4]: isolated SpMV passes on configs[2]-geometry matrices with every voxel labelled; spot sigma
    3 -> 10 mm, non-zeros 1e7 -> 1.2e9 (through pitch and layer count); x log-uniform on [1e-3, 1].  One JSON line per
    (sigma, nnz) point with GB/s (algorithmic bytes: the stored index -- 2 B, or 4 B for columns when there are more than
    65536 spots -- + 4 B per value array per non-zero) of every pass, timed
    with CUDA events around the C-ABI call (its vector conversions included), median of `--steps` repetitions."""
    import gc
    from paper_2509_20012_b200 import fredopt, plangen as pg
    torch.cuda.set_device(0)
    stream = torch.cuda.Stream()          # the plans' stream: kernels and timing events are on it
    torch.cuda.set_stream(stream)
    peak, peak_src = _peaks()
    l2 = torch.cuda.get_device_properties(0).L2_cache_size
    flush = torch.empty(int(1.5 * l2), dtype=torch.uint8, device="cuda")
    reps = args.steps or 10
    sigmas = [3.0, 5.0, 7.0, 10.0]
    targets = [1e7, 3e7, 1e8, 3e8, 1.2e9]
    if args.quick:
        sigmas, targets = [5.0], [1e7, 1e8]

    def timed(fn, nbytes, resident):
        ts = []
        for i in range(reps + 3):
            if resident:
                flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); fn(); e1.record(stream)
            torch.cuda.synchronize()
            if i >= 3:
                ts.append(e0.elapsed_time(e1))
        ms = float(np.median(ts))
        return {"ms": ms, "gbs": nbytes / ms / 1e6, "frac_of_measured_peak": nbytes / ms / 1e6 / peak}

    def spec_of(sigma, pitch, layers):
        # SURVEY sec. 8d labels every voxel so that "active = all"; here the passes run with the ROWS_ALL selector
        # instead (same rows, same arithmetic) and the ordinary structure labels are kept, so that the plan does not
        # hold a second, labelled copy of the whole matrix in HBM
        sp = pg.sweep_spec(sigma, pitch, layers)
        sp.label_all = False
        return sp

    for sigma in sigmas:
        # probe: non-zeros at a coarse lattice, then scale the spot count (pitch) and layer count to the target
        probe = pg.build_plan(spec_of(sigma, 12.0, 6), device="cuda")
        nnz0 = probe.nnz
        del probe
        for target in targets:
            ratio = target / nnz0                                  # nnz ~ layers / pitch^2
            layers = int(min(40, max(6, round(6 * ratio ** 0.4))))
            pitch = 12.0 / math.sqrt(max(ratio * 6 / layers, 1e-9))
            pitch = min(max(pitch, 0.8), 40.0)
            plan = pg.build_plan(spec_of(sigma, pitch, layers), device="cuda")
            for _ in range(2):                                     # the lattice is discrete: correct the pitch
                if 0.85 < plan.nnz / target < 1.18 or pitch <= 0.8:
                    break
                pitch = min(max(pitch * math.sqrt(plan.nnz / target), 0.8), 40.0)
                del plan
                plan = pg.build_plan(spec_of(sigma, pitch, layers), device="cuda")
            gp = fredopt.from_plan(plan, stream=stream.cuda_stream)
            V, S, nnz = plan.n_rows, plan.n_cols, plan.nnz
            x = torch.from_numpy(pg.log_uniform_weights(5, S)).cuda()
            r = torch.from_numpy(pg.log_uniform_weights(6, V)).cuda()
            d = torch.empty(V, dtype=torch.float32, device="cuda"); l = torch.empty_like(d)
            o = torch.empty(S, dtype=torch.float32, device="cuda")
            resident = 10 * nnz < 2 * l2
            gp.spmv_transpose(fredopt.ROWS_ALL, r, None, o)        # builds the transposed copy of the full matrix
            ibf = 2 if S <= 65536 else 4                           # index bytes as stored (16-bit columns if they fit)
            ibt = 2                                                # transposed: 16-bit row index inside 65536-row blocks
            res = {
                "forward_D": timed(lambda: gp.spmv_forward(fredopt.ROWS_ALL, x, d, None), (ibf + 4) * nnz, resident),
                "forward_DL_fused": timed(lambda: gp.spmv_forward(fredopt.ROWS_ALL, x, d, l), (ibf + 8) * nnz, resident),
                "transpose_D": timed(lambda: gp.spmv_transpose(fredopt.ROWS_ALL, r, None, o), (ibt + 4) * nnz, resident),
                "transpose_L": timed(lambda: gp.spmv_transpose(fredopt.ROWS_ALL, None, r, o), (ibt + 4) * nnz, resident),
                "transpose_DL_fused": timed(lambda: gp.spmv_transpose(fredopt.ROWS_ALL, r, r, o), (ibt + 8) * nnz, resident),
            }
            rows_ne = int((plan.row_ptr[1:] > plan.row_ptr[:-1]).sum().item())
            print(json.dumps({"sweep": "configs[4]", "sigma_mm": sigma, "pitch_mm": round(pitch, 3), "layers": layers,
                              "n_voxels": V, "n_spots": S, "nnz": nnz, "mean_row": nnz / max(rows_ne, 1),
                              "mean_col": nnz / max(S, 1), "index_bytes": [ibf, ibt], "l2": "L2 flushed before every repetition" if resident
                              else "larger than L2", "peak_gbs": peak, "passes": res}), flush=True)
            gp.destroy()
            del plan, gp, x, r, d, l, o
            gc.collect(); torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--block-sequential", action="store_true",
                    help="feasibility-seeking step in the block-sequential form of Fig. 2's loop nest (DESIGN.md R23)")
    ap.add_argument("--ams", action="store_true",
                    help="pure feasibility-seeking (beta0 = 0, the paper's 'AMS' runs, PAPER.md:120): two passes per iteration")
    ap.add_argument("--shard", action="store_true",
                    help="with --gpus N > 1 (torchrun): ONE plan sharded over the ranks by voxel range (strong scaling; DESIGN.md Multi-GPU)")
    ap.add_argument("--no-forms", action="store_true", help="skip the comparison of the two feasibility-seeking forms")
    ap.add_argument("--block-rows", type=int, default=0, help="fredopt_create_options.block_rows (0 = automatic)")
    ap.add_argument("--index-width", type=int, default=0, help="fredopt_create_options.index_width (0 = automatic, 32)")
    ap.add_argument("--value-bits", type=int, default=0, help="fredopt_create_options.value_bits (0 = fp32 values; 16 = values rounded to half)")
    ap.add_argument("--no-pdl", action="store_true", help="FREDOPT_OPT_USE_PDL = 0 (plain launches)")
    ap.add_argument("--skip-satisfied", action="store_true",
                    help="FREDOPT_OPT_SKIP_SATISFIED = 1: the back-projection streams the values of rows with a non-zero coefficient only")
    ap.add_argument("--work-queue", type=int, default=None, help="FREDOPT_OPT_WORK_QUEUE (bit 0 forward, bit 1 transposed passes)")
    ap.add_argument("--sweep", action="store_true", help="BASELINE.json configs[4]: isolated-pass sweep (1 GPU)")
    ap.add_argument("--quick", action="store_true", help="with --sweep: two points only")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.sweep:
        run_sweep(args)
        return
    if args.impl == "reference":
        if args.steps is None:
            args.steps = 5
        run_reference(args)
    else:
        if args.steps is None:
            args.steps = DEFAULT_STEPS.get(args.config, 50)
        run_ours(args)


if __name__ == "__main__":
    main()
