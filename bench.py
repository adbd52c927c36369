#!/usr/bin/env python
"""bench.py -- GP iterations/s of the B200 gradient-projection IMRT optimiser (BASELINE.json metric).

A step is ONE accepted gradient-projection iteration: transpose SpMV g = D^T r, then an Armijo line search in which
every trial is a projection x+ = max(0, x - lambda g), a dose SpMV d = D x+, the fused penalty / residual pass and
the objective reduction, then the accept / stop logic.  The K timed
steps run inside ONE imrt_plan_run_iters(K) call: the loop is device-resident, the host does not see the steps.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--driver persistent|graph|host]
    python bench.py --impl reference ...        # the fp64 CPU oracle on the host cores (reference arm)

Workload: BASELINE.json configs[3], the headline 9-field / 5 mm beamlet / 2.5 mm voxel phantom (the config the
metric's 60 %-of-HBM target is quoted on); it fits one GPU.  Inputs are seeded and synthetic (synth_inputs).
N > 1: `value` is replicas (every rank optimises its own plan -- the unit of production throughput is one patient's
plan; no collective on the data path; sum over ranks / max time), and the line's "sharded" object is the SAME single
workload row-sharded over the N GPUs with the in-kernel exchange (strong scaling).  At N = 1 "sharded" runs
--virtual-ranks ranks co-resident on the one GPU.
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

import synth_inputs  # noqa: E402  (seeded input generator: no optimiser arithmetic)

METRIC = "gp_iterations_per_s"
UNIT = "iterations/s"
DRIVERS = {"graph": 0, "host": 1, "persistent": 2}


def workload_name(cfg_id):
    return synth_inputs.CONFIGS[cfg_id].name


def algorithmic_bytes(prob, R=1):
    """int32/fp32 CSR bytes one pass has to move (independent of how the library lays things out).
    A dose pass that evaluates R line-search trial points streams D once and writes R residual vectors."""
    nnz, n_v, n_b = prob.nnz, prob.n_v, prob.n_b
    fwd = 8 * nnz + 4 * (n_v + 1) + 1 * n_v + R * 4 * n_v + 8 * n_b   # D, row_ptr, sid, r out (per trial), x and g in
    tr = 8 * nnz + 4 * (n_b + 1) + 4 * n_v + 4 * n_b                 # D^T, rowT_ptr, r in once, g out
    return fwd, tr


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def recorded_traffic(kernel, workload):
    """DRAM bytes per launch (read + write) from the committed ncu --set full capture of this workload
    (profiles/traffic.csv), else None."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["kernel"] == kernel and row.get("workload", workload) == workload:
                    return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
    except Exception:
        pass
    return None


class ClockSampler:
    """SM clock and throttle reasons during the timed region (NVML, ~5 ms period)."""

    def __init__(self, index):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.004)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr is not None:
            self._stop.set()
            self._thr.join()
        if not self.samples:   # NVML unavailable: one nvidia-smi reading
            try:
                out = subprocess.check_output(["nvidia-smi", "-i", str(self.index), "--query-gpu=clocks.sm,clocks.max.sm",
                                               "--format=csv,noheader,nounits"], text=True).strip().split(",")
                self.samples, self.max_mhz = [int(out[0])], int(out[1])
            except Exception:
                pass
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------ reference arm
def oracle_iterations(prob, n_iters):
    import oracle   # test infrastructure: allowed in bench.py's cpu_baseline / --impl reference legs only
    oracle.build()
    t0 = time.perf_counter()
    res = oracle.run(prob, n_iters=n_iters, delta=0.0)
    dt = time.perf_counter() - t0
    return res, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    prob = synth_inputs.make_phantom(args.config)
    _, t1 = oracle_iterations(prob, 1)                       # warm-up (page-in) and a cost estimate
    budget_s = 150.0
    k = int(max(1, min(args.steps, budget_s / max(t1, 1e-3))))
    res, dt = oracle_iterations(prob, k)
    value = res.n_iters / dt
    sample = "first %d GP iterations of %s from x0 (of %d requested), serial fp64 oracle/imrt_oracle.c" % (res.n_iters, prob.name, args.steps)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": res.n_iters,
            "warmup": 1, "ms_per_step": 1e3 * dt / res.n_iters, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": prob.name, "n_v": prob.n_v, "n_b": prob.n_b, "nnz": prob.nnz, "lambda0": prob.lambda0,
                       "trials_per_iter": float(res.n_trials.mean())},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_0908_4421_b200 as imrt

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the optimiser has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")        # the ranks' transport log (NVLink / NVLS) goes to stderr
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, W = args.steps, max(args.warmup, 3)
    prob = synth_inputs.make_phantom(args.config)
    driver = DRIVERS[args.driver]
    stream = torch.cuda.current_stream(dev)

    t0 = time.perf_counter()
    plan = imrt.Plan(prob, max_iters=W + K, driver=driver, device=dev, ls_batch=args.ls_batch, tune_level=args.tune_level)
    torch.cuda.synchronize()
    plan_create_s = time.perf_counter() - t0
    info = plan.info()
    R = info["ls_batch"]
    fwd_bytes, tr_bytes = algorithmic_bytes(prob, R)

    # ---------------- timed region: W warm-up iterations, then exactly K iterations in one device-resident run
    plan.set_x(prob.x0)
    plan.run_iters(W)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    plan.run_iters(K)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    # per-CTA %globaltimer stamps of the LAST dose / transpose pass of the timed run: what a pass takes INSIDE the
    # device-resident loop (no launch, no cold start), mean over the CTAs and first-start-to-last-end span
    in_loop = {}
    for kind, name in ((0, "k_dose"), (1, "k_transpose")):
        t0s, t1s = plan.pass_timing(kind)
        if t0s.size:
            in_loop[name] = (float((t1s - t0s).mean()) * 1e-6, float(t1s.max() - t0s.min()) * 1e-6)

    # ---------------- the two streaming kernels alone (roofline): isolated launches, matrices >> L2
    def time_pass(kind, n=40):
        plan.launch_pass(kind, 5)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        plan.launch_pass(kind, n)
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    dose_ms = time_pass(0)
    tr_ms = time_pass(1)
    # read-only streaming ceilings: the same rings / stages move the same bytes, the consumers only wait and release
    dose_stream_ms = time_pass(2)
    tr_stream_ms = time_pass(3) if info["tr_format"] == 2 else None
    clocks = sampler.stop()

    tr = plan.trace()
    fwd_passes, tr_passes = plan.counters()
    if tr.n_iters != W + K or tr.stop_reason != 0:
        raise SystemExit("bench.py: the run did %d of %d iterations (stop reason %s); the timing is not K steps"
                         % (tr.n_iters, W + K, imrt.STOP_NAMES[tr.stop_reason]))
    trials_timed = int(tr.n_trials[W:].sum())
    passes_timed = int(np.ceil(tr.n_trials[W:] / R).sum())     # one dose pass evaluates up to R trial points
    loop_bytes = passes_timed * fwd_bytes + K * tr_bytes

    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    value = world * K / (ms * 1e-3)

    # ---------------- the same workload row-sharded over ranks (all ranks take part): the in-kernel exchange path
    sharded_res = None
    if world > 1 or args.virtual_ranks > 1:
        sharded_res = run_sharded(args, prob, dev, rank, world, dist, barrier)

    extra = {}
    if rank == 0:
        peak, peak_src = measured_peak()
        l2_bytes = torch.cuda.get_device_properties(dev).L2_cache_size
        flush = "inputs larger than L2 (D and D^T %.0f MB each vs %.0f MB L2)" % (8 * prob.nnz / 1e6, l2_bytes / 1e6) \
            if 8 * prob.nnz > 2 * l2_bytes else "matrices are L2-resident: GB/s figures are L2, not HBM, bandwidth"
        # the library re-encodes the matrices, so the roofline fraction uses the bytes its own layouts make
        # a pass move (packed D + residual writes + x, g; the D^T stream + one read of r + g), and the CSR-equivalent
        # "effective" GB/s (algorithmic bytes / time) is quoted separately
        dose_layout = info["pack_bytes"] + 16 * info["fwd_blocks"] + R * 4 * info["nonempty_rows"] + 8 * prob.n_b
        tr_layout = info["tr_stream_bytes"] + 4 * prob.n_v + 4 * prob.n_b
        dose_gbs = dose_layout / (dose_ms * 1e-3) / 1e9
        tr_gbs = tr_layout / (tr_ms * 1e-3) / 1e9
        dose_eff = fwd_bytes / (dose_ms * 1e-3) / 1e9
        tr_eff = tr_bytes / (tr_ms * 1e-3) / 1e9
        t_dose, t_tr = recorded_traffic("k_dose", prob.name), recorded_traffic("k_transpose", prob.name)

        def roof(kernel, what, ms, layout, csr, traffic, stream_ms, read_bytes):
            gbs = layout / (ms * 1e-3) / 1e9
            d = {"bound": "hbm", "kernel": what, "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "peak_source": peak_src,
                 "traffic": traffic, "bytes_per_launch": layout, "ms_per_launch": ms,
                 # the two fractions under their own names: DRAM bytes actually moved (ncu capture of this kernel and workload,
                 # else the layout bytes) and the CSR-equivalent bytes of SURVEY.md 8(d), each / time / measured peak
                 "frac_dram": (traffic if traffic else layout) / (ms * 1e-3) / 1e9 / peak,
                 "frac_csr_equiv": csr / (ms * 1e-3) / 1e9 / peak,
                 "effective_csr_gbs": csr / (ms * 1e-3) / 1e9, "algorithmic_csr_bytes": csr,
                 "frac_of_nominal_8TBs": gbs / 8000.0}
            if kernel in in_loop and args.driver == "persistent":
                mean_ms, span_ms = in_loop[kernel]
                f_loop = layout / (span_ms * 1e-3) / 1e9 / peak
                d["in_loop"] = {"ms_mean_over_ctas": mean_ms, "ms_span": span_ms, "achieved_gbs": layout / (span_ms * 1e-3) / 1e9,
                                "frac": f_loop, "valid": bool(f_loop <= 1.0),
                                "note": "the same pass inside the persistent loop (per-CTA %globaltimer stamps of the last pass of the "
                                        "timed run; span = first CTA's start to last CTA's end): no launch, no cold start.  A "
                                        "diagnostic, not the roofline fraction: the span leaves out the barrier and the scalar phases, "
                                        "and part of x / r / g is L2-resident inside the loop, so it can come out above a copy-kernel "
                                        "peak -- `valid` is false then and the figure must not be quoted as a fraction of HBM peak"}
            if stream_ms:
                d["stream_ceiling_gbs"] = read_bytes / (stream_ms * 1e-3) / 1e9     # the pass's reads with the arithmetic left out
                d["stream_ceiling_ms"] = stream_ms
                d["frac_of_stream_ceiling"] = stream_ms / ms
            return d

        r_dose = roof("k_dose", "k_dose (dose SpMV for %d trial point(s) + penalty + residual + objective partials)" % R,
                      dose_ms, dose_layout, fwd_bytes, t_dose, dose_stream_ms, info["pack_bytes"] + 16 * info["fwd_blocks"])
        r_tr = roof("k_transpose", "k_transpose (D^T r on the explicit transpose, %s)" % ("plain CSR", "16-bit offsets", "row pairs")[info["tr_format"]],
                    tr_ms, tr_layout, tr_bytes, t_tr, tr_stream_ms, info["tr_stream_bytes"])
        r_dose["note"] = ("achieved / frac use the bytes of the library's own layouts (they agree with the ncu DRAM traffic to 1 %); "
                          "frac_csr_equiv counts the int32/fp32 CSR bytes the layouts avoid moving")
        # `roofline` is the LONGER of the two kernels of a step; the other one rides along
        roofline, roofline_other = (r_dose, r_tr) if dose_ms >= tr_ms else (r_tr, r_dose)
        roofline_tr = roofline_other

        # ---------------- time-to-plan: the config's own stopping rule from x0 (device-resident, inputs in HBM)
        cfg = synth_inputs.CONFIGS[args.config]
        plan2 = imrt.Plan(prob, max_iters=cfg.n_iters, driver=driver, device=dev, ls_batch=args.ls_batch, tuning=plan.tuning())
        plan2.set_x(prob.x0)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        if cfg.delta > 0:
            plan2.run_to_tol(cfg.delta, cfg.n_iters)
        else:
            plan2.run_iters(cfg.n_iters)
        b.record(stream)
        torch.cuda.synchronize()
        tr2 = plan2.trace()
        ttp = {"seconds": a.elapsed_time(b) * 1e-3, "iterations": tr2.n_iters, "stop_reason": imrt.STOP_NAMES[tr2.stop_reason],
               "rule": ("delta=%g or %d iterations" % (cfg.delta, cfg.n_iters)) if cfg.delta > 0 else "%d iterations" % cfg.n_iters,
               "final_objective": float(tr2.obj[-1])}
        plan2.close()
        del plan2

        # ---------------- the same K timed iterations with the LIBRARY DEFAULT partition (imrt_options.tune_level = 0: cost model
        # only, no measured rebalancing, ~9 ms less plan creation) -- printed beside the headline, which uses --tune-level
        default_rate = None
        if args.tune_level != 0:
            plan0 = imrt.Plan(prob, max_iters=W + K, driver=driver, device=dev, ls_batch=args.ls_batch, tune_level=0)
            plan0.set_x(prob.x0)
            plan0.run_iters(W)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            plan0.run_iters(K)
            b.record(stream)
            torch.cuda.synchronize()
            ms0 = a.elapsed_time(b)
            default_rate = {"value": K / (ms0 * 1e-3), "unit": "iterations/s", "ms_per_step": ms0 / K, "tune_level": 0,
                            "note": "library default partition; the headline `value` uses tune_level %d, whose measured rebalancing "
                                    "(~9 ms at cfg3) happens at plan creation, outside the timed region" % args.tune_level}
            plan0.close()
            del plan0

        # ---------------- end to end through the C-ABI with HOST buffers: upload D, create the plan (builds D^T), set x,
        # run K iterations, read x, dose and the trace back -- all inside the timed region
        import ctypes
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        h_rp, h_col, h_val, h_sid, h_x0 = pin(prob.row_ptr), pin(prob.col), pin(prob.val), pin(prob.sid), pin(prob.x0)
        h_x = torch.empty(prob.n_b, dtype=torch.float32).pin_memory()
        h_d = torch.empty(prob.n_v, dtype=torch.float32).pin_memory()
        ws_bytes = imrt.imrt_workspace_bytes(prob.n_v, prob.n_b, prob.nnz, prob.n_structures, K)
        d_ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
        d_rp, d_col, d_val, d_sid = (torch.empty_like(t, device=dev) for t in (h_rp, h_col, h_val, h_sid))
        d_x0 = torch.empty(prob.n_b, dtype=torch.float32, device=dev)
        d_x = torch.empty(prob.n_b, dtype=torch.float32, device=dev)
        d_d = torch.empty(prob.n_v, dtype=torch.float32, device=dev)
        prm = imrt.Params(prob.eps, prob.alpha, prob.lambda0, prob.max_ls, K, driver, args.ls_batch)
        # the measured rebalancing (tune_level 2, ~9 ms) buys ~12 % of loop speed: it pays for itself after ~600 iterations
        e2e_tune = args.tune_level if K >= 1000 else 0
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for dst, src in ((d_rp, h_rp), (d_col, h_col), (d_val, h_val), (d_sid, h_sid), (d_x0, h_x0)):
            dst.copy_(src, non_blocking=True)
        t_c0 = time.perf_counter()      # imrt_plan_create synchronises the stream: this interval also waits for the H2D copies
        handle = imrt.imrt_plan_create(prob.n_v, prob.n_b, prob.nnz, d_rp, d_col, d_val, d_sid, prob.t_under, prob.t_over,
                                       prob.w_under, prob.w_over, prm, d_ws, stream.cuda_stream, imrt.Options(tune_level=e2e_tune))
        t_c1 = time.perf_counter()
        imrt.imrt_plan_set_x(handle, d_x0)
        imrt.imrt_plan_run_iters(handle, K)
        imrt.imrt_plan_get_x(handle, d_x)
        imrt.imrt_plan_get_dose(handle, d_d)
        h_x.copy_(d_x, non_blocking=True)
        h_d.copy_(d_d, non_blocking=True)
        tr3 = imrt.imrt_plan_get_trace(handle, K)     # synchronises; the trace is the step's "loss"
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        imrt.imrt_plan_destroy(handle)
        h2d = sum(t.numel() * t.element_size() for t in (h_rp, h_col, h_val, h_sid, h_x0))
        d2h = h_x.numel() * 4 + h_d.numel() * 4 + (tr3.n_iters + 1) * 8 + tr3.n_iters * 20
        e2e = {"value": tr3.n_iters / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d / max(tr3.n_iters, 1),
               "d2h_bytes_per_step": d2h / max(tr3.n_iters, 1), "seconds": e2e_s, "iterations": tr3.n_iters, "tune_level": e2e_tune,
               "h2d_plus_plan_create_s": t_c1 - t0,        # warm: the process has created plans before (plan_create_s at the top
                                                           # level is the first, cold, creation through the Python convenience class)
               "includes": "H2D of CSR D + structure ids + x0 from pinned memory, plan create (builds D^T), set_x, run, D2H of x, dose, trace"}
        del d_ws, d_col, d_val

        # ---------------- the oracle on the host cores, bounded sample (reported baseline, not the target)
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            n_cpu = max(2, min(K, args.cpu_iters))
            res, dt = oracle_iterations(prob, n_cpu)
            try:
                with open("/proc/cpuinfo") as f:
                    model = next((ln.split(":", 1)[1].strip() for ln in f if ln.startswith("model name")), "unknown")
            except OSError:
                model = "unknown"
            cpu = {"value": res.n_iters / dt, "unit": UNIT, "cores": 1, "nproc": os.cpu_count(), "cpu_model": model, "kind": "oracle",
                   "sample": "first %d GP iterations of %s from x0 (%.1f s), serial fp64 oracle/imrt_oracle.c" % (res.n_iters, prob.name, dt),
                   "trials_per_iter": float(res.n_trials.mean())}

        extra = {"roofline": roofline, "roofline_other_kernel": roofline_tr, "time_to_plan": ttp, "e2e": e2e, "cpu_baseline": cpu,
                 "value_default_partition": default_rate,
                 "loop_effective_csr_gbs": loop_bytes / (ms * 1e-3) / 1e9,
                 "loop_gbs": (passes_timed * dose_layout + K * tr_layout) / (ms * 1e-3) / 1e9,
                 "loop_frac_of_peak": (passes_timed * dose_layout + K * tr_layout) / (ms * 1e-3) / 1e9 / peak,
                 "flush": flush}

    if rank == 0:
        n_launch = {0: 2, 1: 2 + K + passes_timed, 2: 2}[driver]   # k_set_target + graph/persistent launch (+ passes)
        if driver == 0:
            n_launch = 1 + 1 + K + passes_timed                    # k_set_target, k_begin, K transposes, the dose passes
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic",
                "config": {"workload": prob.name, "n_v": prob.n_v, "n_b": prob.n_b, "nnz": prob.nnz,
                           "nonempty_rows": info["nonempty_rows"], "lambda0": prob.lambda0, "eps": prob.eps, "alpha": prob.alpha,
                           "driver": args.driver, "tune_level": args.tune_level, "parallelism": "replicas x%d" % world if world > 1 else "single GPU",
                           "l2": extra.get("flush"), "trials_per_iter": trials_timed / K, "ls_batch": R,
                           "fwd_passes_timed": passes_timed, "tr_passes_timed": K},
                "clocks": clocks, "gpu_launches": n_launch, "plan_create_s": plan_create_s,
                "objective": {"first": float(tr.obj[0]), "after_warmup": float(tr.obj[W]), "last": float(tr.obj[-1])}}
        line.update({k: v for k, v in extra.items() if k != "flush"})
        line["sharded"] = sharded_res
        print(json.dumps(line))
    plan.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_sharded(args, prob, dev, rank, world, dist, barrier):
    """ONE problem over several ranks, rows of D in contiguous slabs (paper_0908_4421_b200/sharded.py): the partial
    gradients and objectives are summed INSIDE the persistent kernel through peer-memory inboxes.  world > 1: one rank per
    GPU (torch symmetric memory over NVLink), strong scaling of the fixed workload; world == 1: --virtual-ranks V ranks
    co-resident on the one GPU, each on SMs / V CTAs, one cooperative launch.  Returns a dict (rank 0) for the JSON line."""
    import torch
    from paper_0908_4421_b200 import sharded
    K, W = args.steps, max(args.warmup, 3)
    virtual = world == 1
    n_ranks = args.virtual_ranks if virtual else world
    try:
        if virtual:
            sp = sharded.CoResidentRanks(prob, n_ranks, max_iters=W + K, device=dev, tune_level=args.tune_level)
        else:
            sp = sharded.PeerRank(prob, max_iters=W + K, device=dev, tune_level=args.tune_level)
    except Exception as exc:       # e.g. no peer access / symmetric memory on this box
        return {"error": "%s: %s" % (type(exc).__name__, exc)}
    sp.set_x(prob.x0)
    sp.run_iters(W)
    barrier()
    stream = torch.cuda.current_stream(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    sp.run_iters(K)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    tr = sp.trace()
    out = {"value": (tr.n_iters - W) / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms / max(tr.n_iters - W, 1), "scaling": "strong",
           "ranks": n_ranks, "placement": "co-resident on one GPU (%d CTAs each, one cooperative launch)" % sp.plans[0].info()["fwd_grid"] if virtual
           else "one rank per GPU, inboxes in symmetric memory (NVLink peer stores)",
           "exchange": "in-kernel: g (n_b fp32) per iteration, R objectives per batch; fixed rank-order sums",
           "iterations": tr.n_iters - W, "stop_reason": tr.stop_reason, "objective_last": float(tr.obj[-1]),
           "caveat": ("co-resident ranks on ONE device: the exchange goes through that device's memory, not NVLink; the "
                      "one-rank-per-GPU path (sharded.PeerRank) has never been executed on > 1 GPU") if virtual
           else "first hardware runs of the one-rank-per-GPU path: compare objective_last with the single-GPU run"}
    sp.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=sorted(synth_inputs.CONFIGS))
    ap.add_argument("--driver", default="persistent", choices=sorted(DRIVERS))
    ap.add_argument("--ls-batch", type=int, default=0, choices=[0, 1, 2, 4],
                    help="line-search trial points per dose pass (0 = library default, 4)")
    ap.add_argument("--tune-level", type=int, default=2, choices=[0, 1, 2],
                    help="imrt_options.tune_level: 0 modelled partitions, 1 + isolated measurements, 2 + measurements inside the loop")
    ap.add_argument("--cpu-iters", type=int, default=60, help="oracle iterations timed for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--virtual-ranks", type=int, default=2,
                    help="ranks of the row-sharded run that share the GPU when there is only one (0 = skip the sharded run)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
