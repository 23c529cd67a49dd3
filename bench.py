#!/usr/bin/env python
"""bench.py -- throughput of the GDA hot path on synthetic BASELINE.json workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

A "step" is one pass of the whole hot path over the batch of B restarts: `eval_every` GDA iterations
(gradient S1/S2/S3 + fused update S4, one kernel each) followed by one evaluation (round + exact score
S5 + best-so-far), i.e. one CUDA-graph launch of the library; the arg-best S6 closes every call.
metric = restart-iterations/s = B * eval_every * K / time.

Timed region: K resumed gda_run calls of one step each, every one bracketed by CUDA events on the
launching stream; the L2 is flushed (a 256 MiB write, not timed) between steps because the state of
the sparse configs (61.5 MB) is smaller than the 126 MB L2.  `whole_run` repeats the measurement as ONE
gda_run of K steps without flushes (the way a user runs it).  `e2e` is gda_run_host: pinned HOST
buffers in, HOST results out, copies inside the timed region.

Under torchrun (N > 1) every rank runs its own B restarts of the same instance (restarts are
independent): weak scaling, no collective on the data path; the best objective is
combined with one all-reduce(MIN) after the timed region.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2509_21064_b200 import workloads as wl  # noqa: E402

HEADLINE_CONFIG = 3   # BASELINE.json configs[2]: Max-Cut n=20000, B=256 -- the config the HBM target is quoted on


def load_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        d = json.loads(f.read_text())
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d["bf16_tflops"]),
                    bf16_tflops_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


def algorithmic_work(w: wl.Workload):
    """Per GDA step (one launch of the step kernel): algorithmic bytes / flops."""
    P, B = w.problem, w.B
    n = P.n
    state = (8 if getattr(w.hyper, "dual", 0) else 16) * n * B   # read x, y; write x, y (fp32); PDBO-s has no y array
    if w.kind == "qubo_csr":
        nnz = int(P.rowptr[-1])
        return dict(bound="hbm", bytes=state + 8 * nnz + 4 * (n + 1) + 4 * n, flops=2 * nnz * B)
    if w.kind == "maxkcut":                  # read X, Z (k planes each) and y; write the same
        nnz = int(P.rowptr[-1])
        return dict(bound="hbm", bytes=(4 * P.k + 2) * 4 * n * B + 8 * nnz + 4 * (n + 1), flops=2 * nnz * B * P.k)
    if w.kind == "maxsat":
        L = int(P.lit.shape[0])
        k = L // P.m
        return dict(bound="hbm", bytes=state + 4 * (n + 1) + L * (4 + 4 * max(k - 1, 1)), flops=(k + 1) * L * B)
    return dict(bound="tensor", bytes=state + 2 * 2 * n * B + 2 * n * n, flops=2 * n * n * B)


# ------------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """SM clock and clock-event reasons DURING a measurement.  NVML polled from a thread every ~2 ms (a secondary workload is
    timed for a few hundred ms, so every record has well over 10 samples); `nvidia-smi -lms 20` if NVML cannot be loaded."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    PERIOD_S = 0.002

    def __init__(self, gpu_index: int):
        self.gpu, self.rows, self.proc = gpu_index, [], None
        self.sm, self.smax, self.reasons, self.power = [], 0.0, set(), []
        self._stop, self._thread, self.source = threading.Event(), None, None

    def _nvml_loop(self, nv, handle):
        bits = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown, "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown, "sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(handle, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(handle))
                for name, bit in bits.items():
                    if r & bit:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(handle) / 1e3)
            except Exception:
                pass
            time.sleep(self.PERIOD_S)

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[self.gpu]) if vis and all(v.strip().isdigit() for v in vis.split(",")) else self.gpu
            handle = nv.nvmlDeviceGetHandleByIndex(phys)
            self.smax = float(nv.nvmlDeviceGetMaxClockInfo(handle, nv.NVML_CLOCK_SM))
            self._thread = threading.Thread(target=self._nvml_loop, args=(nv, handle), daemon=True)
            self._thread.start()
            self.source = "nvml"
            return
        except Exception:
            self._thread = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(self.gpu)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
            self.source = "nvidia-smi"
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self._thread:
            self._stop.set()
            self._thread.join(timeout=1)
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        sm, smax, reasons = list(self.sm), self.smax, set(self.reasons)
        for r in self.rows:
            try:
                sm.append(float(r[1]))
                smax = max(smax, float(r[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        busy = [v for v in sm if v > 0]
        return dict(sm_mhz=statistics.median(busy) if busy else None, sm_max_mhz=smax or None,
                    reasons=sorted(reasons), samples=len(sm), source=self.source,
                    power_w_max=max(self.power) if self.power else None)


# ------------------------------------------------------------------------------------------------
# the oracle arm (cpu_baseline leg and --impl reference): the ONLY place bench.py executes oracle/
# ------------------------------------------------------------------------------------------------
def oracle_problem(P):
    from oracle import pdbo
    if isinstance(P, wl.MaxKCut):
        from oracle import kcut
        return kcut.Problem(P.n, P.k, P.rowptr, P.col, P.val.astype(np.float64))
    if isinstance(P, wl.QuboCSR):
        return pdbo.Problem.qubo_csr(P.n, P.rowptr, P.col, P.val, P.c)
    if isinstance(P, wl.QuboDense):
        return pdbo.Problem.qubo_dense(P.n, P.Q, P.c)
    return pdbo.Problem.maxsat(P.n, P.m, P.cptr, P.lit, P.w)


def start_point(w: wl.Workload, seed: int) -> np.ndarray:
    """x0 ~ U[0,1) [n][B], or the logits Z0 [k][n][B] of a Max-k-Cut workload."""
    if w.kind == "maxkcut":
        return wl.z0_uniform(w.problem.k, w.problem.n, w.B, seed)
    return wl.x0_uniform(w.problem.n, w.B, seed)


def oracle_run(w: wl.Workload, OP, X, Y, iters, eval_every, nthreads, t0=0):
    """One oracle call on the columns X[..., :]; returns (x, y) of the last iterate."""
    h = w.hyper
    f = lambda v: float(np.float32(v))
    if w.kind == "maxkcut":
        from oracle import kcut
        r = kcut.run(OP, X, Y, alpha=f(h.alpha), beta=f(h.beta), gfun=h.gfun, log_eps=f(h.log_eps), iters=iters,
                     eval_every=eval_every, nthreads=nthreads)
        return r["z"], r["y"]
    from oracle import pdbo
    kw = oracle_kwargs(h, iters)
    kw["eval_every"] = eval_every
    r = pdbo.run(OP, X, Y, nthreads=nthreads, t0=t0, **kw)
    return r["x"], r["y"]


def oracle_kwargs(h, iters):
    f = lambda v: float(np.float32(v))
    return dict(alpha=f(h.alpha), beta=f(h.beta), delta=f(h.delta), gfun=h.gfun, log_eps=f(h.log_eps),
                iters=iters, eval_every=h.eval_every, seed=h.seed, dual=getattr(h, "dual", 0))


def oracle_sample_columns(w: wl.Workload, cores: int) -> int:
    """Restart columns per oracle step: one per core, fewer for the dense config (n^2 work per column-step)."""
    return max(1, min(w.B, cores if w.kind != "qubo_dense" else min(cores, 8)))


def _time_oracle_once(w: wl.Workload, budget_s: float, cores: int, Bo: int):
    OP = oracle_problem(w.problem)
    X0 = start_point(w, w.x0_seed)[..., :Bo].copy()
    h = w.hyper
    lam = float(np.float32(h.lambda0)) if not getattr(h, "dual", 0) else np.full(Bo, np.float32(h.lambda0), dtype=np.float64)
    it = 2 if w.kind == "qubo_dense" else 10
    oracle_run(w, OP, X0, lam, it, h.eval_every, cores)                                       # thread-pool warm-up
    t0 = time.perf_counter()
    oracle_run(w, OP, X0, lam, it, h.eval_every, cores)
    per_iter = (time.perf_counter() - t0) / it
    iters = int(max(it, min(h.iters, budget_s / max(per_iter, 1e-9))))
    mult = int(min(w.B // Bo, max(1.0, budget_s / max(iters * per_iter, 1e-9))))   # more columns if the budget allows
    if mult > 1:
        Bo *= mult
        X0 = start_point(w, w.x0_seed)[..., :Bo].copy()
        if getattr(h, "dual", 0):
            lam = np.full(Bo, np.float32(h.lambda0), dtype=np.float64)
    t0 = time.perf_counter()
    oracle_run(w, OP, X0, lam, iters, h.eval_every, cores)
    dt = time.perf_counter() - t0
    return Bo, iters, dt


def time_oracle(w: wl.Workload, budget_s: float):
    """cpu_baseline: the oracle as it stands (fp64, gcc -O2, OpenMP over restarts) on a bounded sample -- on all host
    cores, and (`one_core`) single-threaded with the process pinned to one core."""
    from oracle import pdbo
    pdbo.build()
    cores = max(1, min(pdbo.max_threads(), os.cpu_count() or 1))
    Bo, iters, dt = _time_oracle_once(w, budget_s, cores, oracle_sample_columns(w, cores))
    out = dict(value=Bo * iters / dt, unit="restart-iters/s", cores=cores, kind="oracle",
               sample=f"{Bo} of {w.B} restarts x {iters} GDA iterations of {w.name}, fp64, gcc -O2 -fopenmp, {dt:.1f} s")
    try:
        allowed = os.sched_getaffinity(0)
        os.sched_setaffinity(0, {min(allowed)})
        try:
            B1, it1, dt1 = _time_oracle_once(w, max(2.0, budget_s / 4), 1, 1)
        finally:
            os.sched_setaffinity(0, allowed)
        out["one_core"] = dict(value=B1 * it1 / dt1, unit="restart-iters/s", cores=1, pinned_to_core=min(allowed),
                               sample=f"{B1} restart(s) x {it1} GDA iterations, single thread, {dt1:.1f} s")
    except (AttributeError, OSError) as e:            # no affinity control on this host
        out["one_core"] = dict(unavailable=str(e))
    return out


def config_dict(args, w: wl.Workload):
    """The `config` both arms print (identical keys and values: the driver compares them)."""
    h = w.hyper
    return {"workload": w.name, "baseline_config_index": args.config if not (args.mis or args.maxkcut) else None,
            "kind": w.kind, "n": w.problem.n, "B_per_gpu": w.B,
            "step": f"{h.eval_every} GDA iterations + 1 evaluation (one CUDA graph launch on the GPU arm)",
            "hyper": {"lambda0": h.lambda0, "alpha": h.alpha, "beta": h.beta, "delta": h.delta, "gfun": h.gfun,
                      "dual": "scalar (PDBO-s)" if getattr(h, "dual", 0) else "per-variable (PDBO)"},
            "l2": "flushed between timed steps (256 MiB write, untimed)", "note": w.note}


def run_reference(args, w: wl.Workload):
    """--impl reference: K steps of the oracle, each `eval_every` iterations + evaluation on a column sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import pdbo
    pdbo.build()
    cores = max(1, min(pdbo.max_threads(), os.cpu_count() or 1))
    OP = oracle_problem(w.problem)
    Bo = oracle_sample_columns(w, cores)
    h = w.hyper
    per_step = h.eval_every if w.kind != "qubo_dense" else max(1, h.eval_every // 50)
    X = start_point(w, w.x0_seed)[..., :Bo].copy().astype(np.float64)
    Y = np.full((w.problem.n, Bo), float(np.float32(h.lambda0)))
    if getattr(h, "dual", 0):
        Y = Y[0].copy()                      # PDBO-s: one multiplier per restart
    t = 0
    for _ in range(args.warmup):
        X, Y = oracle_run(w, OP, X, Y, per_step, per_step, cores, t0=t)
        t += per_step
    t0 = time.perf_counter()
    for _ in range(args.steps):
        X, Y = oracle_run(w, OP, X, Y, per_step, per_step, cores, t0=t)
        t += per_step
    dt = time.perf_counter() - t0
    value = Bo * per_step * args.steps / dt
    sample = f"{Bo} of {w.B} restarts, {per_step} GDA iterations + 1 evaluation per step, fp64 oracle"
    print(json.dumps({
        "impl": "reference", "metric": "restart-iterations/s", "value": value, "unit": "restart-iters/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(args, w),
        "cpu_baseline": {"value": value, "unit": "restart-iters/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "restart-iters/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
L2_BYTES = 126 * 1024 * 1024


def state_bytes(w: wl.Workload) -> int:
    """x double buffer + y (sparse / MaxSAT), x + y + two bf16 operands (dense), k planes for Max-k-Cut."""
    n, B = w.problem.n, w.B
    if w.kind == "qubo_dense":
        return 12 * n * B
    if w.kind == "maxkcut":
        return (3 * w.problem.k + 1) * 4 * n * B
    return 12 * n * B


def ncu_record(w: wl.Workload) -> dict:
    tf = ROOT / "profiles" / "ncu_traffic.json"
    if not tf.exists():
        return {}
    d = json.loads(tf.read_text())
    rec = d.get(f"{w.name}_B{w.B}", d.get(w.name, {}))
    return rec if rec.get("B", w.B) == w.B else {}          # a capture at another batch size says nothing about this one


def l2_block(w: wl.Workload, rec: dict, t_kernel: float):
    """L2 roofline of a step kernel whose state is L2-resident: the bytes ncu saw cross the L2 <-> SM boundary per launch
    (profiles/ncu_traffic.json) / the kernel's duration, against the measured ceiling in profiles/measured_l2.json (the
    probe and its access shapes: profiles/l2_peak.md).  `shape_floor` is a kernel with this workload's access shape and no
    arithmetic, timed by the same probe: frac_of_shape_floor = its time / this kernel's time."""
    f = ROOT / "profiles" / "measured_l2.json"
    if not f.exists() or not rec.get("l2_to_sm_bytes"):
        return None
    m = json.loads(f.read_text())
    nbytes = rec["l2_to_sm_bytes"] + rec.get("sm_to_l2_bytes", 0)
    out = {"bytes_per_launch": nbytes, "achieved": nbytes / t_kernel / 1e12, "peak": m["l2_peak_tbps"], "unit": "TB/s",
           "frac": nbytes / t_kernel / 1e12 / m["l2_peak_tbps"], "peak_source": "profiles/measured_l2.json"}
    floor = m.get("shape_floor", {}).get(f"{w.name}_B{w.B}")
    if floor:
        out["shape_floor_us"] = floor["us"]
        out["frac_of_shape_floor"] = floor["us"] * 1e-6 / t_kernel
    return out


def roofline_block(w: wl.Workload, peaks, t_step_mean, t_step_median, t_eval):
    """roofline of the step kernel: algorithmic work per launch / its average duration, the duration being
    (one captured chunk - one evaluation) / eval_every from CUDA events (it includes the graph's launch gaps)."""
    work = algorithmic_work(w)
    ipe = w.hyper.eval_every
    t_kernel = max(t_step_mean - t_eval, 1e-9) / ipe
    t_kernel_med = max(t_step_median - t_eval, 1e-9) / ipe
    if work["bound"] == "hbm":
        achieved, peak, unit = work["bytes"] / t_kernel / 1e9, peaks["hbm_gbs"], "GB/s"
    else:
        achieved, peak, unit = work["flops"] / t_kernel / 1e12, peaks["bf16_tflops_sustained"], "TFLOP/s"
    rec = ncu_record(w)
    resident = state_bytes(w) < L2_BYTES
    if work["bound"] == "tensor":
        basis = "algorithmic flops / step-kernel time, against the measured SUSTAINED cuBLAS bf16 peak (the kernel is timed inside a long step)"
    elif resident:
        basis = (f"ALGORITHMIC bytes (16 B per variable-restart + structure, each once) / step-kernel time against the measured HBM copy peak; "
                 f"the state ({state_bytes(w) / 1e6:.1f} MB) is L2-RESIDENT on a B200 (126 MB L2), so this is not achieved HBM bandwidth: "
                 f"warm DRAM traffic is ~0 and what bounds the kernel is L2 -> SM delivery (l2_to_sm_bytes)")
    else:
        basis = (f"algorithmic bytes / step-kernel time against the measured HBM copy peak; the state ({state_bytes(w) / 1e6:.1f} MB) exceeds "
                 f"the 126 MB L2, so the step streams from HBM")
    extra = {}
    if work["bound"] == "hbm" and resident and not getattr(w.hyper, "dual", 0):
        l2 = l2_block(w, rec, t_kernel)
        if l2:
            extra["l2"] = l2
    if work["bound"] == "tensor":       # the timed loop is short (well under a second): the burst peak applies as well -- both are quoted
        extra = {"peak_burst": peaks["bf16_tflops"], "frac_burst": achieved / peaks["bf16_tflops"]}
    return {"bound": work["bound"], "achieved": achieved, "peak": peak, "unit": unit, "frac": achieved / peak, **extra,
            "traffic": rec.get("bytes"), "l2_to_sm_bytes": rec.get("l2_to_sm_bytes"), "traffic_source": rec.get("source"),
            "peak_source": peaks["source"], "kernel": rec.get("kernel", "step kernel (gradient + fused update)"),
            "us_per_launch": t_kernel * 1e6, "us_per_launch_median": t_kernel_med * 1e6,
            "frac_median": achieved / peak * t_kernel / t_kernel_med,
            "algorithmic_bytes_per_launch": work["bytes"], "algorithmic_flops_per_launch": work["flops"],
            "eval_us": t_eval * 1e6, "state_l2_resident": resident, "basis": basis}


def smem_roofline(w: wl.Workload, t_kernel_s: float, sm_count: int, sm_max_mhz: float):
    """The slab kernel (small n: state in shared memory, one launch per chunk) is bound by shared-memory gathers, not by
    HBM: nnz x B x 4 bytes of neighbour values per step against 128 B per clock and SM."""
    nnz = int(w.problem.rowptr[-1])
    gathered = nnz * w.B * 4
    peak = sm_count * 128 * sm_max_mhz * 1e6 / 1e9
    ach = gathered / t_kernel_s / 1e9
    return {"bound": "smem", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
            "gathered_bytes_per_step": gathered, "ctas": (w.B + 7) // 8,
            "basis": f"shared-memory bytes gathered per GDA step / step time against {sm_count} SMs x 128 B/clk x {sm_max_mhz:.0f} MHz "
                     f"(the launch has {(w.B + 7) // 8} CTAs of 8 restarts: at most that many SMs work)"}


class Session:
    """One device, one stream, the flush buffer; measures workloads one after the other."""

    def __init__(self, local_rank, rank, world):
        import torch
        self.torch, self.rank, self.world, self.local_rank = torch, rank, world, local_rank
        self.dev = torch.device("cuda", local_rank)
        self.stream = torch.cuda.Stream(self.dev)
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)

    def sync_all(self):
        import torch.distributed as dist
        self.torch.cuda.synchronize(self.dev)
        if self.world > 1:
            dist.barrier()
            self.torch.cuda.synchronize(self.dev)

    def measure(self, w: wl.Workload, K: int, W: int, peaks, full: bool, min_seconds: float = 0.0):
        """K timed steps (flushed L2), the evaluation alone, clocks; with full=True also the whole run, the trace and
        the end-to-end numbers through gda_run_host.  min_seconds > 0 raises K (up to 400) until the timed steps alone keep
        the GPU busy for that long, so that the clock record of a short workload has enough samples under load."""
        torch = self.torch
        from paper_2509_21064_b200 import api, multirank
        h, B, n = w.hyper, w.B, w.problem.n
        P = api.create_from_workload(w.problem)
        x0_host = torch.from_numpy(start_point(w, multirank.rank_x0_seed(w.x0_seed, self.rank))).pin_memory()
        x0 = x0_host.to(self.dev, non_blocking=True)
        stream, flush = self.stream, self.flush
        prm_step = api.params_from_hyper(h, iters=h.eval_every)
        prm0 = api.params_from_hyper(h, iters=0)
        res = {}
        with torch.cuda.stream(stream):
            out = P.run(x0, h.lambda0, prm_step)                          # warm-up: captures the graph, warms clocks
            for _ in range(W - 1):
                P.resume(prm_step, out)
            self.sync_all()
            if min_seconds > 0:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                P.resume(prm_step, out)
                e1.record(stream)
                self.sync_all()
                K = int(min(400, max(K, np.ceil(min_seconds * 1e3 / max(e0.elapsed_time(e1), 1e-3)))))
            res["K"] = K
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
            sampler = ClockSampler(self.local_rank)
            sampler.start()
            out = P.run(x0, h.lambda0, prm0)
            launches = P.info().last_run_kernel_launches
            self.sync_all()
            for k in range(K):                                            # timed: K steps, L2 flushed (untimed) between them
                flush.fill_(k & 0xFF)
                ev[k][0].record(stream)
                P.resume(prm_step, out)
                ev[k][1].record(stream)
                launches += P.info().last_run_kernel_launches
            self.sync_all()
            step_ms = [a.elapsed_time(b) for a, b in ev]
            res["best_flushed"] = float(out["obj"].min().item())
            res["chunk_fused"] = h.eval_every > 1 and P.info().last_run_step_launches == 1   # the slab kernel ran the chunk
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            P.resume(prm0, out)                                           # evaluation alone (one evaluation-only call)
            self.sync_all()
            e0.record(stream)
            for _ in range(10):
                P.resume(prm0, out)
            e1.record(stream)
            self.sync_all()
            t_eval = e0.elapsed_time(e1) / 1e3 / 10
            if not full:
                res["clocks"] = sampler.stop()
            else:
                prm_all = api.params_from_hyper(h, iters=h.eval_every * K)
                self.sync_all()
                e0.record(stream)                                         # whole_run: one gda_run of K steps, no flush
                out = P.run(x0, h.lambda0, prm_all, trace_cap=min(K, 4096))
                e1.record(stream)
                self.sync_all()
                res["t_whole"] = e0.elapsed_time(e1) / 1e3
                res["clocks"] = sampler.stop()
                res["trace"] = (out["trace_best"].cpu().numpy(), out["trace_ns"].cpu().numpy())
                # ---- e2e through gda_run_host, HOST buffers (pinned), copies inside the timed region ----
                xb_host = torch.empty((n, B), dtype=torch.uint8).pin_memory()
                obj_host = torch.empty(B, dtype=torch.float64).pin_memory()
                best_host = torch.empty(1, dtype=torch.int32).pin_memory()
                hp = (x0_host.data_ptr(), h.lambda0)
                op = (xb_host.data_ptr(), obj_host.data_ptr(), best_host.data_ptr(), stream.cuda_stream)
                P.run_host_ptrs(B, *hp, prm_step, *op)
                self.sync_all()
                w0 = time.perf_counter()                                  # (1) per step: H2D of the step's input, D2H of its result
                for _ in range(K):
                    P.run_host_ptrs(B, *hp, prm_step, *op)
                self.sync_all()
                res["t_e2e_steps"] = time.perf_counter() - w0
                w0 = time.perf_counter()                                  # (2) the way a user runs it: one call of K steps
                P.run_host_ptrs(B, *hp, prm_all, *op)
                self.sync_all()
                res["t_e2e_one_call"] = time.perf_counter() - w0
                res["h2d"] = x0_host.numel() * 4
                res["d2h"] = n * B + 8 * B + 4
                res["out"] = out
        res.update(step_ms=step_ms, t_eval=t_eval, launches=int(launches))
        res["roofline"] = roofline_block(w, peaks, sum(step_ms) / 1e3 / K, statistics.median(step_ms) / 1e3, t_eval)
        if w.kind == "qubo_csr" and res.get("chunk_fused"):
            props = torch.cuda.get_device_properties(self.dev)
            res["roofline"]["kernel"] = "spmm_chunk_slab (one launch = eval_every steps + the evaluation, state in shared memory)"
            res["roofline"]["on_chip"] = smem_roofline(w, res["roofline"]["us_per_launch"] * 1e-6, props.multi_processor_count,
                                                       (res["clocks"] or {}).get("sm_max_mhz") or 1965.0)
        res["P"] = P
        return res


def workload_tag(w: wl.Workload) -> str:
    return w.name + ("_pdbo_s" if getattr(w.hyper, "dual", 0) and "pdbo_s" not in w.name else "")


def secondary_line(w: wl.Workload, r, K):
    """One entry of `secondary`: the same measurement (K flushed steps, CUDA events) on another workload.  Numbers only: the
    prose of the roofline block (basis, sources) stays on the headline."""
    t = sum(r["step_ms"]) / 1e3
    roof = {k: v for k, v in r["roofline"].items() if not isinstance(v, str) or k in ("bound", "unit")}
    if "on_chip" in roof:
        roof["on_chip"] = {k: v for k, v in roof["on_chip"].items() if k != "basis"}
    return {"workload": workload_tag(w), "kind": w.kind, "n": w.problem.n, "B": w.B, "steps": K,
            "value": w.B * w.hyper.eval_every * K / t, "unit": "restart-iters/s", "ms_per_step": 1e3 * t / K,
            "ms_per_step_median": statistics.median(r["step_ms"]), "roofline": roof, "clocks": r["clocks"],
            "best_objective": r["best_flushed"], "gpu_launches": r["launches"]}


def summary_entry(w: wl.Workload, r):
    """[workload, B, us per GDA iteration (mean, median), bound, fraction of that bound's peak, SM MHz (median under load),
    clock samples, clock-event reasons] -- one short list per workload; `summary` is the LAST key of the JSON line."""
    roof, ck = r["roofline"], r["clocks"] or {}
    bound, frac = roof["bound"], roof["frac"]
    if "on_chip" in roof:                       # slab kernel: shared-memory bound
        bound, frac = roof["on_chip"]["bound"], roof["on_chip"]["frac"]
    elif "l2" in roof:                          # L2-resident state: the measured L2 -> SM ceiling is the honest one
        bound, frac = "l2", roof["l2"]["frac"]
    e = [workload_tag(w), w.B, round(roof["us_per_launch"], 2), round(roof["us_per_launch_median"], 2), bound, round(frac, 3),
         ck.get("sm_mhz"), ck.get("samples"), ck.get("reasons")]
    if roof["bound"] == "tensor":
        e += [{"frac_sustained": round(roof["frac"], 3), "frac_burst": round(roof["frac_burst"], 3)}]
    elif bound != "hbm":
        e += [{"hbm_algorithmic_frac": round(roof["frac"], 3)}]
    return e


def run_ours(args, w: wl.Workload):
    import torch
    import torch.distributed as dist
    from paper_2509_21064_b200 import api, build, multirank

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus != world and world > 1:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    api.lib()

    peaks = load_peaks()
    h, B, n = w.hyper, w.B, w.problem.n
    K, W = args.steps, max(args.warmup, 3)
    S = Session(local_rank, rank, world)
    r = S.measure(w, K, W, peaks, full=True)
    out, P = r["out"], r["P"]
    t_steps = multirank.max_over_ranks(sum(r["step_ms"]) / 1e3, world, dev)
    t_whole, t_e2e, t_e2e1 = (multirank.max_over_ranks(r[k], world, dev) for k in ("t_whole", "t_e2e_steps", "t_e2e_one_call"))
    best, best_rank, best_restart = multirank.combine_best(float(out["obj"].min().item()),
                                                            int(out["best_restart"].item()), rank, world, dev)
    launches = r["launches"]
    P.destroy()

    # ---- secondary workloads, same process, same method (default headline run on one GPU only) ----
    secondary, summary = [], []
    if world == 1 and not args.no_secondary and args.config == HEADLINE_CONFIG and not (args.mis or args.maxkcut or args.pdbo_s or args.B):
        Ks = max(5, min(K, args.secondary_steps))
        # the configs of BASELINE.json, config 3's graph at the paper's largest batch (HBM-streaming), PDBO-s, and two of the
        # paper's own small-batch settings (Max-k-SAT and MIS run B = 10: Table 6, 1040-1048 Table 13)
        # (ordered so that the BASELINE.json configs close the line: a log tail that is cut short still holds them)
        for sw in (wl.mis(10000, 100, B=10), wl.config(5, B=10), wl.pdbo_s_variant(wl.config(2)), wl.pdbo_s_variant(wl.config(3)),
                   wl.config(1), wl.config(3, B=1024), wl.config(2), wl.config(5), wl.config(4)):
            rs = S.measure(sw, Ks, 3, peaks, full=False, min_seconds=args.secondary_seconds)
            rs["P"].destroy()
            secondary.append(secondary_line(sw, rs, rs["K"]))
            summary.append(summary_entry(sw, rs))

    iters_per_step = h.eval_every
    units = world * B * iters_per_step * K
    tb_, tn_ = r["trace"]
    sel = sorted(set([0, len(tb_) // 4, len(tb_) // 2, len(tb_) - 1]))
    # device timestamps (globaltimer) of the evaluations; the run's start is the last evaluation minus the event-timed run
    t_end_ns = float(tn_[-1])
    ms_at = lambda i: max(0.0, t_whole * 1e3 - (t_end_ns - float(tn_[i])) / 1e6)
    trace = [{"ms": ms_at(i), "best": float(tb_[i])} for i in sel]
    first_best = int(np.argmax(tb_ == tb_[-1]))                # earliest evaluation that holds the final best

    if rank == 0:
        cpu = time_oracle(w, args.cpu_budget) if world == 1 and not args.no_cpu_baseline else None
        line = {
            "metric": "restart-iterations/s", "value": units / t_steps, "unit": "restart-iters/s",
            "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": 1e3 * t_steps / K,
            "ms_per_step_median": statistics.median(r["step_ms"]),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if w.kind != "qubo_dense" else "bf16 x bf16 -> f32 (state f32)", "data": "synthetic",
            "config": config_dict(args, w),
            "whole_run": {"value": units / t_whole, "unit": "restart-iters/s", "ms_total": 1e3 * t_whole,
                          "iters": iters_per_step * K, "l2": "not flushed (one gda_run call)", "best_objective": best,
                          "best_vs_time": trace, "time_to_best_ms": ms_at(first_best),
                          "time_to_best_note": "earliest evaluation at which the best objective of the run was held (PAPER.md:214), "
                                               "from the device-side globaltimer trace"},
            "e2e": {"value": units / t_e2e, "unit": "restart-iters/s", "h2d_bytes_per_step": r["h2d"],
                    "d2h_bytes_per_step": r["d2h"], "ms_total": 1e3 * t_e2e,
                    "note": "K calls of gda_run_host, one step each: every step copies its start point x0 from pinned host memory "
                            "(H2D) and reads x_bin / obj / best_restart back (D2H) inside the timed region (host wall clock)",
                    "one_call": {"value": units / t_e2e1, "ms_total": 1e3 * t_e2e1, "h2d_bytes": r["h2d"], "d2h_bytes": r["d2h"],
                                 "note": "the way a solver is used: ONE gda_run_host call of K steps, copies once"}},
            "gpu_launches": int(launches),
            "roofline": r["roofline"],
            "clocks": r["clocks"],
            "best_objective": best, "best_rank": best_rank, "best_restart": best_restart,
            "best_objective_flushed_run": r["best_flushed"],
        }
        if secondary:
            line["secondary"] = secondary
        if cpu:
            line["cpu_baseline"] = cpu
        # LAST key, compact: one entry per workload, the headline closing the list
        line["summary_fields"] = "workload,B,us_per_iter_mean,us_per_iter_median,bound,frac,sm_mhz_median,clock_samples,reasons[,more]"
        line["summary"] = summary + [summary_entry(w, r)]
        print(json.dumps(line, separators=(",", ":")))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=HEADLINE_CONFIG, help="BASELINE.json config, 1-based")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle time for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the secondary workloads of the default run")
    ap.add_argument("--secondary-steps", type=int, default=20, help="timed steps per secondary workload (at least)")
    ap.add_argument("--secondary-seconds", type=float, default=0.25,
                    help="a secondary workload is timed for at least this long (more steps, up to 400), for its clock record")
    ap.add_argument("--B", type=int, default=None)
    ap.add_argument("--pdbo-s", action="store_true", help="run the PDBO-s ablation (one multiplier per restart, PAPER.md:630-648)")
    ap.add_argument("--maxkcut", default=None, metavar="N,M,K", help="instead of --config: Max-K-Cut on G(N, M) (PAPER.md:784-828)")
    ap.add_argument("--mis", default=None, metavar="N,D", help="instead of --config: MIS as a QUBO on a D-regular graph with N vertices (PAPER.md:1030-1036)")
    args = ap.parse_args()
    if args.mis:
        n_mis, d_mis = (int(v) for v in args.mis.split(","))
        w = wl.mis(n_mis, d_mis, B=args.B or 12)
    elif args.maxkcut:
        n_k, m_k, k_k = (int(v) for v in args.maxkcut.split(","))
        w = wl.maxkcut(n_k, m_k, k_k, B=args.B or 128)
    else:
        w = wl.config(args.config, B=args.B)
    if args.pdbo_s:
        w = wl.pdbo_s_variant(w)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
