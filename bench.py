#!/usr/bin/env python
"""bench.py -- throughput of the batched lens-model likelihood (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config i]

A "step" is one pass of the whole hot path (DESIGN.md steps a0-a7: prologue, ray-trace, light,
bin, PSF convolution, chi^2 -> logL) over one batch of B synthetic parameter rows.  At N = 1 the
workload is BASELINE.json configs[1] (CSST-like 100x100, 4x4 supersampling, 21x21 PSF, B = 4096).
For N > 1 (torchrun, one process per GPU) every rank evaluates its own B rows: the path shards
over independent rows with no data-path collective ("scaling": "weak").

Prints ONE JSON line on rank 0.  --impl reference times the FP64 CPU oracle instead (the
deliberately slow checker).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2503_08586_b200 import workloads as W  # noqa: E402

METRIC = "likelihood evals/s"
UNIT = "likelihoods/s"

# ---- frozen algorithmic op model (BASELINE.md section 3 / SURVEY.md 8(d), op model v0) ----------
# FP32-pipe instruction slots (FMA = MUL = ADD = 1) and MUFU operations the METHOD needs per
# sub-sample; precision overhead (hi/lo constants, FP64 refinement, accurate-function
# polynomials) is not algorithmic work and is not counted.
OP_POS_FP32 = 2
OP_SIE_FP32, OP_SIE_MUFU = 46, 4
OP_SERSIC_FP32, OP_SERSIC_MUFU = 11, 3
OP_CHI2_FP32 = 4
# EPL (NEXT-2, --mass epl), same counting rules: shift/rotate 6; R^2 2; rsqrt (MUFU); e^{i phi} 3;
# e^{2 i phi} 4; Clenshaw recurrence 2 per series term + 4 to close it; radial factor
# (R^2/b^2)^kappa: 3 + lg2, ex2 (MUFU); Omega x radial 6; rotate back 4; shear + subtract 6.
OP_EPL_FP32, OP_EPL_FP32_PER_TERM, OP_EPL_MUFU = 38, 2, 3
SM_FP32_LANES = 128          # thread-instruction issue slots per SM per clock (4 warps x 32), measured 122-128
SM_MUFU_LANES = 16           # measured 15.96 (profiles/r2_peaks.md)

def ncu_dram_bytes(summary="r2_fused_kernel.md"):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, parsed from the
    committed `ncu --set full` summary under profiles/ (None when there is none)."""
    import re
    try:
        txt = open(os.path.join(ROOT, "profiles", summary)).read()
    except OSError:
        return None
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    tot, seen = 0.0, 0
    for name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        m = re.search(r"`%s`\s*\|\s*([0-9.eE+-]+)\s*\|\s*(\w+)" % re.escape(name), txt)
        if m and m.group(2) in unit:
            tot += float(m.group(1)) * unit[m.group(2)]
            seen += 1
    return int(round(tot)) if seen == 2 else None



def epl_mean_terms(rows: np.ndarray) -> float:
    """Mean number of angular-series terms a row needs for a truncation error below 2e-8 (FP32
    resolution): |a_{N+1}| < 2e-8 (1 - f), a_n = a_{n-1} (-f) (2n - (2-t)) / (2n + (2-t))."""
    e = np.hypot(rows[:, 1].astype(np.float64), rows[:, 2].astype(np.float64))     # f = (1-q)/(1+q) = |e|
    t = rows[:, 7].astype(np.float64) - 1.0
    an = np.ones_like(e)
    need = np.zeros_like(e)
    done = np.zeros(e.shape, bool)
    for n in range(1, 400):
        an = an * e * np.abs(2.0 * n - (2.0 - t)) / (2.0 * n + (2.0 - t))
        newly = (~done) & (an < 2e-8 * (1.0 - e))
        need[newly] = n - 1
        done |= newly
        if done.all():
            break
    need[~done] = 400
    return float(need.mean())


def op_model(w: W.Workload, rows=None) -> dict:
    ncomp = w.n_lens_light + w.n_source
    samples = w.samples_per_likelihood
    if w.mass_model == W.MASS_EPL:
        mass_fp32 = OP_EPL_FP32 + OP_EPL_FP32_PER_TERM * epl_mean_terms(rows)
        mass_mufu = OP_EPL_MUFU
    else:
        mass_fp32, mass_mufu = OP_SIE_FP32, OP_SIE_MUFU
    fp32 = samples * (OP_POS_FP32 + mass_fp32 + ncomp * OP_SERSIC_FP32) \
        + w.ny * w.nx * (w.psf_size ** 2 + OP_CHI2_FP32)
    mufu = samples * (mass_mufu + ncomp * OP_SERSIC_MUFU)
    return {"fp32_slots": fp32, "mufu_ops": mufu, "issue_slots": fp32 + mufu, "samples": samples}


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region (NVML in-process, every
    20 ms; falls back to polling nvidia-smi when pynvml is unavailable)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx, self.sm, self.mx, self.reasons, self.stop, self.t = gpu_index, [], [], set(), False, None
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            # NVML enumerates physical devices: honour CUDA_VISIBLE_DEVICES when it lists indices
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            phys = gpu_index
            if vis and all(v.strip().isdigit() for v in vis.split(",")):
                phys = int(vis.split(",")[gpu_index])
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        self.sm.append(float(n.nvmlDeviceGetClockInfo(self.h, n.NVML_CLOCK_SM)))
        self.mx.append(float(n.nvmlDeviceGetMaxClockInfo(self.h, n.NVML_CLOCK_SM)))
        try:
            r = n.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            r = n.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        for name, bit in (("hw_slowdown", 0x8), ("sw_power_cap", 0x4), ("sw_thermal_slowdown", 0x20),
                          ("hw_thermal_slowdown", 0x40)):
            if r & bit:
                self.reasons.add(name)

    def _sample_smi(self):
        out = subprocess.run(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                              "--format=csv,noheader,nounits"], capture_output=True, text=True,
                             timeout=5).stdout.strip()
        if not out:
            return
        r = [x.strip() for x in out.split(",")]
        self.sm.append(float(r[0])); self.mx.append(float(r[1]))
        for n, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[4:8]):
            if v.lower().startswith("active"):
                self.reasons.add(n)

    def _run(self):
        while not self.stop:
            try:
                if self.nvml is not None:
                    self._sample_nvml()
                else:
                    self._sample_smi()
            except Exception:
                pass
            time.sleep(0.02 if self.nvml is not None else 0.1)

    def __enter__(self):
        self.t = threading.Thread(target=self._run, daemon=True)
        self.t.start()
        return self

    def __exit__(self, *exc):
        self.stop = True
        self.t.join(timeout=10)

    def summary(self) -> dict:
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None,
                "sm_max_mhz": float(max(self.mx)) if self.mx else None,
                "reasons": sorted(self.reasons), "samples": len(self.sm),
                "source": "nvml" if self.nvml is not None else "nvidia-smi"}


def measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def oracle_time(w: W.Workload, prob, rows: np.ndarray, threads: int = 0, mode: str = "fixed", sigmas=None):
    from oracle import oracle as O
    cfg = O.config_of(w)
    t0 = time.perf_counter()
    if mode == "linear":
        O.loglike_linear_batch(cfg, prob.psf, prob.data, prob.noise, rows, n_lens=w.n_lens, threads=threads)
        used = os.cpu_count()
    elif mode == "mge":
        O.loglike_mge_batch(cfg, prob.psf, prob.data, prob.noise, rows, sigmas, n_lens=w.n_lens, threads=threads)
        used = os.cpu_count()
    else:
        _, used = O.loglike_batch(cfg, prob.psf, prob.data, prob.noise, rows, n_lens=w.n_lens, threads=threads)
    return time.perf_counter() - t0, used


def reference_problem(w: W.Workload):
    """Inputs for the reference arm: data from the oracle's own renderer."""
    from oracle import oracle as O
    return W.make_problem(w, O.render_for_workloads)


def run_reference(args, w: W.Workload):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    O.lib()
    prob = reference_problem(w)
    rows_all = W.batch_rows(w)
    n = args.ref_rows
    mode_tag, sigmas = "", None
    if args.mode == "linear":
        n = min(n, 128); mode_tag = " (linear amplitudes, NNLS per row)"
    elif args.mode == "mge":
        n = min(n, 64); sigmas = W.mge_sigmas(w, args.n_gauss)
        mode_tag = " (MGE lens light, %d Gaussians + %d source amplitudes by NNLS per row)" % (len(sigmas), w.n_source)
    # bounded sample per step: the first n rows of each step's window of the workload
    times, used = [], 1
    for s in range(args.warmup + args.steps):
        lo = (s * n) % max(1, len(rows_all) - n)
        dt, used = oracle_time(w, prob, rows_all[lo:lo + n], mode=args.mode, sigmas=sigmas)
        if s >= args.warmup:
            times.append(dt)
    tot = float(np.sum(times))
    value = n * len(times) / tot
    line = {
        "impl": "reference", "metric": METRIC + mass_tag(w) + mode_tag, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": config_dict(w, "none (CPU)"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle",
                         "sample": "%d of the %d rows per step" % (n, w.batch)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "pixel_evals_per_s": value * w.ny * w.nx, "gpu_launches": 0,
    }
    print(json.dumps(line))


def mass_tag(w: W.Workload) -> str:
    return " (EPL mass model)" if w.mass_model == W.MASS_EPL else ""


def config_dict(w: W.Workload, l2: str) -> dict:
    return {"workload": "BASELINE.json configs[%d] %s: %dx%d px, %.3g\"/px, %dx%d supersampling, %dx%d %s PSF, "
                        "%s+shear, %d lens-light + %d source Sersic, B=%d rows/GPU%s"
                        % (w.index, w.name, w.ny, w.nx, w.pix_scale, w.supersample, w.supersample, w.psf_size,
                           w.psf_size, w.psf_kind, "EPL (free slope)" if w.mass_model == W.MASS_EPL else "SIE",
                           w.n_lens_light, w.n_source, w.batch,
                           (", %d lenses" % w.n_lens) if w.n_lens > 1 else ""),
            "batch_per_gpu": w.batch, "n_params": w.n_params, "l2": l2, "parallelism": "rows sharded, no collective"}


def run_ours(args, w: W.Workload):
    import torch
    import torch.distributed as dist
    from paper_2503_08586_b200 import api

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    use_dist = world > 1 or "TORCHELASTIC_RUN_ID" in os.environ      # under torchrun, even with one rank
    if use_dist:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    # mock data = model(truth) + noise, the model coming from the library's own renderer
    def gpu_render(w1, psf, row):
        ctx = api.LensContext(w1.ny, w1.nx, w1.pix_scale, w1.supersample, w1.n_lens_light, w1.n_source,
                              psf[None], np.zeros((1, w1.ny, w1.nx), np.float32),
                              np.ones((1, w1.ny, w1.nx), np.float32), w1.edge_mode, mass_model=w1.mass_model)
        im = ctx.render(torch.from_numpy(np.ascontiguousarray(row[None])).to(dev)).cpu().numpy()[0]
        ctx.close()
        return im

    prob = W.make_problem(w, gpu_render)
    ctx = api.LensContext.from_problem(prob)
    PREC = {"fp32": api.TL_PRECISION_FP32, "fp64": api.TL_PRECISION_FP64, "fp64-libm": api.TL_PRECISION_FP64_LIBM,
            "auto": api.TL_PRECISION_AUTO}
    if args.precision != "fp32":
        ctx.set_precision(PREC[args.precision])
    info = ctx.info()
    # each rank draws its own rows (weak scaling): stream id offset by rank
    rows = W.batch_rows(w) if rank == 0 else \
        np.concatenate([W.draw_params(w, W.rng_for(w.index, W.STREAM_BATCH + 16 * rank, l), w.rows_per_lens)
                        for l in range(w.n_lens)], axis=0)
    if args.rows == "near-truth":
        rows = W.near_truth_rows(prob, w.rows_per_lens)
    B = rows.shape[0]
    d_rows = torch.from_numpy(rows).to(dev)
    d_out = torch.empty(B, dtype=torch.float32, device=dev)
    h_rows = torch.from_numpy(rows).pin_memory()
    h_out = torch.empty(B, dtype=torch.float32).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def barrier():
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    stream = torch.cuda.current_stream()
    if args.streams > 1:
        run_streams(args, w, ctx, info, d_rows, d_out, rows, clk_dev=local)
        return
    ctx.set_profiling(True)
    clk = ClockSampler(local)
    clk.__enter__()                      # samples through warm-up, the timed steps and the e2e loop
    for _ in range(max(args.warmup, 3)):
        ctx.loglike(d_rows, d_out)
    torch.cuda.synchronize()

    # ---- device-resident timing: K steps, L2 flushed between steps, CUDA events per step -------
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms = []
    if True:
        barrier()
        for s in range(args.steps):
            flush.fill_(s & 0xff)
            ev[s][0].record(stream)
            ctx.loglike(d_rows, d_out)
            ev[s][1].record(stream)
            kern_ms.append(ctx.last_kernel_ms())      # waits for the kernel; keeps steps separate
        barrier()
        step_ms = [a.elapsed_time(b) for a, b in ev]
        # ---- end to end through the host entry point (H2D + kernels + D2H + sync per step) ----
        for _ in range(2):
            ctx.loglike_host(h_rows, h_out)
        barrier()
        t0 = time.perf_counter()
        for s in range(args.steps):
            ctx.loglike_host(h_rows, h_out)
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        barrier()
        # ---- sampler-like loop through the asynchronous host entry: batch k + 1 is submitted (its upload
        # overlapping the kernels of batch k) before batch k is waited for ----
        pipelined = []
        if world == 1 and args.precision == "fp32":
            for pb in (74, 300, 4096):
                if pb > B or pb % w.n_lens:
                    continue
                hp = h_rows[:pb].contiguous().pin_memory()
                outs = [torch.empty(pb, dtype=torch.float32).pin_memory() for _ in range(2)]
                nbat = 40
                ctx.wait(ctx.loglike_host_async(hp, outs[0]))
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                prev = ctx.loglike_host_async(hp, outs[0])
                for k in range(1, nbat):
                    cur = ctx.loglike_host_async(hp, outs[k & 1])
                    ctx.wait(prev)
                    prev = cur
                ctx.wait(prev)
                dt_pipe = time.perf_counter() - t0
                t0 = time.perf_counter()
                for k in range(nbat):
                    ctx.loglike_host(hp, outs[0])
                dt_sync = time.perf_counter() - t0
                dsub = d_rows[:pb].contiguous()
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                for k in range(nbat):
                    ctx.loglike(dsub, d_out[:pb])
                e1.record(stream)
                torch.cuda.synchronize()
                pipelined.append({"B": pb, "batches": nbat, "pipelined_per_s": pb * nbat / dt_pipe, "sync_per_s": pb * nbat / dt_sync,
                                  "device_resident_per_s": pb * nbat / (e0.elapsed_time(e1) * 1e-3)})
    clk.__exit__(None, None, None)
    clocks = clk.summary()
    total_ms = float(np.sum(step_ms))
    logl_sum = float(h_out.double().sum())

    if use_dist:
        t = torch.tensor([total_ms, e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, e2e_s = float(t[0]), float(t[1])
    if rank != 0:
        if use_dist:
            dist.destroy_process_group()
        return

    value = world * B * args.steps / (total_ms * 1e-3)
    e2e_value = world * B * args.steps / e2e_s
    om = op_model(w, rows)
    peaks = measured_peaks()
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    k_ms = float(np.mean(kern_ms))
    # a call of more than chunk_rows rows is several launches; the events are around the last one
    k_rows = B - ((B - 1) // info["chunk_rows"]) * info["chunk_rows"]
    whole_step = info["path"] == 1 or args.precision != "fp32"
    if whole_step:
        # split path (large images) and the FP64 / AUTO modes: several kernels share the work of the op
        # model, so the fraction is taken over the whole step, not over one kernel
        k_ms, k_rows = total_ms / args.steps, B
    achieved = om["issue_slots"] * k_rows / (k_ms * 1e-3) / 1e12     # algorithmic Tinst/s
    peak = info["n_sm"] * SM_FP32_LANES * sm_max * 1e6 / 1e12
    mufu_frac = om["mufu_ops"] * k_rows / (k_ms * 1e-3) / (info["n_sm"] * SM_MUFU_LANES * sm_max * 1e6)
    fp32_frac = om["fp32_slots"] * k_rows / (k_ms * 1e-3) / (info["n_sm"] * SM_FP32_LANES * sm_max * 1e6)
    hbm_bytes = B * (w.n_params + 1) * 4 + (2 * w.ny * w.nx + w.psf_size ** 2) * 4 * w.n_lens
    line = {
        "metric": METRIC + mass_tag(w), "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": {"fp32": "f32", "auto": "f32+f64"}.get(args.precision, "f64"),
        "data": "synthetic", "precision": args.precision, "rows": args.rows,
        "config": config_dict(w, "flushed between steps (256 MiB fill)"),
        "pixel_evals_per_s": value * w.ny * w.nx,
        "sample_evals_per_s": value * om["samples"],
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": B * w.n_params * 4,
                "d2h_bytes_per_step": B * 4, "api": "tl_loglike_batch_host (pinned host buffers)"},
        "e2e_pipelined": pipelined,
        "gpu_launches": ({"fp64": 4, "fp64-libm": 2}.get(args.precision,
                                                         (3 if (B <= info["small_batch_rows"] and args.precision == "fp32") else info["launches_per_call"])
                                                         + (4 if args.precision == "auto" else 0))
                         * ((B + info["chunk_rows"] - 1) // info["chunk_rows"] if args.precision in ("fp32", "auto") else 1)) * args.steps,
        "roofline": {
            "bound": "alu", "kernel": ("whole step (all kernels)" if whole_step else
                                       "fused_kernel" if B > info["small_batch_rows"] else "trace_kernel + conv_small_kernel"),
            "achieved": achieved, "peak": peak, "unit": "Tinst/s", "frac": achieved / peak,
            "traffic": ncu_dram_bytes() if (w.mass_model == W.MASS_SIE and w.index == 1 and args.precision == "fp32"
                                            and args.rows == "prior") else None,
            "peak_source": "derived: %d SMs x %d issue slots/clk x %.0f MHz (MEASURED_PEAKS.json sm_max_mhz; "
                           "slots/clk measured, profiles/r2_peaks.md)" % (info["n_sm"], SM_FP32_LANES, sm_max),
            "kernel_ms": k_ms, "kernel_rows": k_rows, "fp32_pipe_frac": fp32_frac, "mufu_pipe_frac": mufu_frac,
            "algorithmic_issue_slots_per_likelihood": om["issue_slots"],
            **({"epl_mean_series_terms": epl_mean_terms(rows)} if w.mass_model == W.MASS_EPL else {}),
            "hbm": {"algorithmic_bytes_per_step": hbm_bytes,
                    "achieved_GBs": hbm_bytes * (k_rows / B) / (k_ms * 1e-3) / 1e9,
                    "peak_GBs": peaks.get("hbm_gbs"), "note": "compute-bound by design; HBM traffic is negligible"},
        },
        **({"roofline_fp64": {"bound": "alu", "note": "FP64 pipe: 64 DFMA lanes/clk/SM; op model v0 with every FP32 slot and every "
                              "transcendental counted as ONE FP64 operation (the polynomials are overhead)",
                              "achieved": (om["fp32_slots"] + om["mufu_ops"]) * B / (total_ms / args.steps * 1e-3) / 1e12,
                              "peak": info["n_sm"] * 64 * sm_max * 1e6 / 1e12, "unit": "Tinst/s",
                              "frac": (om["fp32_slots"] + om["mufu_ops"]) * B / (total_ms / args.steps * 1e-3) / (info["n_sm"] * 64 * sm_max * 1e6)}}
           if args.precision == "fp64" else {}),
        "launch": {**{k: info[k] for k in ("path", "block_threads", "ctas_per_sm", "grid", "smem_bytes")},
                   "small_batch_path": bool(B <= info["small_batch_rows"])},
        "checksum_logL": logl_sum,
    }
    if world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as O
        O.lib()
        n = args.ref_rows
        dt, used = oracle_time(w, prob, rows[:n])
        line["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": used, "kind": "oracle", "per_core": n / dt / max(1, used),
                                "sample": "first %d of the %d rows of the step, %.1f s" % (n, B, dt)}
    print(json.dumps(line))
    if use_dist:
        dist.destroy_process_group()


def run_streams(args, w, ctx, info, d_rows, d_out, rows, clk_dev=0):
    """The batch as sub-batches of --sub-batch rows issued round-robin on --streams streams that share
    one context (BASELINE configs[4]: "B = 65536 split across streams on one GPU").  Timed on the
    device: a start event all streams wait for, an end event per stream, the latest end counts."""
    import torch
    B = rows.shape[0]
    sub = min(args.sub_batch, B)
    if w.n_lens > 1:
        raise SystemExit("--streams: single-lens workloads only")
    streams = [torch.cuda.Stream() for _ in range(args.streams)]
    chunks = [(lo, min(B, lo + sub)) for lo in range(0, B, sub)]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=d_rows.device)

    def issue():
        for k, (lo, hi) in enumerate(chunks):
            st = streams[k % len(streams)]
            ctx.loglike(d_rows[lo:hi], d_out[lo:hi], stream=st)

    for _ in range(max(1, min(args.warmup, 2))):
        issue()
    torch.cuda.synchronize()
    steps = args.steps
    times = []
    with ClockSampler(clk_dev) as clk:
        for s in range(steps):
            flush.fill_(s & 0xff)
            start = torch.cuda.Event(enable_timing=True)
            ends = [torch.cuda.Event(enable_timing=True) for _ in streams]
            start.record(torch.cuda.current_stream())
            for st in streams:
                st.wait_event(start)
            issue()
            for st, e in zip(streams, ends):
                e.record(st)
            torch.cuda.synchronize()
            times.append(max(start.elapsed_time(e) for e in ends))
    total_ms = float(np.sum(times))
    value = B * steps / (total_ms * 1e-3)
    om = op_model(w, rows)
    sm_max = float(measured_peaks().get("sm_max_mhz", 1965.0))
    peak = info["n_sm"] * SM_FP32_LANES * sm_max * 1e6 / 1e12
    ach = om["issue_slots"] * B * steps / (total_ms * 1e-3) / 1e12
    launches = (3 if sub <= info["small_batch_rows"] else info["launches_per_call"]) * len(chunks) * steps
    print(json.dumps({
        "metric": METRIC + mass_tag(w), "value": value, "unit": UNIT, "n_gpus": 1, "steps": steps, "warmup": max(1, min(args.warmup, 2)),
        "ms_per_step": total_ms / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {"fp32": "f32", "auto": "f32+f64"}.get(args.precision, "f64"), "data": "synthetic", "precision": args.precision,
        "config": config_dict(w, "flushed between steps (256 MiB fill)"),
        "streams": args.streams, "sub_batch_rows": sub, "sub_batches": len(chunks),
        "pixel_evals_per_s": value * w.ny * w.nx, "sample_evals_per_s": value * om["samples"], "clocks": clk.summary(),
        "gpu_launches": launches,
        "roofline": {"bound": "alu", "kernel": "whole step (all sub-batches, all kernels)", "achieved": ach, "peak": peak, "unit": "Tinst/s",
                     "frac": ach / peak, "traffic": None, "algorithmic_issue_slots_per_likelihood": om["issue_slots"],
                     "peak_source": "derived: %d SMs x %d issue slots/clk x %.0f MHz" % (info["n_sm"], SM_FP32_LANES, sm_max)},
        "checksum_logL": float(d_out.double().sum())}))


def run_linear(args, w: W.Workload):
    """Secondary line: the paper's linear/non-linear split (NEXT-1).  Same workload, amplitudes
    solved per row; value = rows / device time (CUDA events), oracle timed on a bounded sample."""
    import torch
    from paper_2503_08586_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    dev = torch.device("cuda", 0)

    def gpu_render(w1, psf, row):
        ctx = api.LensContext(w1.ny, w1.nx, w1.pix_scale, w1.supersample, w1.n_lens_light, w1.n_source,
                              psf[None], np.zeros((1, w1.ny, w1.nx), np.float32),
                              np.ones((1, w1.ny, w1.nx), np.float32), w1.edge_mode, mass_model=w1.mass_model)
        im = ctx.render(torch.from_numpy(np.ascontiguousarray(row[None])).to(dev)).cpu().numpy()[0]
        ctx.close()
        return im

    prob = W.make_problem(w, gpu_render)
    ctx = api.LensContext.from_problem(prob)
    if args.precision != "fp32" and args.mode in ("linear", "mge"):
        ctx.set_precision({"fp64": api.TL_PRECISION_FP64, "fp64-libm": api.TL_PRECISION_FP64_LIBM, "auto": api.TL_PRECISION_AUTO}[args.precision])
    rows = W.batch_rows(w)
    B = rows.shape[0]
    mge = args.mode == "mge"
    if mge:
        run_mge(args, w, prob, ctx, rows)
        return
    d_rows = torch.from_numpy(rows).to(dev)
    out = torch.empty(B, dtype=torch.float32, device=dev)
    amps = torch.empty((B, w.n_lens_light + w.n_source), dtype=torch.float32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ctx.set_profiling(True)
    for _ in range(max(args.warmup, 3)):
        ctx.loglike_linear(d_rows, out, amps)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms = []
    with ClockSampler(0) as clk:
        for s in range(args.steps):
            flush.fill_(s & 0xff)
            ev[s][0].record(); ctx.loglike_linear(d_rows, out, amps); ev[s][1].record()
            kern_ms.append(ctx.last_kernel_ms())
        torch.cuda.synchronize()
    total_ms = float(np.sum([a.elapsed_time(b) for a, b in ev]))
    value = B * args.steps / (total_ms * 1e-3)
    line = {"metric": METRIC + mass_tag(w) + " (linear amplitudes, NNLS per row)", "value": value, "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if args.precision == "fp32" else "f64", "precision": args.precision, "data": "synthetic",
            "config": config_dict(w, "flushed between steps (256 MiB fill)"), "clocks": clk.summary(),
            "pixel_evals_per_s": value * w.ny * w.nx, "mode": "linear",
            "gpu_launches": args.steps * (2 if args.precision == "fp32" else 4), "checksum_logL": float(out.double().sum())}
    # roofline of the fused linear kernel: op model v0 per sample (unchanged) + per native pixel
    # C convolutions, the Gram matrix / right-hand side (C (C + 3)) and the residual (C + 3)
    C_ = w.n_lens_light + w.n_source
    om = op_model(w, rows)
    slots = om["issue_slots"] + w.ny * w.nx * ((C_ - 1) * w.psf_size ** 2 + C_ * (C_ + 3) + C_ + 3 - OP_CHI2_FP32)
    info = ctx.info()
    sm_max = float(measured_peaks().get("sm_max_mhz", 1965.0))
    k_ms = float(np.mean(kern_ms))
    ach = slots * B / (k_ms * 1e-3) / 1e12
    peak = info["n_sm"] * SM_FP32_LANES * sm_max * 1e6 / 1e12
    line["roofline"] = {"bound": "alu", "kernel": "fused_lin_kernel", "achieved": ach, "peak": peak, "unit": "Tinst/s",
                        "frac": ach / peak, "traffic": None, "kernel_ms": k_ms,
                        "algorithmic_issue_slots_per_likelihood": slots,
                        "peak_source": "as in the default mode"}
    if args.precision != "fp32":
        # FP64 pipeline: several kernels; the fraction is taken over the whole step against the same issue roofline
        ach = slots * B / (total_ms / args.steps * 1e-3) / 1e12
        line["roofline"] = {"bound": "alu", "kernel": "whole step (trace_dp + conv_dp + solve_dp)", "achieved": ach, "peak": peak,
                            "unit": "Tinst/s", "frac": ach / peak, "traffic": None, "kernel_ms": total_ms / args.steps}
    if not args.no_cpu_baseline:
        from oracle import oracle as O
        O.lib()
        n = min(args.ref_rows, 128)
        t0 = time.perf_counter()
        O.loglike_linear_batch(O.config_of(w), prob.psf, prob.data, prob.noise, rows[:n], n_lens=w.n_lens)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                                "sample": "first %d of the %d rows, %.1f s" % (n, B, dt)}
    print(json.dumps(line))


def run_mge(args, w: W.Workload, prob, ctx, rows):
    """Secondary line: MGE lens light with linear amplitudes (NEXT-3, tl_loglike_mge_batch): the
    same workload, its lens light fitted by n_gauss elliptical Gaussians, n_gauss + n_source
    amplitudes solved per row."""
    import torch
    from paper_2503_08586_b200 import api
    dev = torch.device("cuda", 0)
    sigmas = W.mge_sigmas(w, args.n_gauss)
    ctx.set_mge(sigmas)
    B = rows.shape[0]
    NC = len(sigmas) + w.n_source
    d_rows = torch.from_numpy(rows).to(dev)
    out = torch.empty(B, dtype=torch.float32, device=dev)
    amps = torch.empty((B, NC), dtype=torch.float32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ctx.set_profiling(True)
    for _ in range(max(args.warmup, 3)):
        ctx.loglike_mge(d_rows, out, amps)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms = []
    with ClockSampler(0) as clk:
        for s in range(args.steps):
            flush.fill_(s & 0xff)
            ev[s][0].record(); ctx.loglike_mge(d_rows, out, amps); ev[s][1].record()
            kern_ms.append(ctx.last_kernel_ms())
        torch.cuda.synchronize()
    total_ms = float(np.sum([a.elapsed_time(b) for a, b in ev]))
    value = B * args.steps / (total_ms * 1e-3)
    chunk = api.tl_mge_chunk_rows(ctx.handle)
    n_chunks = (B + chunk - 1) // chunk
    last_rows = B - (n_chunks - 1) * chunk
    line = {"metric": METRIC + mass_tag(w) + " (MGE lens light, %d Gaussians + %d source amplitudes by NNLS per row)" % (len(sigmas), w.n_source),
            "value": value, "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if args.precision == "fp32" else "f64", "precision": args.precision, "data": "synthetic",
            "config": config_dict(w, "flushed between steps (256 MiB fill)"), "clocks": clk.summary(),
            "pixel_evals_per_s": value * w.ny * w.nx, "mode": "mge", "mge_sigmas_arcsec": [float(x) for x in sigmas],
            "chunk_rows": int(chunk), "gpu_launches": int(args.steps * 6 * n_chunks), "checksum_logL": float(out.double().sum())}
    # (the events bracket the gauss_conv launch of the call's last chunk)
    info = ctx.info()
    sm_max = float(measured_peaks().get("sm_max_mhz", 1965.0))
    k_ms = float(np.mean(kern_ms))
    # dominant kernel: gauss_conv_kernel -- per Gaussian, 4 slots per sub-sample (t from its row / column parts,
    # scale, MUFU.EX2, accumulate) and the PSF convolution (K^2 FMAs per native pixel)
    slots = len(sigmas) * (4 * w.samples_per_likelihood + w.psf_size ** 2 * w.ny * w.nx)
    ach = slots * last_rows / (k_ms * 1e-3) / 1e12
    peak = info["n_sm"] * SM_FP32_LANES * sm_max * 1e6 / 1e12
    line["roofline"] = {"bound": "alu", "kernel": "gauss_conv_kernel", "achieved": ach, "peak": peak, "unit": "Tinst/s",
                        "frac": ach / peak, "traffic": None, "kernel_ms": k_ms, "kernel_rows": int(last_rows),
                        "algorithmic_issue_slots_per_likelihood": slots,
                        "peak_source": "as in the default mode (FP32 FMA issue slots)",
                        "note": "the slots are those of evaluating and blurring every Gaussian over the whole image; the kernel "
                                "leaves out the part of a narrow Gaussian that is exactly 0 (DESIGN.md 13), so the fraction of "
                                "what it executes is lower (profiles/r2_modes.md: issue port, FMA pipe)"}
    if args.precision != "fp32":
        # FP64 pipeline (trace_dp / gauss_dp / conv_dp / gram / nnls): the fraction over the whole step, same issue roofline
        ach = slots * B / (total_ms / args.steps * 1e-3) / 1e12
        line["roofline"] = {"bound": "alu", "kernel": "whole step (FP64 MGE pipeline)", "achieved": ach, "peak": peak,
                            "unit": "Tinst/s", "frac": ach / peak, "traffic": None, "kernel_ms": total_ms / args.steps}
    if not args.no_cpu_baseline:
        from oracle import oracle as O
        O.lib()
        n = min(args.ref_rows, 64)
        t0 = time.perf_counter()
        O.loglike_mge_batch(O.config_of(w), prob.psf, prob.data, prob.noise, rows[:n], sigmas, n_lens=w.n_lens)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                                "sample": "first %d of the %d rows, %.1f s" % (n, B, dt)}
    print(json.dumps(line))


def run_peaks(args):
    """`--peaks`: the committed pipe micro-benchmarks (tl_measure_peaks) as one JSON line."""
    import torch
    from paper_2503_08586_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(0)
    with ClockSampler(0) as clk:
        probes, err = api.tl_measure_peaks()
    print(json.dumps({"peaks": probes, "clocks": clk.summary(),
                      "fp64_seed_rel_err": {"rcp.approx.f64": err[0], "rcp + 1 Newton": err[1],
                                            "rsqrt.approx.f64": err[2], "rsqrt + 1 Newton": err[3]}}))


def run_serve(args):
    """`--serve`: host-to-host latency of small requests through the persistent serving kernel (tl_serve_eval)
    beside the ordinary host entry point (tl_loglike_batch_host), configs[`--config`], as one JSON line."""
    import torch
    from paper_2503_08586_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(0)
    w = W.workload(args.config)
    dev = torch.device("cuda", 0)

    def gpu_render(w1, psf, row):
        ctx = api.LensContext(w1.ny, w1.nx, w1.pix_scale, w1.supersample, w1.n_lens_light, w1.n_source,
                              psf[None], np.zeros((1, w1.ny, w1.nx), np.float32),
                              np.ones((1, w1.ny, w1.nx), np.float32), w1.edge_mode, mass_model=w1.mass_model)
        im = ctx.render(torch.from_numpy(np.ascontiguousarray(row[None])).to(dev)).cpu().numpy()[0]
        ctx.close()
        return im

    prob = W.make_problem(w, gpu_render)
    ctx = api.LensContext.from_problem(prob)
    rows = W.batch_rows(w, 16)
    res = []
    with ClockSampler(0) as clk:
        for B in (1, 2, 4, 8, 16):
            r = np.ascontiguousarray(rows[:B])
            out = np.empty(B, np.float32)
            for _ in range(20):
                ctx.loglike_host(r)
            t0 = time.perf_counter()
            for _ in range(200):
                ctx.loglike_host(r)
            t_host = (time.perf_counter() - t0) / 200
            ref = ctx.loglike_host(r)
            ctx.serve_start(max_rows=16, idle_timeout_s=1.0)
            try:
                for _ in range(50):
                    ctx.serve_eval(r, out)
                t0 = time.perf_counter()
                for _ in range(1000):
                    ctx.serve_eval(r, out)
                t_serve = (time.perf_counter() - t0) / 1000
            finally:
                ctx.serve_stop()
            res.append({"B": B, "served_us": 1e6 * t_serve, "host_entry_us": 1e6 * t_host,
                        "served_per_s": B / t_serve, "host_entry_per_s": B / t_host,
                        "bitwise_equal": bool(np.array_equal(np.asarray(ref), out))})
    print(json.dumps({"metric": "host-to-host latency of a small request", "unit": "us", "higher_is_better": False,
                      "config": config_dict(w, "n/a (one request at a time)"), "requests": res, "clocks": clk.summary(),
                      "data": "synthetic", "dtype": "f32"}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index (default 1, the metric's)")
    ap.add_argument("--batch", type=int, default=0, help="override rows per GPU (parity/debug only)")
    ap.add_argument("--ref-rows", type=int, default=512, help="oracle sample size per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mode", default="fixed", choices=["fixed", "linear", "mge"],
                    help="fixed: amplitudes are parameters (the headline metric); linear: amplitudes solved by NNLS "
                         "per row (tl_loglike_linear_batch, PAPER.md Eq. 6-7) -- a secondary line; mge: the lens "
                         "light as n_gauss elliptical Gaussians with NNLS amplitudes (tl_loglike_mge_batch, "
                         "PAPER.md:291-293) -- a secondary line")
    ap.add_argument("--n-gauss", type=int, default=10, help="--mode mge: Gaussians in the lens-light set (<= 16)")
    ap.add_argument("--mass", default="sie", choices=["sie", "epl"],
                    help="sie: the headline workload; epl: the same workload with the elliptical power-law mass "
                         "model and a free slope per row (NEXT-2, PAPER.md Eq. 12) -- a secondary line")
    ap.add_argument("--precision", default="fp32", choices=["fp32", "fp64", "fp64-libm", "auto"],
                    help="fp32: the headline kernels; fp64: every per-sample quantity in FP64 with polynomial functions "
                         "(meets north_star on rows near the best fit too); fp64-libm: CUDA's double math library "
                         "(slow cross-check); auto: FP32, then FP64 for the rows whose FP32 error bound exceeds the tolerance")
    ap.add_argument("--rows", default="prior", choices=["prior", "near-truth"],
                    help="prior: the BASELINE batch (independent prior draws); near-truth: truth (1 + 1e-3 N(0,1)) rows, "
                         "the regime a converged sampler works in (SURVEY.md 8(d) near-truth slice)")
    ap.add_argument("--streams", type=int, default=1,
                    help="issue the batch as sub-batches on this many CUDA streams sharing one context "
                         "(BASELINE configs[4]: B = 65536 split across streams); with --sub-batch rows per sub-batch")
    ap.add_argument("--sub-batch", type=int, default=4096, help="rows per sub-batch when --streams > 1")
    ap.add_argument("--peaks", action="store_true",
                    help="run the pipe micro-benchmarks (tl_measure_peaks: FFMA, FFMA2, MUFU, DFMA and mixes) and exit")
    ap.add_argument("--all-configs", action="store_true",
                    help="one JSON line per BASELINE.json config (0..4), each from a run of this script with --config i "
                         "(config 4: 2 steps); the other options are passed on")
    ap.add_argument("--serve", action="store_true",
                    help="latency of 1..16-row requests through the persistent serving kernel (tl_serve_eval) and exit")
    args = ap.parse_args()
    if args.peaks:
        run_peaks(args)
        return
    if args.serve:
        run_serve(args)
        return
    if args.all_configs:
        import subprocess
        rest = [x for x in sys.argv[1:] if x != "--all-configs"]
        for i in range(5):
            cmd = [sys.executable, os.path.abspath(__file__), "--config", str(i), "--no-cpu-baseline"] + rest + (["--steps", "2"] if i == 4 else [])
            out = subprocess.run(cmd, stdout=subprocess.PIPE, text=True).stdout.strip().splitlines()
            print(out[-1] if out else json.dumps({"config": i, "error": "no output"}), flush=True)
        return
    w = W.workload(args.config)
    if args.mass == "epl":
        w = w.with_epl()
    if args.batch:
        w = w.scaled(batch=args.batch)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus and world > 1:
        raise SystemExit("--gpus %d does not match WORLD_SIZE %d" % (args.gpus, world))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        # not under torchrun: launch one rank per GPU ourselves (same command line), NCCL's own
        # communicator log left on (stderr) so that the transport it picked is on record
        import socket
        import torch
        if torch.cuda.device_count() < args.gpus:
            raise SystemExit("bench.py: --gpus %d but only %d CUDA device(s) visible" % (args.gpus, torch.cuda.device_count()))
        sk = socket.socket(); sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]; sk.close()
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "INFO")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd, env=env))
    if args.mode == "mge" and w.n_lens_light != 1:
        raise SystemExit("bench.py --mode mge needs a workload with lens light (configs 1-4)")
    if args.impl == "reference":
        run_reference(args, w)
    elif args.mode in ("linear", "mge"):
        run_linear(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
