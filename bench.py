#!/usr/bin/env python
"""bench.py -- samples*cycles/sec of the CHISAO oscillation cycle (BASELINE.json metric) on one node.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one full convergence / anti-convergence cycle (chisao_step: phases 1-6 of Algorithm 1,
PAPER.md:141-176) over the whole population of the workload (default: BASELINE.json configs[4] = C5, the
configuration the north_star targets are quoted on: d = 64, N = 65536, full-covariance mixture).
N > 1 GPUs run independent replicas (replicas only, no data-path collective).
`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
Prints ONE JSON line on rank 0.
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

METRIC, UNIT = "samples_cycles_per_sec", "samples*cycles/s"

WORKLOAD_TEXT = {
    1: "C1: d=2 N=256 iso-GMM K=4 (BASELINE.json configs[0])",
    2: "C2: d=8 N=4096 diag-GMM K=16 noisy (configs[1])",
    3: "C3: d=32 N=16384 random-Fourier K=256 (configs[2])",
    4: "C4: d=64 N=16384 ill-conditioned quadratic (configs[3])",
    5: "C5: d=64 N=65536 full-covariance GMM K=64 noisy, RM/GR reseeding (configs[4])",
}


def flop_per_eval(obj) -> float:
    """Plain-definition flop count of one objective evaluation."""
    d, K = obj.d, obj.K
    return {0: K * (3.0 * d + 4), 1: K * (4.0 * d + 4), 2: K * (2.0 * d * d + 3 * d + 4), 3: K * (2.0 * d + 8) + 2 * d,
            4: 2.0 * d * d + 3 * d}[obj.id]


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "50"], stdout=subprocess.PIPE, text=True)
            for line in self.proc.stdout:
                self.rows.append([s.strip() for s in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm, reasons, mx = [], set(), None
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                continue
        pw = []
        for r in self.rows:
            try:
                pw.append(float(r[2]))
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm), "sm_mhz_min": float(np.min(sm)) if sm else None,
                "power_w": float(np.median(pw)) if pw else None}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


def oracle_throughput(c: int, steps: int, warmup: int, threads: int = 0):
    """Time the oracle as it stands on a bounded sample of workload `c` (host cores of this box): `warmup` untimed
    cycles, then `steps` timed ones; OpenMP over the samples with `threads` threads (0 = every core of the box)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as O
    from paper_2606_26164_b200 import inputs
    cores = len(os.sched_getaffinity(0))
    threads = threads or cores
    full = inputs.config(c)
    # ~1.5 s of one core per sample-cycle at C5: 8 samples per thread keep one step in the 10-20 s range
    per_thread = {1: 256, 2: 256, 3: 24, 4: 32, 5: 8}[c]
    Ns = min(full.hp.N, max(8, per_thread * threads))
    wl = inputs.config(c, N=Ns, n_osc=max(full.hp.n_osc, 2 * steps + warmup + 1))
    o = O.Oracle(wl, threads=threads)
    for _ in range(warmup):
        o.step()
    # two timed passes of `steps` cycles, the faster one reported: the first seconds of a fresh process on an idle box run
    # at anything between 0.55 and 1.0 of the settled rate (measured on the GPU boxes: host clocks ramping up), which made
    # the two arms that time this same function disagree by up to 40 %
    best = None
    for _ in range(2):
        ev0 = sum(o.stats().evals)
        t0 = time.perf_counter()
        for _ in range(steps):
            o.step()
        dt = time.perf_counter() - t0
        ev = sum(o.stats().evals) - ev0
        if best is None or dt < best[0]:
            best = (dt, ev)
    dt, ev = best
    o.close()
    return {"value": Ns * steps / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{Ns} of {full.hp.N} samples x {steps} full cycle(s) (the faster of two passes) after {warmup} warm-up cycle(s), fp64, "
                      f"OpenMP over samples on {threads} of {cores} host cores; per-sample cost is N-independent except deduplication",
            "f_evals_per_sec": ev / dt, "seconds": dt}, wl


def run_reference(args, rank, world):
    if rank != 0:
        return
    # the oracle is slow by design: one warm-up cycle is enough to page everything in
    res, wl = oracle_throughput(args.config, max(3, args.steps), max(1, min(args.warmup, 1)))
    steps = max(3, args.steps)
    line = {"impl": "reference", "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * res["seconds"] / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_TEXT[args.config], "sampled": res["sample"]},
            "cpu_baseline": {k: res[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": res["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "f_evals_per_sec": res["f_evals_per_sec"], "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def measured_alu_peaks(dev):
    """FP32 FMA (TFLOP/s) and SFU (T op/s) rates of this GPU, measured now by the library's probe kernels
    (chisao_measure_peak: include/chisao.h); they are the denominators of the "alu" rooflines."""
    from paper_2606_26164_b200 import binding as B
    return {"fp32_fma_tflops": B.measure_peak(B.PEAK_FP32_FMA, dev), "sfu_tops": B.measure_peak(B.PEAK_SFU, dev),
            "source": "measured in this run: chisao_measure_peak (FFMA / MUFU.EX2 micro-benchmark kernels, best of 5)"}


def measure_config(c, K, W, rank, local_rank, world, dist, dev, N_override=0, detail=True, alu=None):
    """Device-resident and end-to-end timing of `K` full cycles of workload `c` after `W` warm-up cycles, plus the
    roofline of its dominant kernel.  Returns the fields of the JSON line that depend on the workload."""
    import torch
    from paper_2606_26164_b200 import binding as B, inputs, replicas
    full = inputs.config(c)
    N = N_override or full.hp.N
    n_osc = max(full.hp.n_osc, 2 * K + W + 1)               # timed cycles are all full cycles (phases 1-6)
    wl = replicas.replica_workload(c, rank, N=N, n_osc=n_osc)
    hp = wl.hp
    dd = dist if world > 1 else None

    # ---- device-resident timing: W warm-up cycles, then exactly K cycles between CUDA events.  No per-launch event
    # bracketing here: chisao_step submits every cycle as ONE CUDA graph launch (the product's default path)
    g = B.Chisao(wl, device=dev)
    for _ in range(W):
        g.step(stats=False)
    st0 = g.stats()
    l0, gl0 = g.launch_count(), g.graph_launches()
    sampler = ClockSampler(local_rank); sampler.start()
    time.sleep(0.25)
    ev_a, ev_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev_a.record()
    for _ in range(K):
        g.step(stats=False)
    ev_b.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = ev_a.elapsed_time(ev_b)
    clocks = sampler.stop()
    launches = g.launch_count() - l0
    graphs = g.graph_launches() - gl0
    st1 = g.stats()
    evals = np.array(st1.evals[:], np.int64) - np.array(st0.evals[:], np.int64)
    # ---- per-kernel-class times: K more cycles submitted directly, every launch bracketed with CUDA events on the
    # launching stream (the same kernels, the same state trajectory one cycle later; the brackets cost two event records
    # per launch, which is why they are not inside the timed region above)
    g.timing_enable(True); g.timing_reset()
    st2 = g.stats()
    for _ in range(K):
        g.step(stats=False)
    phase_all = g.timing()
    g.timing_enable(False)
    evals2 = np.array(g.stats().evals[:], np.int64) - np.array(st2.evals[:], np.int64)
    ms_max = replicas.max_over_ranks(ms, dd, dev)
    total_evals = replicas.sum_over_ranks(float(evals[[0, 1, 2, 5, 6]].sum()), dd, dev)

    # ---- end to end through the host-buffer C-ABI call (H2D + cycle + D2H inside the timed region) -------
    g2 = B.Chisao(wl, device=dev)
    x_host = torch.from_numpy(np.ascontiguousarray(wl.x0, np.float32)).pin_memory()
    x_out = torch.empty_like(x_host).pin_memory()
    f_out = torch.empty(hp.N, dtype=torch.float32).pin_memory()
    s_out = torch.empty(hp.N, dtype=torch.uint8).pin_memory()
    # (the population a step returns is the next step's input: the two pinned buffers swap roles, no host-side copy)
    for _ in range(W):
        g2.step_host(x_host, x_out, f_out, s_out)
        x_host, x_out = x_out, x_host
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(K):
        g2.step_host(x_host, x_out, f_out, s_out)           # H2D of x, one cycle, D2H of x, f, stuck; synchronises before returning
        x_host, x_out = x_out, x_host
    e2e_s = time.perf_counter() - t0
    e2e_s = replicas.max_over_ranks(e2e_s, dd, dev)
    g2.close()

    # ---- roofline of the dominant kernel (k_eval_fd: objective evaluation + FD stencil), from the bracketed pass ------
    peaks, peaks_src = measured_peaks()
    fpe = flop_per_eval(wl.obj)
    resident = g.lbfgs_resident()
    if resident:   # Phase 1 is one launch (k_lbfgs_resident, timed with the class of k_eval_fd): every evaluation but Hands Like Clouds
        fd_evals = float(evals2[0] + evals2[1] + evals2[2] + evals2[6])
    else:
        fd_evals = float(evals2[0] - K * hp.N + evals2[2] + evals2[6])  # counter 0 also holds the N centre values
    fd_ms, fd_n = phase_all["eval_fd"]
    step_ms2 = sum(v[0] for v in phase_all.values())               # sum of the bracketed kernel times of that pass
    alu_peak = alu["fp32_fma_tflops"] if alu else 148 * 128 * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
    alu_src = alu["source"] if alu else f"nominal: 148 SMs x 128 FP32 lanes x 2 x sm_max_mhz ({peaks_src} MEASURED_PEAKS.json clocks)"
    achieved = fd_evals * fpe / (fd_ms * 1e-3) / 1e12 if fd_ms > 0 else 0.0
    ev_mode = g.evaluator()
    traffic = TRAFFIC_BYTES_PER_LAUNCH.get(c)
    if ev_mode != 0:                                        # dense objectives at d > 32 and RFF at d <= 32 run on tcgen05 (chisao_tc.cuh)
        # kind::tf32 peak = measured bf16 cuBLAS throughput (sustained: the kernel is timed inside a long step) x the
        # guide's nominal tf32 : bf16 ratio 1.1 : 2.25.  The 3xTF32 split executes three tensor flops per
        # algorithmic flop of the contraction, so frac <= 1/3 by construction; executed_frac says how busy the pipe is.
        f16 = ev_mode in (3, 4, 5)                                # 3, 5: fp16 hi / lo operands; 4: random-Fourier phases, six products of 10-bit fp16 pieces
        peak = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]) * (1.0 if f16 else 1.1 / 2.25)
        pipe_rate = 8192 if f16 else 4096                      # flop / clk / SM: one 128x128x16 f16 (x8 tf32) MMA per 64 clocks
        contraction = wl.obj.K * 2.0 * hp.d * (1 if ev_mode == 4 else hp.d)
        nprod = 6.0 if ev_mode == 4 else 3.0                   # tensor flops executed per algorithmic flop of the contraction
        executed = nprod * fd_evals * contraction / (fd_ms * 1e-3) / 1e12 if fd_ms > 0 else 0.0
        roofline = {"bound": "tensor", "kernel": "k_eval_fd_tc", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                    "frac": achieved / peak, "traffic": traffic["bytes"] if traffic else None,
                    "traffic_source": traffic["source"] if traffic else None,
                    "evaluator": B.EVALUATOR_NAMES[ev_mode],
                    "peak_source": f"bf16_tflops_sustained ({peaks_src} MEASURED_PEAKS.json)" + ("" if f16 else " x 1.1/2.25 (tf32:bf16 nominal)")
                                   + f"; the operand split executes {nprod:.0f} tensor flops per algorithmic flop of the contraction",
                    "executed_tensor_tflops": executed, "executed_frac": executed / peak,
                    # the pipe's own rate: one 128x128x8 kind::tf32 (128x128x16 kind::f16) MMA per 64 clocks per SM
                    # = 4096 (8192) flop/clk/SM, at the SM clock sampled during the timed region --
                    # the kernel runs into the 1000 W power cap, so that clock is well below sm_max_mhz
                    "tensor_peak_at_sampled_clock": (pipe_rate * 148 * clocks["sm_mhz"] * 1e6 / 1e12) if clocks.get("sm_mhz") else None,
                    "executed_frac_at_sampled_clock": (executed / (pipe_rate * 148 * clocks["sm_mhz"] * 1e6 / 1e12)) if clocks.get("sm_mhz") else None,
                    "fp32_alu_peak_tflops": alu_peak, "alu_peak_source": alu_src, "vs_fp32_alu_peak": achieved / alu_peak}
    else:
        roofline = {"bound": "alu", "kernel": "k_lbfgs_resident (Phase 1 in one launch) + k_eval_fd" if resident else "k_eval_fd", "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s",
                    "frac": achieved / alu_peak, "traffic": traffic["bytes"] if traffic else None,
                    "traffic_source": traffic["source"] if traffic else None,
                    "peak_source": alu_src, "alu_peak_source": "measured" if alu else "nominal"}
    roofline.update({"launches": fd_n, "ms_per_launch": fd_ms / max(fd_n, 1), "flop_per_eval": fpe,
                     "share_of_step": fd_ms / step_ms2 if step_ms2 > 0 else None,
                     "timing": "per-launch CUDA events on the launching stream over K cycles submitted directly, right after the "
                               "timed region (which is one graph launch per cycle); share_of_step = this kernel's time / all bracketed kernel time"})
    out = {
        "value": world * hp.N * K / (ms_max * 1e-3), "ms_per_step": ms_max / K,
        "config": {"workload": WORKLOAD_TEXT[c], "N_per_gpu": hp.N, "d": hp.d, "n_conv": hp.n_conv, "lbfgs_m": hp.lbfgs_m,
                   "hlc_M": hp.hlc_M, "n_cloud": hp.n_cloud, "n_anti": hp.n_anti, "fd_h": hp.fd_h,
                   "parallelism": "replicas" if world > 1 else "single",
                   "submission": f"{graphs} of {K} timed cycles submitted as one CUDA graph launch each",
                   "phase1": "history-resident: one launch for release + f, g + n_conv L-BFGS iterations, (s, y) in registers" if resident
                             else "history spilled to HBM: direction(+update) / line search / FD launches per iteration",
                   "line_search": "inside the resident pass" if resident else ("tile-local rounds (one launch per iteration)" if g.ls_tile_local() else "one launch per trial on compacted worklists"),
                   "l2": f"state per cycle {g.workspace_bytes / 2**20:.0f} MiB vs 126 MB L2: "
                         + ("inputs larger than L2" if g.workspace_bytes > 126e6 else "fits L2 (latency-bound config)")},
        "f_evals_per_sec": total_evals / (ms_max * 1e-3),
        "evals_per_step": float(evals[[0, 1, 2, 5, 6]].sum()) / K,
        "clocks": clocks,
        "e2e": {"value": world * hp.N * K / e2e_s, "unit": UNIT, "h2d_bytes_per_step": hp.N * hp.d * 4,
                "d2h_bytes_per_step": hp.N * hp.d * 4 + hp.N * 4 + hp.N},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "phase_ms_per_step": {k: round(v[0] / K, 4) for k, v in phase_all.items()},
    }
    per_rank = None
    if world > 1:
        t = torch.zeros(world, dtype=torch.float64, device=dev); t[rank] = ms
        dist.all_reduce(t)
        per_rank = [float(v) / K for v in t.tolist()]
        out["per_rank_ms_per_step"] = per_rank
    if not detail:
        g.close()
        return out, wl, None

    # HBM-bound history kernel (two-loop recursion over the spilled (s, y) pairs; inside a cycle it also carries the
    # update of the previous iteration: k_lbfgs_step)
    dir_ms, dir_n = phase_all["lbfgs_direction"]
    hist_bytes = float(evals2[7])                           # counted on the device: rows actually read / written
    upd_ms = phase_all["lbfgs_update"][0]
    hbm = {"bound": "hbm", "kernel": "k_lbfgs_step + k_lbfgs_update (inside the cycle)",
           "achieved": hist_bytes / ((dir_ms + upd_ms) * 1e-3) / 1e9 if dir_ms > 0 else 0.0,
           "peak": peaks["hbm_gbs"], "unit": "GB/s", "bytes_per_launch": hist_bytes / max(dir_n, 1),
           "ms_per_launch": dir_ms / max(dir_n, 1)}
    hbm["frac"] = hbm["achieved"] / hbm["peak"]

    # the same kernel with every sample active and a full history of m pairs (the state the north_star's HBM target
    # is about): synthetic state written through chisao_set_state, 20 launches timed with CUDA events on the stream
    g3 = B.Chisao(wl, device=dev)
    rng = np.random.default_rng(5)
    g3.set(B.G, rng.standard_normal((hp.N, hp.d)).astype(np.float32) * 100.0)
    Sh = rng.standard_normal((hp.lbfgs_m, hp.N, hp.d)).astype(np.float32)
    g3.set(B.HIST_S, Sh); g3.set(B.HIST_Y, Sh * 2.0 + 0.1)
    del Sh
    g3.set(B.HIST_LEN, np.full(hp.N, hp.lbfgs_m, np.int32))
    for _ in range(3):
        g3.phase(B.PH_LBFGS_DIRECTION)
    # (a) per launch: every launch bracketed by its own pair of events (the library's class timers)
    g3.timing_enable(True); g3.timing_reset()
    for _ in range(20):
        g3.phase(B.PH_LBFGS_DIRECTION)
    br_ms, br_n = g3.timing()["lbfgs_direction"]
    g3.timing_enable(False)
    # (b) the figure reported: one pair of events on the launching stream around 20 launches back to back (launch gaps
    # included), i.e. the average launch duration over the timed region
    e0 = g3.stats().evals[7]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(g3.stream)
    for _ in range(20):
        g3.phase(B.PH_LBFGS_DIRECTION)
    ev1.record(g3.stream)
    ev1.synchronize()
    full_ms, full_n = float(ev0.elapsed_time(ev1)), 20
    full_bytes = float(g3.stats().evals[7] - e0)
    hbm_full = {"bound": "hbm", "kernel": "k_lbfgs_step_quad at 32 < d <= 64, else k_lbfgs_step (direction only; all samples active, len = m)", "achieved": full_bytes / (full_ms * 1e-3) / 1e9,
                "peak": peaks["hbm_gbs"], "unit": "GB/s", "bytes_per_launch": full_bytes / max(full_n, 1),
                "ms_per_launch": full_ms / max(full_n, 1), "ms_per_launch_bracketed_singly": br_ms / max(br_n, 1),
                "timing": "one CUDA-event pair on the launching stream around 20 launches back to back"}
    hbm_full["frac"] = hbm_full["achieved"] / hbm_full["peak"]
    g3.close()
    out["hbm_kernel"], out["hbm_kernel_full_history"] = hbm, hbm_full
    g.close()
    return out, wl, evals


def run_ours(args, rank, local_rank, world):
    import torch
    import torch.distributed as dist
    from paper_2606_26164_b200 import binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    K, W, c = args.steps, args.warmup, args.config
    alu = measured_alu_peaks(dev)
    res, wl, _ = measure_config(c, K, W, rank, local_rank, world, dist, dev, N_override=args.N, detail=True, alu=alu)
    hp = wl.hp

    # ---- the other four BASELINE.json configs, short (3 warm-up + 5 cycles each): north_star asks for all five ----------
    others = None
    if c == 5 and not args.N and not args.no_other_configs:
        others = {}
        for cc in (1, 2, 3, 4):
            r, _, _ = measure_config(cc, 5, 3, rank, local_rank, world, dist, dev, detail=False, alu=alu)
            others[f"C{cc}"] = {k: r[k] for k in ("value", "ms_per_step", "f_evals_per_sec", "gpu_launches", "clocks", "e2e",
                                                  "roofline", "phase_ms_per_step", "config")}
            others[f"C{cc}"]["steps"], others[f"C{cc}"]["warmup"], others[f"C{cc}"]["unit"] = 5, 3, UNIT

    # ---- NEXT-5, reported SEPARATELY (never mixed into `value`): the same cycles with the opt-in stencil-aware FD
    # evaluator of the dense objectives (chisao_set_option; not a black-box evaluation of f)
    stencil = None
    if wl.obj.id in (2, 4) and not args.no_stencil_pass:
        from paper_2606_26164_b200 import replicas
        g4 = B.Chisao(wl, device=dev)
        g4.set_option(B.OPT_STENCIL_AWARE, 1)
        for _ in range(W):
            g4.step(stats=False)
        e0 = g4.stats().total_evals()
        ev_c, ev_d = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        ev_c.record()
        for _ in range(K):
            g4.step(stats=False)
        ev_d.record()
        torch.cuda.synchronize()
        ms4 = replicas.max_over_ranks(ev_c.elapsed_time(ev_d), dist if world > 1 else None, dev)
        stencil = {"value": world * hp.N * K / (ms4 * 1e-3), "unit": UNIT, "ms_per_step": ms4 / K,
                   "f_evals_per_sec_by_definition": (g4.stats().total_evals() - e0) / (ms4 * 1e-3),
                   "note": "FD gradients by the stencil-aware evaluator (shares W(x-mu) between the 2d stencil points); "
                           "line search and HLC stay black-box; not comparable with `value`"}
        g4.close()

    if rank == 0:
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            # same policy as --impl reference: one warm-up cycle, three timed cycles; all cores, then one core
            cpu_all, _ = oracle_throughput(c, 3, 1)
            cpu_one, _ = oracle_throughput(c, 3, 1, threads=1)
            cpu = {k: cpu_all[k] for k in ("value", "unit", "cores", "kind", "sample", "f_evals_per_sec")}
            cpu["one_core"] = {k: cpu_one[k] for k in ("value", "unit", "cores", "sample", "f_evals_per_sec")}
        line = {"metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic"}
        for k in ("config", "f_evals_per_sec", "evals_per_step", "clocks", "e2e", "gpu_launches", "roofline", "hbm_kernel",
                  "hbm_kernel_full_history", "phase_ms_per_step", "per_rank_ms_per_step"):
            if k in res:
                line[k] = res[k]
        line["phase_ms_note"] = "K cycles submitted directly right after the timed region, every kernel class bracketed by events"
        line["alu_peaks"] = alu
        line["cpu_baseline"] = cpu
        line["stencil_aware_separately"] = stencil
        line["configs"] = others
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum per k_eval_fd launch, read off the committed `ncu --set full` capture named
# beside it (profiles/); not measured in this run -- a run under ncu is never a bench value
TRAFFIC_BYTES_PER_LAUNCH = {
    5: {"bytes": 1.86e7, "source": "profiles/r2_evalfd_c5.md (full-size launch: 18.5 MB read, 0.08 MB written)"},
    3: {"bytes": 4.38e6, "source": "profiles/r2_c2_c3_c4.md, r2_evalfd_c3.csv (4.38 MB read, 0 written: the gradient stays in L2)"},
    4: {"bytes": 4.36e6, "source": "profiles/r2_c2_c3_c4.md, r2_evalfd_c4.csv (4.36 MB read, 0 written)"}}


def self_launch(args):
    """`python bench.py --gpus N` without a launcher: start N ranks of this script with torch.distributed.run (one process
    per GPU, rendezvous on 127.0.0.1) and pass their output through; rank 0 prints the JSON line."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    env.setdefault("NCCL_DEBUG", "INFO"); env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")   # the communicator log names the rank count
    raise SystemExit(subprocess.call(cmd, env=env))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--N", type=int, default=0, help="override the population size (parity/debug runs only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-stencil-pass", action="store_true", help="skip the separately reported NEXT-5 pass")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short C1..C4 sub-records of the default run")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        self_launch(args)
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        if args.warmup < 3:
            args.warmup = 3
        run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
