#!/usr/bin/env python
"""bench.py -- throughput of the resampling F-statistic hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one pass of the whole hot path (sky-dependent kernels, fused FFT passes, 2F) over
one batch of synthetic input: `fstat_compute` on the full template bank of the workload
(default: BASELINE.json configs[1] -- 2 detectors, 10 d at 2 Hz, 30 % gaps, 1024 fdot templates,
FFT 2^21).  Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement".
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

from paper_2201_00451_b200 import synth  # noqa: E402

METRIC = "2F_bins_per_s"
UNIT = "2F-bins/s"


def make_workload(name: str, rank: int = 0):
    if name.startswith("config2"):            # config2[:n_templates]
        parts = name.split(":")
        p = synth.config2(n_templates=int(parts[1])) if len(parts) > 1 else synth.config2()
    elif name == "config1":
        p = synth.config1()
    elif name.startswith("config3"):          # config3:<days>:<band>
        _, d, b = name.split(":")
        p = synth.config3(float(d) if "." in d else int(d), float(b))
    elif name.startswith("config4"):          # config4:<target>[:n_fdot]
        parts = name.split(":")
        p = synth.config4(int(parts[1]), n_fdot=int(parts[2]) if len(parts) > 2 else 256)
    elif name.startswith("config5"):          # config5[:n_sky]
        parts = name.split(":")
        p = synth.config5(n_sky=int(parts[1]) if len(parts) > 1 else 512)
    elif name == "small":
        p = synth.small_problem(n_samples=20000, n_fft=1 << 15, n_templates=64)
    else:
        raise SystemExit(f"unknown workload {name}")
    p.templates = replica_templates(p.templates, rank)
    return p


def replica_templates(templates, rank: int):
    """Multi-GPU = independent replicas: rank r searches the fdot sub-bank shifted by r spans,
    so the ranks' banks tile the fdot axis without overlap; no data-path collective."""
    t = np.array(templates, dtype=np.float64, copy=True)
    if rank > 0:
        span = float(np.ptp(t[:, 3])) or 1e-9
        step = span / max(len(np.unique(t[:, 3])) - 1, 1)
        t[:, 3] -= rank * (span + step)
    return t


def aggregate_ranks(total_ms: float, units: int, steps: int, dist=None, device=None):
    """Whole-job value: units all ranks processed / the slowest rank's device time (max over ranks)."""
    world = 1
    if dist is not None and dist.is_initialized():
        import torch
        world = dist.get_world_size()
        t = torch.tensor([total_ms], dtype=torch.float64, device=device or "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / steps
    return world * units / (ms_per_step * 1e-3), ms_per_step


def algorithmic_bytes(p):
    """Per-template algorithmic bytes of the two FFT passes:
    pass 1 reads the detector-summed resampled series (16 B x n_src) and writes the four-step
    intermediate (16 B x n_fft); pass 2 reads it back and writes 2F (4 B x n_bins).  Their sum is
    SURVEY.md 8(d)'s B_2pass."""
    n_src = p.n_samples + 2 * int(np.ceil(512.0 / p.dt))
    b1 = 16 * n_src + 16 * p.n_fft
    b2 = 16 * p.n_fft + 4 * p.n_bins
    return b1, b2


def ncu_traffic(cls: str, n_fft: int, launches: int, templates: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of this kernel class from the committed
    `ncu --set full` capture (profiles/r01_traffic.csv holds bytes per template; a launch of the timed run
    processes templates/launches of them).  None when no capture exists for this FFT length."""
    path = os.path.join(ROOT, "profiles", "r01_traffic.csv")
    try:
        for line in open(path):
            f = [c.strip() for c in line.split(",")]
            if len(f) >= 4 and f[0] == cls and f[1].isdigit() and int(f[1]) == n_fft:
                per_t = float(f[2]) + float(f[3])
                return per_t * templates / max(launches, 1), "profiles/r01_traffic.csv (ncu --set full, per template x templates per launch)"
    except OSError:
        pass
    return None, None


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15 and len(r) >= 7] or [r for (_, r) in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "power_w_max": max(float(r[2]) for r in rows),
                "samples": len(rows), "reasons": reasons}


# ------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py touches oracle/)
# ------------------------------------------------------------------------------------------
def oracle_step(p, n_templates: int):
    """One bounded oracle sample: the sky-dependent work once, then n_templates templates."""
    from oracle import fstat_oracle as O
    t0 = time.perf_counter()
    sky = O.per_sky(p, float(p.templates[0, 0]), float(p.templates[0, 1]))
    t1 = time.perf_counter()
    for i in range(n_templates):
        O.fstat_2F(p, p.templates[i], sky)
    t2 = time.perf_counter()
    return t1 - t0, (t2 - t1) / n_templates


def cpu_baseline(p, n_templates: int = 8):
    t_sky, t_tmpl = oracle_step(p, n_templates)
    n_groups = len({(float(a), float(d)) for a, d in p.templates[:, :2]})
    n_t = len(p.templates)
    full = n_groups * t_sky + n_t * t_tmpl             # extrapolated to the whole bank
    return {"value": n_t * p.n_bins / full, "unit": UNIT, "cores": 1, "kind": "oracle",
            "templates_per_s": n_t / full,
            "sample": f"numpy fp64 oracle, 1 sky preparation ({t_sky:.2f} s) + {n_templates} of {n_t} templates "
                      f"({t_tmpl:.3f} s each), extrapolated to the bank ({n_groups} sky position(s))"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    p = make_workload(args.workload)
    n_per_step = 2
    times = []
    for s in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle_step(p, n_per_step)
        dt = time.perf_counter() - t0
        if s >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = n_per_step * p.n_bins / (ms * 1e-3)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "n_det": p.n_det, "n_samples": p.n_samples, "n_fft": p.n_fft,
                       "n_bins": p.n_bins, "templates_per_step": n_per_step,
                       "note": "CPU oracle (numpy fp64) on a bounded sample: one sky preparation + 2 templates per step"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "sample": f"{n_per_step} templates + 1 sky preparation per step"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------
# Our arm
# ------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2201_00451_b200.binding import FstatPlan

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    p = make_workload(args.workload, rank)
    plan = FstatPlan(p)
    if args.inflight:
        plan.set_inflight(args.inflight)
    n_t, nb = len(p.templates), plan.n_bins
    topk = args.mode == "topk"
    if topk:                      # config-4 style: only the k loudest bins of every template leave the GPU
        out = (torch.empty((n_t, args.k), dtype=torch.float32, device="cuda"),
               torch.empty((n_t, args.k), dtype=torch.int32, device="cuda"))
    else:
        out = torch.empty((n_t, nb), dtype=torch.float32, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step():
        if topk:
            plan.compute_topk(p.templates, args.k, out=out)
        else:
            plan.compute(p.templates, out=out)

    for _ in range(args.warmup):
        step()
    plan.sync()
    # ---- timed region: K steps, per-step CUDA events on the plan's stream, L2 flushed between steps
    plan.set_profile(not args.no_kernel_events)
    l0 = plan.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    t_wall0 = time.time()
    for s in range(args.steps):
        flush.zero_()
        ev[s][0].record(stream)
        step()
        ev[s][1].record(stream)
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1)
    prof = plan.get_profile() if not args.no_kernel_events else None
    plan.set_profile(False)
    launches = plan.launch_count() - l0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    value, ms_per_step = aggregate_ranks(total_ms, n_t * nb, args.steps, dist if world > 1 else None, "cuda")
    total_ms = ms_per_step * args.steps

    # ---- roofline of the dominant kernel class (CUDA events inside the library, same timed steps)
    roofline = None
    kernels = None
    if prof is not None:
        b1, b2 = algorithmic_bytes(p)
        peak, peak_src = measured_peaks()
        per_launch_t = plan_inflight = None
        kernels = {}
        for cls, bytes_per_t in (("fft_pass1", b1), ("fft_pass2", b2)):
            ms, n = prof[cls]
            tot_bytes = bytes_per_t * n_t * args.steps
            kernels[cls] = {"ms_total": ms, "launches": n, "avg_launch_us": 1e3 * ms / max(n, 1),
                            "algorithmic_bytes_per_template": bytes_per_t,
                            "achieved_gbs": tot_bytes / (ms * 1e-3) / 1e9 if ms > 0 else None}
        kernels["sky"] = {"ms_total": prof["sky"][0], "launches": prof["sky"][1]}
        kernels["topk"] = {"ms_total": prof["topk"][0], "launches": prof["topk"][1]}
        dom = max(("fft_pass1", "fft_pass2"), key=lambda c: prof[c][0])
        ach = kernels[dom]["achieved_gbs"]
        both = (b1 + b2) * n_t * args.steps / ((prof["fft_pass1"][0] + prof["fft_pass2"][0]) * 1e-3) / 1e9
        # fp32 work of the two FFTs of a template (2 x 5 N log2 N flop) against the plain-FMA peak
        fft_ms = prof["fft_pass1"][0] + prof["fft_pass2"][0]
        flops = 2 * 5.0 * p.n_fft * float(np.log2(p.n_fft)) * n_t * args.steps
        alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12
        traffic, traffic_src = ncu_traffic(dom, p.n_fft, kernels[dom]["launches"], n_t * args.steps)
        roofline = {"bound": "hbm", "kernel": dom + "_kernel", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                    "fft_pair_achieved": both, "fft_pair_frac": both / peak,
                    # SURVEY.md 8(d) R_min: compulsory traffic only (raw series in, 2F out) over the whole step
                    "r_min_frac": (8 * p.n_samples * p.n_det + 4 * nb) * n_t * args.steps / (total_ms * 1e-3) / 1e9 / peak,
                    "alu_tflops": flops / (fft_ms * 1e-3) / 1e12, "alu_peak_tflops": alu_peak,
                    "alu_frac": flops / (fft_ms * 1e-3) / 1e12 / alu_peak,
                    "share_of_step": prof[dom][0] / total_ms if world == 1 else None}

    # ---- end to end through the host-buffer entry point (pinned host 2F, D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        if topk:
            def e2e_step():
                return plan.compute_topk_host(p.templates, args.k)    # blocks until (val, bin) are in host memory
            d2h = n_t * args.k * 8
            api = "fstat_compute_topk_host (host templates in, host top-k values + bins out)"
        else:
            host_out = torch.empty((n_t, nb), dtype=torch.float32, pin_memory=True)

            def e2e_step():
                return plan.compute_host(p.templates, out=host_out)   # blocks until the rows have landed
            d2h = n_t * nb * 4
            api = "fstat_compute_host (host templates in, pinned host 2F[n_tmpl][n_bins] out)"
        e2e_step()                                                    # warm-up (allocates the device ring)
        n_e2e = max(1, min(args.steps, 3))
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        torch.cuda.synchronize()
        e_ms = 1e3 * (time.perf_counter() - t0) / n_e2e
        if world > 1:
            t = torch.tensor([e_ms], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e_ms = float(t.item())
        e2e = {"value": world * n_t * nb / (e_ms * 1e-3), "unit": UNIT, "ms_per_step": e_ms, "steps": n_e2e,
               "h2d_bytes_per_step": int(p.templates.nbytes), "d2h_bytes_per_step": int(d2h),
               "api": api + "; the series is uploaded once by fstat_setup (PAPER.md:93) and is not part of a step"}

    # ---- context only: the library FFT alone (cuFFT through torch.fft) on the same shape: two batched complex64
    # transforms of n_fft points per template, nothing else of the path (no resampling, phases or 2F)
    cufft = None
    if args.cufft_compare and rank == 0:
        nb_t = max(1, min(32, (1 << 28) // p.n_fft))
        x = torch.randn((2 * nb_t, p.n_fft), dtype=torch.complex64, device="cuda")
        for _ in range(3):
            y = torch.fft.fft(x)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(10):
            y = torch.fft.fft(x)
        e1.record()
        torch.cuda.synchronize()
        us = 1e3 * e0.elapsed_time(e1) / 10 / nb_t
        cufft = {"us_per_template_two_ffts": us, "ours_us_per_template_whole_path": 1e3 * ms_per_step / n_t,
                 "note": "torch.fft.fft (cuFFT) on [2 x %d, %d] complex64, out of place; comparison baseline only, "
                         "not on the product path" % (nb_t, p.n_fft)}
        del x, y

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(p, args.cpu_templates)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "templates_per_s": world * n_t / (ms_per_step * 1e-3),
                "tau_eff_s_per_bin_per_detector": ms_per_step * 1e-3 / (n_t * nb * p.n_det),
                "config": {"workload": args.workload, "n_det": p.n_det, "n_samples": p.n_samples, "dt": p.dt, "n_fft": p.n_fft,
                           "n_bins": nb, "n_templates": n_t, "dterms": p.dterms,
                           "output": f"top-{args.k} per template" if topk else "full 2F[n_templates][n_bins]", "multi_gpu": "independent replicas, no collective",
                           "l2": "256 MiB flush buffer written between timed steps; each step also writes "
                                 f"{n_t * nb * 4 / 1e9:.2f} GB of 2F (> L2)"},
                "clocks": clocks, "gpu_launches": launches, "e2e": e2e, "roofline": roofline, "kernels": kernels,
                "cpu_baseline": cpu, "cufft_compare": cufft}
        print(json.dumps(line))
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2")
    ap.add_argument("--inflight", type=int, default=0)
    ap.add_argument("--mode", default="full", choices=["full", "topk"])
    ap.add_argument("--k", type=int, default=8)
    ap.add_argument("--cpu-templates", type=int, default=32)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-kernel-events", action="store_true")
    ap.add_argument("--cufft-compare", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
