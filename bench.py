#!/usr/bin/env python
"""bench.py -- throughput of the resampling F-statistic hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one pass of the whole hot path (sky-dependent kernels, fused FFT passes, 2F) over
one batch of synthetic input: `fstat_compute` on the full template bank of the workload
(default: BASELINE.json configs[1] -- 2 detectors, 10 d at 2 Hz, 30 % gaps, 1024 fdot templates,
FFT 2^21).  Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement".

Workloads: config1 | config2[:n_templates] | config3:<days>:<band> | config4:<target>[:n_fdot] |
config5[:n_sky] | sky100:<days>:<band> (the paper's timing protocol: 100 sky positions x one
spin-down template on a config-3 cell) | small.
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
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12      # plain fp32 FMA peak (SMs x lanes x 2 flop x max SM clock)
# config-3 cells of the bounded sweep carried by the default line: one per FFT length 2^15 .. 2^23
CONFIG3_SWEEP = [(1, 0.1), (2, 0.1), (1, 0.5), (1, 1.0), (1, 2.0), (2, 2.0), (5, 2.0), (10, 2.0), (20, 2.0)]


def make_workload(name: str, rank: int = 0):
    if name.startswith("config2"):            # config2[:n_templates]
        parts = name.split(":")
        p = synth.config2(n_templates=int(parts[1])) if len(parts) > 1 else synth.config2()
    elif name == "config1":
        p = synth.config1()
    elif name.startswith("config3"):          # config3:<days>:<band>
        _, d, b = name.split(":")
        p = synth.config3(float(d) if "." in d else int(d), float(b))
    elif name.startswith("sky100"):           # sky100:<days>:<band>[:n_sky]
        parts = name.split(":")
        d, b = parts[1], parts[2]
        p = synth.config3(float(d) if "." in d else int(d), float(b), n_templates=1)
        sky = synth.disc_sky_points(int(parts[3]) if len(parts) > 3 else 100, seed=77, radius=0.3)
        p.templates = np.array([(a, dl, p.f_min, -5e-10, 0.0) for (a, dl) in sky], dtype=np.float64)
        p.name = name
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
    pass 1 reads the detector-summed resampled series S (16 B x n_src; served by L2 after the first template of a
    sky position) and writes the four-step intermediate T (16 B x n_fft); pass 2 reads T back and writes 2F
    (4 B x n_bins).  Their sum is SURVEY.md 8(d)'s B_2pass."""
    n_src = p.n_samples + 2 * int(np.ceil(512.0 / p.dt))
    return {"S_read": 16 * n_src, "T_write": 16 * p.n_fft, "T_read": 16 * p.n_fft, "twoF_write": 4 * p.n_bins}


def ncu_traffic_table():
    """{(class, n_fft): dram bytes per template} from `paper_2201_00451_b200/traffic_table.csv` (ncu dram__bytes_read.sum +
    dram__bytes_write.sum per launch / templates per launch, written by `python -m paper_2201_00451_b200.capture_traffic`),
    and a description that names the commit the table was captured on."""
    path = os.path.join(ROOT, "paper_2201_00451_b200", "traffic_table.csv")
    tab, commits = {}, set()
    try:
        for line in open(path):
            f = [c.strip() for c in line.split(",")]
            if len(f) >= 5 and f[1].isdigit():
                tab[(f[0], int(f[1]))] = float(f[2]) + float(f[3])
                commits.add(f[4])
    except OSError:
        return {}, None
    return tab, f"paper_2201_00451_b200/traffic_table.csv, captured on commit {'/'.join(sorted(commits))}"


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
# CPU oracle legs (the only places bench.py touches oracle/).  ONE protocol for `cpu_baseline` and for
# `--impl reference`: the sky-dependent preparation once (one core; it is amortised over the bank exactly as the
# GPU path amortises it), then a bounded sample of templates spread over all host cores by a process pool.
# ------------------------------------------------------------------------------------------
_ORACLE_STATE = {}


def _oracle_worker(i):
    from oracle import fstat_oracle as O
    p, sky = _ORACLE_STATE["p"], _ORACLE_STATE["sky"]
    t = p.templates[i]
    if sky is None or (float(t[0]), float(t[1])) != _ORACLE_STATE["sky_key"]:
        return float(O.fstat_2F(p, t).max())           # sky-varying bank: the per-sky work belongs to the template
    return float(O.fstat_2F(p, t, sky).max())


class OraclePool:
    """Fork pool over the host cores; the problem and the per-sky cache are inherited copy-on-write.  Must be created
    before CUDA is initialised in this process (fork)."""

    def __init__(self, p):
        import multiprocessing as mp
        from oracle import fstat_oracle as O
        self.p = p
        self.cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
        groups = {(float(a), float(d)) for a, d in p.templates[:, :2]}
        self.n_groups = len(groups)
        self.sky_varying = self.n_groups > 1
        t0 = time.perf_counter()
        sky = O.per_sky(p, float(p.templates[0, 0]), float(p.templates[0, 1]))
        self.t_sky = time.perf_counter() - t0
        _ORACLE_STATE.update(p=p, sky=sky, sky_key=(float(p.templates[0, 0]), float(p.templates[0, 1])))
        self.pool = mp.get_context("fork").Pool(self.cores)
        self.pool.map(_oracle_worker, [0] * self.cores)             # start the workers (untimed)

    def step(self, idxs):
        """Wall seconds for the oracle to compute the 2F rows of templates idxs on all cores."""
        t0 = time.perf_counter()
        self.pool.map(_oracle_worker, list(idxs), chunksize=1)
        return time.perf_counter() - t0

    def sample_indices(self, per_core: int):
        n_t = len(self.p.templates)
        n = min(n_t, per_core * self.cores)
        return [int(i) for i in np.linspace(0, n_t - 1, n).astype(int)]

    def rate(self, idxs, t_pool: float):
        """2F-bins/s and templates/s of the whole bank extrapolated from the sample: per-template pool time x
        templates + one sky preparation per sky position (already inside the template cost for sky-varying banks)."""
        n_t = len(self.p.templates)
        full = n_t * t_pool / len(idxs) + (0.0 if self.sky_varying else self.n_groups * self.t_sky)
        return n_t * self.p.n_bins / full, n_t / full

    def describe(self, idxs, t_pool):
        return (f"numpy fp64 oracle on {self.cores} cores (process pool over templates): 1 sky preparation "
                f"({self.t_sky:.2f} s, one core) + {len(idxs)} of {len(self.p.templates)} templates in {t_pool:.2f} s wall, "
                f"extrapolated to the bank ({self.n_groups} sky position(s))")

    def close(self):
        self.pool.close()
        self.pool.join()


def cpu_baseline(p, per_core: int = 2):
    pool = OraclePool(p)
    try:
        idxs = pool.sample_indices(per_core)
        t_pool = pool.step(idxs)
        value, tps = pool.rate(idxs, t_pool)
        return {"value": value, "unit": UNIT, "cores": pool.cores, "kind": "oracle", "templates_per_s": tps,
                "sample": pool.describe(idxs, t_pool)}
    finally:
        pool.close()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    p = make_workload(args.workload)
    pool = OraclePool(p)
    try:
        idxs = pool.sample_indices(1)                   # one template per core and step
        times = []
        for s in range(args.warmup + args.steps):
            dt = pool.step(idxs)
            if s >= args.warmup:
                times.append(dt)
        t_pool = float(np.mean(times))
        value, tps = pool.rate(idxs, t_pool)
        sample = pool.describe(idxs, t_pool) + f"; mean of {args.steps} steps"
        line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": 1e3 * t_pool, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "templates_per_s": tps,
                "config": {"workload": args.workload, "n_det": p.n_det, "n_samples": p.n_samples, "dt": p.dt, "n_fft": p.n_fft,
                           "n_bins": p.n_bins, "n_templates": len(p.templates), "dterms": p.dterms,
                           "templates_per_step": len(idxs),
                           "note": "CPU oracle (numpy fp64) on a bounded sample per step; value = whole-bank rate extrapolated "
                                   "from it with the sky preparation amortised over the bank as the GPU path does"},
                "cpu_baseline": {"value": value, "unit": UNIT, "cores": pool.cores, "kind": "oracle", "sample": sample},
                "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
    finally:
        pool.close()


# ------------------------------------------------------------------------------------------
# Our arm
# ------------------------------------------------------------------------------------------
def time_bank(plan, p, steps, warmup, topk, k, flush, barrier=None, sampler=None):
    """W warm-up steps, then K timed steps of the whole bank (CUDA events on the plan's stream, L2 flushed between
    steps) with the library's per-class event recording OFF, then a separate repetition of the same K steps with it ON,
    from which only the split of the time over the kernel classes is taken (its event pairs per launch group would
    otherwise sit inside the steps whose launch overhead decides the small cells).
    Returns (per-step ms, class profile of the profiled repetition, its total ms, launches, clocks)."""
    import torch
    n_t, nb = len(p.templates), plan.n_bins
    if topk:
        out = (torch.empty((n_t, k), dtype=torch.float32, device="cuda"), torch.empty((n_t, k), dtype=torch.int32, device="cuda"))
    else:
        out = torch.empty((n_t, nb), dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        if topk:
            plan.compute_topk(p.templates, k, out=out)
        else:
            plan.compute(p.templates, out=out)

    def timed(n):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for s in range(n):
            flush.zero_()
            ev[s][0].record(stream)
            step()
            ev[s][1].record(stream)
        return ev

    for _ in range(warmup):
        step()
    plan.sync()
    plan.set_profile(False)
    l0 = plan.launch_count()
    if barrier:
        barrier()
    if sampler:
        sampler.start()
    t_wall0 = time.time()
    ev = timed(steps)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    launches = plan.launch_count() - l0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    # class split: the same steps again, profiled
    plan.set_profile(True)
    evp = timed(steps)
    torch.cuda.synchronize()
    prof = plan.get_profile()
    plan.set_profile(False)
    prof_ms = float(sum(a.elapsed_time(b) for a, b in evp))
    del out
    return step_ms, prof, prof_ms, launches, clocks


def roofline_report(p, prof, total_ms, steps, n_t, world, traffic_tab, traffic_src, peak, peak_src, prof_ms=None):
    """Roofline of the dominant FFT kernel and of the pair, on SURVEY.md 8(d)'s algorithmic bytes, plus the DRAM-only
    view: which of those bytes are served by HBM and which by L2 (the resampled series S is re-read by every template
    of a sky position out of L2), and the fraction of the measured HBM peak that the ncu-measured DRAM traffic makes."""
    ab = algorithmic_bytes(p)
    b1, b2 = ab["S_read"] + ab["T_write"], ab["T_read"] + ab["twoF_write"]
    kernels = {}
    single = prof["fft_single"][1] > 0
    fused = prof["fused_sky_pass1"][1] > 0
    classes = [("fft_single", b1 + b2 - ab["T_write"] - ab["T_read"])] if single else \
        [("fused_sky_pass1" if fused else "fft_pass1", b1), ("fft_pass2", b2)]
    for cls, bytes_per_t in classes:
        ms, n = prof[cls]
        kernels[cls] = {"ms_total": ms, "launches": n, "avg_launch_us": 1e3 * ms / max(n, 1),
                        "algorithmic_bytes_per_template": bytes_per_t,
                        "achieved_gbs": bytes_per_t * n_t * steps / (ms * 1e-3) / 1e9 if ms > 0 else None}
    for cls in ("sky", "topk"):
        kernels[cls] = {"ms_total": prof[cls][0], "launches": prof[cls][1]}
    fft_ms = sum(prof[c][0] for c, _ in classes)
    dom = max((c for c, _ in classes), key=lambda c: prof[c][0])
    ach = kernels[dom]["achieved_gbs"]
    # the pair always against B_2pass (SURVEY.md 8(d) convention), also when the intermediate never leaves the chip
    pair = (b1 + b2) * n_t * steps / (fft_ms * 1e-3) / 1e9
    flops = 2 * 5.0 * p.n_fft * float(np.log2(p.n_fft)) * n_t * steps
    per_launch = n_t * steps / max(kernels[dom]["launches"], 1)
    tr = traffic_tab.get((dom, p.n_fft))
    dram_pair = None
    if all((c, p.n_fft) in traffic_tab for c, _ in classes):
        dram_pair = sum(traffic_tab[(c, p.n_fft)] for c, _ in classes)
    n_groups = len({(float(a), float(d)) for a, d in p.templates[:, :2]})
    s_from_hbm = ab["S_read"] * n_groups / n_t            # S is read from HBM once per sky position, then from L2
    hbm_alg = s_from_hbm + (0 if single else ab["T_write"] + ab["T_read"]) + ab["twoF_write"]
    prof_ms = total_ms if prof_ms is None else prof_ms          # duration of the profiled repetition the class times come from
    return {"bound": "hbm", "kernel": dom + "_kernel", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
            "traffic": tr * per_launch if tr is not None else None,
            "traffic_source": ((traffic_src or "") + " (ncu dram__bytes_read.sum + dram__bytes_write.sum per template x templates per launch)") if tr is not None else None,
            "peak_source": peak_src,
            "conventions": "frac / fft_pair_frac: SURVEY 8(d) algorithmic bytes (B_2pass, INCLUDING the per-template re-read of the "
                           "resampled series that L2 serves) over FFT KERNEL time; hbm_algorithmic_frac: the HBM-only part of those bytes "
                           "over kernel time; dram_frac: ncu-measured DRAM bytes over kernel time; step_frac / hbm_algorithmic_step_frac / "
                           "dram_step_frac: the same three over the WHOLE timed step (SURVEY 8(d): t = the timed fstat_compute call, "
                           "class profiling off)",
            "fft_pair_achieved": pair, "fft_pair_frac": pair / peak,
            "step_frac": (b1 + b2) * n_t * steps / (total_ms * 1e-3) / 1e9 / peak,
            "hbm_algorithmic_step_frac": hbm_alg * n_t * steps / (total_ms * 1e-3) / 1e9 / peak,
            "dram_step_frac": dram_pair * n_t * steps / (total_ms * 1e-3) / 1e9 / peak if dram_pair is not None else None,
            # which of the algorithmic bytes are HBM traffic and which are L2 hits (per template)
            "algorithmic_bytes_per_template": {"total_B_2pass": b1 + b2, "hbm": hbm_alg, "l2_served_S_reread": ab["S_read"] - s_from_hbm,
                                               "on_chip_T": (ab["T_write"] + ab["T_read"]) if single else 0},
            "hbm_algorithmic_frac": hbm_alg * n_t * steps / (fft_ms * 1e-3) / 1e9 / peak,
            # measured: ncu DRAM bytes of the FFT kernels per template / their CUDA-event time / measured peak
            "dram_frac": dram_pair * n_t * steps / (fft_ms * 1e-3) / 1e9 / peak if dram_pair is not None else None,
            "dram_bytes_per_template": dram_pair,
            # SURVEY.md 8(d) R_min: compulsory traffic only (raw series in, 2F out) over the whole step
            "r_min_frac": (8 * p.n_samples * p.n_det + 4 * p.n_bins) * n_t * steps / (total_ms * 1e-3) / 1e9 / peak,
            "alu_tflops": flops / (fft_ms * 1e-3) / 1e12, "alu_peak_tflops": ALU_PEAK_TFLOPS,
            "alu_frac": flops / (fft_ms * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
            "share_of_step": prof[dom][0] / prof_ms if world == 1 else None}, kernels


def cufft_variant(plan, p, ours_us_per_template):
    """Comparison baseline only (north_star (3); "FFTs are computed using the cuFFT library"): the paper's
    structure on this GPU -- the same resampled series S from our sky kernel, then separate library kernels per step:
    spin-down phase factor, two cuFFT transforms (torch.fft.fft), the 2F map (torch expression).  Never on the product
    path.  Returns timing per template and the agreement with fstat_compute on the same templates."""
    import torch
    al, de = float(p.templates[0, 0]), float(p.templates[0, 1])
    S, abcd = plan.resample_sky(al, de)
    ya = torch.complex(S[:, 0], S[:, 1]).contiguous()
    yb = torch.complex(S[:, 2], S[:, 3]).contiguous()
    A, B, C, D = [float(v) for v in abcd]
    n_b = max(1, min(16, (1 << 26) // p.n_fft))
    same_sky = [i for i in range(len(p.templates)) if float(p.templates[i, 0]) == al and float(p.templates[i, 1]) == de][:n_b]
    tm = torch.tensor(p.templates[same_sky], dtype=torch.float64, device="cuda")
    km = int(np.ceil(512.0 / p.dt))
    tau = (torch.arange(p.n_fft, dtype=torch.float64, device="cuda") - km) * p.dt
    nb = plan.n_bins

    def path():
        cyc = 0.5 * tm[:, 3:4] * tau * tau + tm[:, 4:5] * tau * tau * tau / 6.0            # [n_b, n_fft] fp64 cycles
        ang = (-2.0 * np.pi) * (cyc - torch.floor(cyc)).to(torch.float32)
        rot = torch.complex(torch.cos(ang), torch.sin(ang))
        fa = torch.fft.fft(ya * rot)[:, :nb]
        fb = torch.fft.fft(yb * rot)[:, :nb]
        return (B * (fa.real ** 2 + fa.imag ** 2) + A * (fb.real ** 2 + fb.imag ** 2)
                - 2.0 * C * (fa.real * fb.real + fa.imag * fb.imag)) / D

    for _ in range(2):
        ref = path()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(5):
        ref = path()
    e1.record()
    torch.cuda.synchronize()
    us_path = 1e3 * e0.elapsed_time(e1) / 5 / len(same_sky)
    x = (ya * 1.0).unsqueeze(0).repeat(2 * len(same_sky), 1)
    for _ in range(2):
        torch.fft.fft(x)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(5):
        torch.fft.fft(x)
    e1.record()
    torch.cuda.synchronize()
    us_fft = 1e3 * e0.elapsed_time(e1) / 5 / len(same_sky)
    ours = plan.compute(p.templates[same_sky])
    plan.sync()
    dev = float(((ours - ref).abs() / torch.clamp(ref, min=4.0)).max().item())
    return {"us_per_template_cufft_path": us_path, "us_per_template_two_ffts_only": us_fft,
            "ours_us_per_template_fft_classes": ours_us_per_template,
            "speedup_vs_cufft_path": us_path / ours_us_per_template,
            "speedup_vs_two_ffts_only": us_fft / ours_us_per_template,
            "max_rel_dev_ours_vs_cufft_path": dev, "templates": len(same_sky),
            "note": "comparison baseline only, never on the product path: our resampled series S, then torch ops per step "
                    "(fp64 spin-down phase -> complex64 factor, two torch.fft.fft = cuFFT, 2F expression).  The torch path is "
                    "dominated by its unfused fp64 elementwise phase; the fairer floor for a cuFFT-based design is "
                    "us_per_template_two_ffts_only (two bare cuFFT transforms, no phase factor, no 2F map), which a fused "
                    "custom phase / 2F kernel pair could approach but not beat.  ours_us_per_template_fft_classes = our two FFT "
                    "kernel classes (spin-down prologue + FFT + 2F epilogue); the sky-dependent work is excluded on both sides"}


def bounded_cell(p, flush, traffic_tab, peak, warmup, topk=False, k=8, steps=3):
    """One bounded measurement of a workload for the blocks the default line carries besides its headline: W warm-up +
    3 timed steps (class profiling off) + 3 profiled steps for the class split, with every roofline convention."""
    from paper_2201_00451_b200.binding import FstatPlan
    with FstatPlan(p) as plan:
        step_ms, prof, prof_ms, launches, _ = time_bank(plan, p, steps, max(3, warmup), topk, k, flush)
        nb = plan.n_bins
    n_t = len(p.templates)
    total_ms = float(sum(step_ms))
    roof, _ = roofline_report(p, prof, total_ms, steps, n_t, 1, traffic_tab, None, peak, None, prof_ms)
    ms = total_ms / steps
    return {"log2_n_fft": int(np.log2(p.n_fft)), "n_det": p.n_det, "n_templates": n_t,
            "n_sky": len({(float(a), float(d)) for a, d in p.templates[:, :2]}), "dterms": p.dterms,
            "output": f"top-{k}" if topk else "full 2F",
            "ms_per_step": ms, "ms_per_step_profiled": prof_ms / steps,
            "bins_per_s": n_t * nb / (ms * 1e-3), "templates_per_s": n_t / (ms * 1e-3),
            "tau_eff_s_per_bin_per_detector": ms * 1e-3 / (n_t * nb * p.n_det),
            "pair_frac": roof["fft_pair_frac"], "step_frac": roof["step_frac"],
            "dom_kernel": roof["kernel"], "dom_frac": roof["frac"],
            "hbm_algorithmic_frac": roof["hbm_algorithmic_frac"], "hbm_algorithmic_step_frac": roof["hbm_algorithmic_step_frac"],
            "dram_frac": roof["dram_frac"], "dram_step_frac": roof["dram_step_frac"],
            "launches_per_step": launches // steps,
            "class_ms_per_step": {c: prof[c][0] / steps for c in prof if prof[c][1] > 0}}


def config3_block(args, flush, traffic_tab, peak):
    """Bounded config-3 sweep carried by the default line: one cell per FFT length 2^15 .. 2^23 (256 fdot templates)."""
    cells = []
    for days, band in CONFIG3_SWEEP:
        p = synth.config3(days, band)
        cell = {"days": days, "band_hz": band}
        cell.update(bounded_cell(p, flush, traffic_tab, peak, args.warmup))
        cells.append(cell)
        del p
    return {"cells": cells, "min_pair_frac": min(c["pair_frac"] for c in cells),
            "min_pair_cell": min(cells, key=lambda c: c["pair_frac"])["log2_n_fft"],
            "min_step_frac": min(c["step_frac"] for c in cells),
            "min_step_cell": min(cells, key=lambda c: c["step_frac"])["log2_n_fft"],
            "min_hbm_algorithmic_step_frac": min(c["hbm_algorithmic_step_frac"] for c in cells),
            "note": "config 3 (2 detectors, 50 % gaps, 256 fdot templates, full 2F output), one cell per FFT length; "
                    "pair_frac = B_2pass / (FFT kernel time) / measured HBM peak; step_frac = B_2pass / (time of the whole "
                    "fstat_compute step, class profiling off) / peak = SURVEY.md 8(d) R_hbm on its own t; the hbm_algorithmic_* "
                    "and dram_* figures leave out the re-reads of the resampled series that L2 serves"}


# the other BASELINE.json configs and the paper's own timing protocol, bounded (3 timed steps each)
EXTRA_BLOCKS = [("config1", False), ("config4:0:256", True), ("config5:512", False), ("sky100:10:1", False), ("sky100:1:0.5", False)]


def extra_blocks(args, flush, traffic_tab, peak):
    out = {}
    for name, topk in EXTRA_BLOCKS:
        p = make_workload(name)
        out[name] = bounded_cell(p, flush, traffic_tab, peak, args.warmup, topk=topk, k=8)
        del p
    out["note"] = ("config1: 16 templates, FFT 2^18; config4:0:256: 256 fdot x 4 fddot = 1024 of target 0's 16384 templates, FFT 2^22, top-8 "
                   "retention (the bank's time is 16 x this step); config5:512: 512 of the 4096 sky positions x 4 spin-downs, FFT 2^18, "
                   "Dterms 16 (one sky batch; the bank is 8 of these); sky100:<days>:<band>: the paper's timing protocol "
                   "(PAPER.md:188), 100 sky positions x 1 template on a config-3 cell")
    return out


def run_ours(args):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    p = make_workload(args.workload, rank)

    # the oracle leg forks a process pool: before CUDA is initialised in this process
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(p, args.cpu_templates_per_core)

    import torch
    import torch.distributed as dist
    from paper_2201_00451_b200.binding import FstatPlan
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    nccl = None
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")               # the communicator lines go to stderr, stdout stays one JSON line
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        nccl = {"backend": "nccl", "version": ".".join(str(v) for v in torch.cuda.nccl.version()),
                "collectives": "all_reduce(MAX) of the device time (1 per timed region); no data-path collective (replicas only)"}

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    plan = FstatPlan(p)
    if args.inflight:
        plan.set_inflight(args.inflight)
    if args.paths:
        plan.debug_set_paths(*[int(v) for v in args.paths.split(",")])
    if args.geometry:
        plan.debug_set_geometry(*[int(v) for v in args.geometry.split(",")])
    if args.sky_slots:
        plan.debug_set_max_sky_slots(args.sky_slots)
    n_t, nb = len(p.templates), plan.n_bins
    topk = args.mode == "topk"
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    step_ms, prof, prof_ms, launches, clocks = time_bank(plan, p, args.steps, args.warmup, topk, args.k, flush, barrier, ClockSampler(local))
    total_ms = float(sum(step_ms))
    value, ms_per_step = aggregate_ranks(total_ms, n_t * nb, args.steps, dist if world > 1 else None, "cuda")
    total_ms = ms_per_step * args.steps

    peak, peak_src = measured_peaks()
    traffic_tab, traffic_src = ncu_traffic_table()
    roofline, kernels = roofline_report(p, prof, total_ms, args.steps, n_t, world, traffic_tab, traffic_src or "", peak, peak_src, prof_ms)

    # ---- end to end through the host-buffer entry point (pinned host 2F, D2H inside the timed region)
    e2e = e2e_topk = None
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
        if not topk:
            del host_out
            # the same bank through fstat_compute_topk_host: only the k loudest bins per template cross PCIe
            # (retain candidates on the GPU instead of copying every 2F value back)
            plan.compute_topk_host(p.templates, args.k)
            barrier()
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                plan.compute_topk_host(p.templates, args.k)
            torch.cuda.synchronize()
            k_ms = 1e3 * (time.perf_counter() - t0) / n_e2e
            if world > 1:
                t = torch.tensor([k_ms], device="cuda", dtype=torch.float64)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                k_ms = float(t.item())
            e2e_topk = {"value": world * n_t * nb / (k_ms * 1e-3), "unit": UNIT, "ms_per_step": k_ms, "steps": n_e2e,
                        "h2d_bytes_per_step": int(p.templates.nbytes), "d2h_bytes_per_step": int(n_t * args.k * 8),
                        "api": f"fstat_compute_topk_host (host templates in, host top-{args.k} values + bins out): every bin is "
                               "searched, only the candidates leave the GPU"}

    cufft = None
    if not args.no_cufft_compare and rank == 0:
        fft_ms = sum(prof[c][0] for c in ("fft_pass1", "fft_pass2", "fused_sky_pass1", "fft_single"))
        cufft = cufft_variant(plan, p, 1e3 * fft_ms / args.steps / n_t)
    plan.close()

    c3 = None
    if rank == 0 and world == 1 and not args.no_config3 and args.workload == "config2":
        del p.series
        torch.cuda.empty_cache()
        c3 = config3_block(args, flush, traffic_tab, peak)
    extra = None
    if rank == 0 and world == 1 and not args.no_extra and args.workload == "config2":
        if hasattr(p, "series"):
            del p.series
        torch.cuda.empty_cache()
        extra = extra_blocks(args, flush, traffic_tab, peak)

    if rank == 0:
        from paper_2201_00451_b200 import build as _b
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
                "clocks": clocks, "gpu_launches": launches, "e2e": e2e, "e2e_topk": e2e_topk, "roofline": roofline, "kernels": kernels,
                "config3": c3, "other_workloads": extra, "cpu_baseline": cpu, "cufft_compare": cufft, "nccl": nccl,
                "library": {"path": os.path.relpath(_b.LIB_PATH, ROOT), "mtime": int(os.path.getmtime(_b.LIB_PATH))}}
        print(json.dumps(line))
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
    ap.add_argument("--paths", default="", help="fused_sky,single overrides for fstat_debug_set_paths (-1 auto, 0 off, 1 on)")
    ap.add_argument("--geometry", default="", help="log_n2,log_tile1,log_tile2,p2_elems overrides for fstat_debug_set_geometry (-1 = default)")
    ap.add_argument("--sky-slots", type=int, default=0, help="fstat_debug_set_max_sky_slots: sky positions resampled per batch (0 = default)")
    ap.add_argument("--mode", default="full", choices=["full", "topk"])
    ap.add_argument("--k", type=int, default=8)
    ap.add_argument("--cpu-templates-per-core", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft-compare", action="store_true")
    ap.add_argument("--no-config3", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the bounded config1 / config4 / config5 / sky100 blocks")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started without torchrun: start the N ranks ourselves (one process per GPU, NCCL over NVLink for the one all_reduce)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--standalone", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--local-addr", "127.0.0.1", os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
