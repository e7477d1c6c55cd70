"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default
templates per launch), on sampled templates the oracle can compute one by one -- plus the
properties that hold at any size (chi^2_4 noise statistics of the full bank, top-k == selection
over the full rows, loudest template)."""
import os
import subprocess
import sys

import numpy as np
import pytest

from oracle import fstat_oracle as O
from paper_2201_00451_b200 import synth

from _parity_util import TOL, compare_rows

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))


def _start_oracle_bank(config, out, rows=()):
    """The oracle over the whole bank of `synth.<config>()` in a process of its own (tests/oracle_bank_maxima.py: a fork
    pool over the host cores), started before the GPU work of the test so that the two overlap."""
    cmd = [sys.executable, os.path.join(HERE, "oracle_bank_maxima.py"), config, str(out), "--rows", ",".join(str(int(r)) for r in rows)]
    return subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)


def _finish_oracle_bank(proc, out, timeout=1000):
    text, _ = proc.communicate(timeout=timeout)
    assert proc.returncode == 0, text
    print("[oracle]", text.strip().splitlines()[-1])
    return np.load(str(out))


def _check_bank_maxima(val, idx, ora, label):
    """GPU top-1 (val[n_t], idx[n_t]) of every template against the oracle's three loudest bins of the same row:
    the GPU's bin is one of them, its value agrees within TOL, and where it is not the oracle's loudest bin the two are a
    tie within the tolerance (S15: what is compared is unique only up to the tolerance); the loudest template
    of the whole bank is identical (same rule)."""
    ov, ob = ora["val"], ora["bin"]
    n_t = len(val)
    assert ov.shape[0] == n_t
    hit = ob == idx[:, None].astype(np.int64)
    assert hit.any(axis=1).all(), np.nonzero(~hit.any(axis=1))[0][:10]
    pos = hit.argmax(axis=1)
    o_at = ov[np.arange(n_t), pos]
    err = np.abs(val.astype(np.float64) - o_at) / np.maximum(o_at, 4.0)
    assert err.max() <= TOL, err.max()
    gap = (ov[:, 0] - o_at) / np.maximum(ov[:, 0], 4.0)
    assert gap.max() <= 2 * TOL, gap.max()
    tg, to = int(np.argmax(val)), int(np.argmax(ov[:, 0]))
    assert tg == to or (ov[to, 0] - ov[tg, 0]) <= 2 * TOL * max(ov[to, 0], 4.0), (tg, to)
    print(f"[parity] {label}: loudest bin of all {n_t} templates: max |d2F|/max(2F,4) = {err.max():.2e}, "
          f"{int((pos != 0).sum())} rows where the GPU's loudest bin is the oracle's second or third (ties within {2 * TOL:g}), "
          f"loudest template {tg} (oracle {to}), 2F = {val[tg]:.3f} (oracle {ov[to, 0]:.3f})")
    return tg


def _plan(prob):
    from paper_2201_00451_b200.binding import FstatPlan
    return FstatPlan(prob)


def _rel_err(gpu, cpu):
    return np.abs(gpu.astype(np.float64) - cpu) / np.maximum(cpu, 4.0)


def test_config1_full_bank_every_bin():
    p = synth.config1()
    cpu = O.fstat_2F_bank(p)
    with _plan(p) as plan:
        gpu = plan.compute(p.templates)
        val, idx = plan.compute_topk(p.templates, 4)
        plan.sync()
        gpu, val, idx = gpu.cpu().numpy(), val.cpu().numpy(), idx.cpu().numpy()
    assert _rel_err(gpu, cpu).max() <= TOL
    assert int(np.argmax(gpu.max(axis=1))) == int(np.argmax(cpu.max(axis=1)))      # loudest template identical
    np.testing.assert_array_equal(idx[:, 0], cpu.argmax(axis=1))
    # config 1 injects rho = 20 at 100.2 Hz: the loudest bin of the loudest template is that frequency
    t = int(np.argmax(cpu.max(axis=1)))
    f_peak = p.f_min + idx[t, 0] * p.df
    assert abs(f_peak - 100.2) < 2 * p.df


def test_config2_full_size_sampled_templates_and_loudest(tmp_path):
    p = synth.config2()                                  # 1024 templates, FFT 2^21, 30 % gaps, weights
    proc = _start_oracle_bank("config2", tmp_path / "config2.npz")      # the oracle runs ALL templates
    sample = sorted({0, 1, p.injection_template - 1, p.injection_template, p.injection_template + 1, 517, 1023})
    cpu = O.fstat_2F_bank(p, sample)
    with _plan(p) as plan:
        val, idx = plan.compute_topk(p.templates, 2)     # whole bank, as bench.py launches it
        rows = plan.compute(p.templates[sample])
        plan.sync()
        val, idx, rows = val.cpu().numpy(), idx.cpu().numpy(), rows.cpu().numpy()
    assert _rel_err(rows, cpu).max() <= TOL
    # the rows of the sampled templates agree with the whole-bank run (same values whatever the batch)
    for r, t in enumerate(sample):
        assert val[t, 0] == rows[r].max() and idx[t, 0] == rows[r].argmax()
    # loudest template of the whole bank = the injected one, which the oracle confirms within the sample
    assert int(np.argmax(val[:, 0])) == p.injection_template
    assert sample[int(np.argmax(cpu.max(axis=1)))] == p.injection_template
    # every one of the 1024 templates: loudest bin and its value against the oracle's row, loudest template of the bank
    ora = _finish_oracle_bank(proc, tmp_path / "config2.npz")
    assert _check_bank_maxima(val[:, 0], idx[:, 0], ora, "config2 full bank") == p.injection_template


CELLS = [(d, b) for d in synth.CONFIG3_DAYS for b in synth.CONFIG3_BANDS]


@pytest.mark.parametrize("days,band", CELLS)
def test_config3_every_cell_noise_statistics_and_sampled_parity(days, band):
    # all 20 cells of the timing sweep (PAPER.md:188-206 shape): 50 % gaps, pure noise.  The bank is cut to what
    # gives >= 1e5 central bins where the cell is small and to 2-8 templates where one row is 2^21-2^22 bins.
    p = synth.config3(days, band, n_templates=256)
    n_t = int(min(256, max(2, (1 << 22) // p.n_bins)))
    p.templates = p.templates[np.linspace(0, 255, n_t).astype(int)]
    with _plan(p) as plan:
        gpu = plan.compute(p.templates)
        plan.sync()
        gpu = gpu.cpu().numpy()
    # pure noise: 2F ~ chi^2 with 4 dof over the central half of the band (pin P1 at full size)
    nb = gpu.shape[1]
    central = gpu[:, nb // 4: 3 * nb // 4].astype(np.float64)
    n_eff = central.size / 4.0          # zero padding correlates neighbouring bins
    assert abs(central.mean() - 4.0) < max(0.1, 6.0 * np.sqrt(8.0 / n_eff)), central.mean()
    assert abs(central.var() - 8.0) < max(0.8, 6.0 * 8.0 * np.sqrt(8.0 / n_eff)), central.var()
    sample = [0, n_t - 1]
    res = compare_rows(p, sample, gpu[sample], label=f"config3 T={days}d B={band}Hz n_fft=2^{int(np.log2(p.n_fft))}")
    assert all(o["finite"] for o in res)
    assert max(o["err"] for o in res) <= TOL
    assert max(o["r2"] for o in res) <= 1e-4 and max(o["theta"] for o in res) <= 1e-3   # paper's own GPU-vs-CPU level: ~1e-5


@pytest.mark.parametrize("target", [0, 1, 2, 3])
def test_config4_full_bank_all_targets_subset_rule(target):
    # config 4 at full geometry (10 d, 2 Hz band = sample rate, FFT 2^22, 4096 fdot x 4 fddot = 16384 templates) for
    # all four targets 320 / 480 / 550 / 680 Hz: whole bank through fstat_compute_topk, then SURVEY.md 8(d)'s subset --
    # every injection template, the GPU's 64 loudest, 16 seeded random ones -- as full rows against the oracle, bin by
    # bin; "loudest template identical" = oracle argmax over the subset equals GPU argmax over the whole bank.
    p = synth.config4(target)
    k = 8
    n_t = len(p.templates)
    assert n_t == 16384 and p.n_fft == 1 << 22 and p.n_bins == 1 << 22
    with _plan(p) as plan:
        val, idx = plan.compute_topk(p.templates, k)
        plan.sync()
        val, idx = val.cpu().numpy(), idx.cpu().numpy()
        loud = np.lexsort((np.arange(n_t), -val[:, 0]))          # descending 2F, ties -> lower template index (S15)
        gpu_best = int(loud[0])
        rng = np.random.default_rng(4000 + target)
        subset = list(loud[:64])
        if p.injection_template is not None:
            subset.append(p.injection_template)
        subset += [int(t) for t in rng.choice(n_t, 16, replace=False)]
        subset = sorted(set(int(t) for t in subset))
        res, rows_top = [], {}
        sky = O.per_sky(p, float(p.templates[0, 0]), float(p.templates[0, 1]))
        for c0 in range(0, len(subset), 16):                     # 16 rows of 2^22 floats at a time
            chunk = subset[c0:c0 + 16]
            rows = plan.compute(p.templates[chunk])
            plan.sync()
            rows = rows.cpu().numpy()
            for r, t in enumerate(chunk):                        # full rows agree with the whole-bank top-k run
                ev, ei = O.topk(rows[r], k)
                np.testing.assert_array_equal(idx[t], ei)
                np.testing.assert_array_equal(val[t], ev)
            res += compare_rows(p, chunk, rows, sky=sky, label=f"config4 target {target} ({synth.CONFIG4_TARGETS[target]:.0f} Hz) rows {c0}-{c0 + len(chunk) - 1}")
    assert all(o["finite"] for o in res)
    worst = max(o["err"] for o in res)
    print(f"[parity] config4 target {target}: {len(subset)} full rows, worst {worst:.2e}")
    assert worst <= TOL
    # loudest template: oracle argmax over the subset == GPU argmax over all 16384
    cpu_max = np.array([o["cpu_max"] for o in res])
    order = np.lexsort((np.array(subset), -cpu_max))
    cpu_best = subset[int(order[0])]
    if cpu_best != gpu_best:        # S15: the oracle's two loudest may differ by less than twice the tolerance
        top2 = cpu_max[order[:2]]
        assert top2[0] - top2[1] <= 2 * TOL * max(top2[0], 4.0), (cpu_best, gpu_best, top2)
        assert gpu_best == subset[int(order[1])]
    for o, t in zip(res, subset):
        assert o["cpu_argmax"] == idx[t, 0] or abs(o["cpu_max"] - val[t, 0]) <= TOL * max(o["cpu_max"], 4.0)
    if p.injection_template is not None:
        # the injected template peaks at the injected frequency with 2F ~ 4 + rho^2 (sd 2 sqrt(1 + rho^2 / 2)... here +- 5 sd);
        # rho = 12 stands above the loudest noise bin of 6.9e10 trials (~57), rho = 8 (2F ~ 68 +- 16) need not
        it, rho = p.injection_template, p.injection.rho
        inj_bin = int(round((p.injection.f - p.f_min) / p.df))
        assert idx[it, 0] == inj_bin
        assert abs(val[it, 0] - (4.0 + rho * rho)) < 5.0 * np.sqrt(2.0 * (4.0 + 2.0 * rho * rho))
        if rho >= 12.0:
            assert gpu_best == it


def test_config5_shape_sky_grid_dterms16():
    # config 5 geometry (Dterms 16, timing redone per sky position), 24 sky points around the injection
    full = synth.config5()
    i_sky = full.injection_template // 4
    lo = i_sky - 11
    p = full
    p.templates = full.templates[lo * 4:(lo + 24) * 4].copy()
    inj_local = full.injection_template - lo * 4
    cpu = O.fstat_2F_bank(p)
    with _plan(p) as plan:
        gpu = plan.compute(p.templates)
        plan.sync()
        gpu = gpu.cpu().numpy()
    assert _rel_err(gpu, cpu).max() <= TOL
    assert int(np.argmax(gpu.max(axis=1))) == int(np.argmax(cpu.max(axis=1)))      # loudest template identical
    # over 2 days neighbouring sky points are degenerate with frequency, so the loudest template need not be the
    # injected one (input recipe); the injected template itself carries 2F ~ 4 + rho^2 = 104 +- 20
    assert 50.0 < gpu[inj_local].max() < 170.0


def test_config5_full_bank_all_sky_batches_and_loudest_template(tmp_path):
    # the whole config-5 bank (4096 sky positions x 4 spin-downs = 16384 templates, FFT 2^18, Dterms 16) in the launch
    # structure bench.py times: 8 sky batches of 512 positions.  From every batch the complete rows of four sky positions
    # (first, last, two seeded random ones; all four spin-downs) are compared bin by bin with the oracle, and the oracle
    # runs over the WHOLE bank (tests/oracle_bank_maxima.py, all host cores) so that the loudest bin of every template
    # and the loudest template of the bank are checked, not only timed (VERDICT r2 missing 1)
    import torch
    p = synth.config5()
    n_t = len(p.templates)
    n_sky, per_batch = n_t // 4, 512
    assert n_sky == 4096 and np.all(p.templates[0::4, :2] == p.templates[3::4, :2])
    rng = np.random.default_rng(505)
    sky_sample = []
    for b in range(n_sky // per_batch):
        lo = b * per_batch
        sky_sample += [lo, lo + per_batch - 1] + [int(x) for x in lo + 1 + rng.choice(per_batch - 2, size=2, replace=False)]
    sample = sorted(4 * s + j for s in sky_sample for j in range(4))
    proc = _start_oracle_bank("config5", tmp_path / "config5.npz", sample)
    with _plan(p) as plan:
        full = plan.compute(p.templates)                        # 16384 x 131072 float32 = 8.6 GB on the GPU
        val, idx = plan.compute_topk(p.templates, 1)
        plan.sync()
        assert bool(torch.isfinite(full).all())
        m = full.max(dim=1)
        assert torch.equal(m.values, val[:, 0])                 # the top-k path agrees with the full rows, every template
        rows = full[sample].cpu().numpy()
        val, idx = val.cpu().numpy()[:, 0], idx.cpu().numpy()[:, 0]
        del full, m
        torch.cuda.empty_cache()
    ora = _finish_oracle_bank(proc, tmp_path / "config5.npz")
    np.testing.assert_array_equal(ora["row_idx"], sample)
    err = _rel_err(rows, ora["rows"])
    print(f"[parity] config5 full bank: {len(sample)} complete rows from all 8 sky batches: max |d2F|/max(2F,4) = {err.max():.2e}")
    assert err.max() <= TOL
    best = _check_bank_maxima(val, idx, ora, "config5 full bank")
    # over 2 days neighbouring sky points are degenerate with frequency (input recipe): the loudest template is
    # near the injected one on the sky, not necessarily it; the injected template carries 2F ~ 4 + rho^2
    assert 50.0 < val[p.injection_template] < 170.0 and val[best] >= val[p.injection_template]


def test_sky100_protocol_on_a_config3_cell():
    # the paper's own timing protocol (100 sky locations, results averaged) on the config-3 cell 5 d x 1 Hz
    # (FFT 2^20): the Farrow-filtered series (110 MB) exceeds what the sky kernel treats as L2-resident, so the batch
    # runs in the sky-position-fastest block order; sampled sky positions against the oracle, every bin, and every
    # sampled row bit-identical to the same template computed alone (one sky position per call: grid-index-fastest
    # order, batch of one)
    p = synth.config3(5, 1.0, n_templates=1)
    sky = synth.disc_sky_points(100, seed=77, radius=0.3)
    p.templates = np.array([(a, d, p.f_min, -5e-10, 0.0) for (a, d) in sky], dtype=np.float64)
    sample = [0, 17, 58, 99]
    with _plan(p) as plan:
        gpu = plan.compute(p.templates)
        plan.sync()
        assert bool(np.isfinite(gpu.cpu().numpy()).all())
        rows = gpu[sample].cpu().numpy()
        alone = np.stack([plan.compute(p.templates[i:i + 1]).cpu().numpy()[0] for i in sample])
        plan.sync()
    np.testing.assert_array_equal(rows, alone)
    for r, i in enumerate(sample):
        out = compare_rows(p, [i], rows[r:r + 1], label=f"sky100 on config3:5:1, sky position {i}")
        assert out[0]["err"] <= TOL
    # pure noise: every row is chi^2_4 distributed (mean 4, variance 8) whatever the sky position
    g = gpu.cpu().numpy().astype(np.float64)
    assert abs(g.mean() - 4.0) < 0.02 and abs(g.var() - 8.0) < 0.2
