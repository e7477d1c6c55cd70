"""GPU parity of the entry points beyond fstat_compute / top-k: the semi-coherent accumulation over segment plans
(PAPER.md:325), the single-detector statistic, selection over caller rows, exact band placement
with an off-grid heterodyne frequency, and the launch-shape / multi-batch paths reached through fstat_debug.h."""
import numpy as np
import pytest

from oracle import fstat_oracle as O
from paper_2201_00451_b200 import synth
from _parity_util import TOL, rel_err

pytestmark = pytest.mark.gpu


def _plan(prob, **kw):
    from paper_2201_00451_b200.binding import FstatPlan
    return FstatPlan(prob, **kw)


@pytest.mark.parametrize("off", [0.45, -0.3])
def test_off_grid_heterodyne_bins_are_labelled_exactly(off):
    # DESIGN.md S13: bin q is f_min + q df whatever f_het; the injection sits exactly on a labelled bin
    q = synth.small_problem(seed=60, rho=12.0, n_templates=3, n_samples=20000, n_fft=1 << 15)
    p = synth.small_problem(seed=60, rho=12.0, n_templates=3, n_samples=20000, n_fft=1 << 15, f_het=q.f_het + off * q.df)
    cpu = O.fstat_2F_bank(p)
    with _plan(p) as plan:
        gpu = plan.compute(p.templates)
        plan.sync()
        gpu = gpu.cpu().numpy()
    assert rel_err(gpu, cpu).max() <= TOL
    inj_bin = int(round((p.injection.f - p.f_min) / p.df))
    assert gpu[p.injection_template].argmax() == inj_bin == cpu[p.injection_template].argmax()


def test_semicoherent_accumulate_three_segments():
    # three segments of a config-2-like problem (two detectors, gaps, weights), each with its own plan; the sum of 2F
    # over segments with per-segment bin offsets, then top-k / threshold on the sum
    import torch
    n_seg = 3
    probs = [synth.small_problem(seed=90 + s, rho=(7.0, 9.0, 8.0)[s], n_samples=60000, dt=0.5, n_fft=1 << 17, n_templates=4, gap_frac=0.3)
             for s in range(n_seg)]
    n_t, nb = len(probs[0].templates), probs[0].n_bins
    offs = np.array([[0, 0, 0, 0], [3, -2, 0, 11], [-5, 0, 7, -1]], dtype=np.int32)      # [segment][template]
    cpu = np.stack([O.fstat_2F_semicoherent(probs, [q.templates[t] for q in probs], offs[:, t]) for t in range(n_t)])
    plans = [_plan(q) for q in probs]
    try:
        tot = torch.zeros((n_t, nb), dtype=torch.float32, device="cuda")
        for s, plan in enumerate(plans):
            plan.compute_accumulate(probs[s].templates, tot, offs[s])
            plan.sync()
        val, idx = plans[0].select_topk(tot, 6)
        tv, ti, tc = plans[0].select_threshold(tot, 40.0, 6)
        plans[0].sync()
        g = tot.cpu().numpy()
        err = np.abs(g - cpu) / np.maximum(cpu, 4.0 * n_seg)
        assert err.max() <= TOL, err.max()
        for t in range(n_t):
            ev, ei = O.topk(g[t], 6)
            np.testing.assert_array_equal(idx.cpu().numpy()[t], ei)
            np.testing.assert_array_equal(val.cpu().numpy()[t], ev)
            cv, ci, cc = O.threshold_candidates(g[t], np.float32(40.0), 6)
            assert tc.cpu().numpy()[t] == cc
            np.testing.assert_array_equal(ti.cpu().numpy()[t, :len(ci)], ci)
            assert idx.cpu().numpy()[t, 0] == cpu[t].argmax()
        # without offsets and on a fresh array == plain sum of fstat_compute rows (bit for bit: same adds in the same order)
        tot2 = torch.zeros((n_t, nb), dtype=torch.float32, device="cuda")
        ref = torch.zeros((n_t, nb), dtype=torch.float32, device="cuda")
        for s, plan in enumerate(plans):
            plan.compute_accumulate(probs[s].templates, tot2)
            ref += plan.compute(probs[s].templates)
            plan.sync()
        assert torch.equal(tot2, ref)
    finally:
        for plan in plans:
            plan.close()


def test_per_detector_statistic_matches_oracle():
    p = synth.small_problem(seed=95, n_det=3, rho=14.0, n_samples=30000, n_fft=1 << 16, n_templates=2, gap_frac=0.3)
    cpu = np.stack([O.fstat_2F_per_detector(p, t) for t in p.templates], axis=1)       # [n_det][n_tmpl][n_bins]
    with _plan(p) as plan:
        gpu = plan.compute_per_detector(p.templates)
        coh = plan.compute(p.templates)
        plan.sync()
        gpu, coh = gpu.cpu().numpy(), coh.cpu().numpy()
    assert gpu.shape == cpu.shape
    assert rel_err(gpu, cpu).max() <= TOL
    assert rel_err(coh, O.fstat_2F_bank(p)).max() <= TOL          # the coherent path is untouched by the masked runs


def test_per_detector_with_an_all_gap_detector_gives_nan_rows_and_edom():
    # detector 1 has no data segment at all: D_1 <= 0, its rows are NaN and fstat_sync reports FSTAT_EDOM; the rows of the
    # detectors that do have data are unaffected
    from paper_2201_00451_b200.binding import FstatError, FSTAT_EDOM
    p = synth.small_problem(seed=97, n_det=3, rho=14.0, n_samples=30000, n_fft=1 << 16, n_templates=2, gap_frac=0.3)
    p.timestamps[1] = p.timestamps[1][:0]
    p.weights[1] = p.weights[1][:0]
    p.series[1] = np.zeros_like(p.series[1])
    with _plan(p) as plan:
        gpu = plan.compute_per_detector(p.templates)
        with pytest.raises(FstatError) as ei:
            plan.sync()
        assert ei.value.code == FSTAT_EDOM
        gpu = gpu.cpu().numpy()
        coh = plan.compute(p.templates)                 # the coherent statistic over the two live detectors is fine
        plan.sync()
        coh = coh.cpu().numpy()
    assert np.isnan(gpu[1]).all()
    for X in (0, 2):
        cpu = np.stack([O.fstat_2F(O.single_detector_view(p, X), t) for t in p.templates])
        assert rel_err(gpu[X], cpu).max() <= TOL
    assert rel_err(coh, O.fstat_2F_bank(p)).max() <= TOL


def test_accumulate_with_bin_offsets_across_several_launches():
    # n_tmpl > templates per launch: the per-template bin offsets must follow their templates through the chunking
    # (fstat_set_inflight(4), 11 templates of 3 sky positions -> 3+ launches); bit-identical to the one-launch result and
    # equal to the oracle's shifted rows
    import torch
    p = synth.small_problem(seed=98, n_samples=9000, n_fft=1 << 14, n_templates=3, rho=9.0)
    sky = [(3.52, -0.83), (1.1, 0.4), (5.0, 1.0)]
    tm = [(a, d, p.f_min, fd, 0.0) for (a, d) in sky for fd in (-2e-9, -1e-9, 0.0, 1e-9)][:11]
    p.templates = np.array(tm)
    n_t, nb = len(tm), p.n_bins
    offs = np.array([0, 5, -3, 17, -40, 0, 1, -1, nb - 1, -(nb - 1), 250], dtype=np.int32)
    cpu = O.fstat_2F_bank(p)
    want = np.zeros_like(cpu)
    for t in range(n_t):
        q = np.arange(nb) - offs[t]                       # bin q of the plan lands on output bin q - off
        ok = (q >= 0) & (q < nb)
        want[t, q[ok]] = cpu[t, ok]
    with _plan(p) as plan:
        one = torch.zeros((n_t, nb), dtype=torch.float32, device="cuda")
        plan.compute_accumulate(p.templates, one, offs)
        plan.sync()
        plan.set_inflight(4)
        many = torch.zeros((n_t, nb), dtype=torch.float32, device="cuda")
        plan.compute_accumulate(p.templates, many, offs)
        plan.compute_accumulate(p.templates, many, offs)             # twice: the second pass adds to the first
        plan.sync()
        one, many = one.cpu().numpy(), many.cpu().numpy()
    assert (np.abs(one - want) / np.maximum(want, 4.0)).max() <= TOL
    np.testing.assert_array_equal(many, one + one)


@pytest.mark.parametrize("log_nfft,n_samples,dt,noise,rho", [
    (15, 20000, 1.0, False, 30.0), (17, 100003, 1.0, True, 8.0), (19, 400001, 0.5, True, 8.0), (20, 700000, 0.5, False, 30.0),
    (21, 1500000, 0.5, True, 8.0)])
def test_fa_fb_spectra_match_oracle(log_nfft, n_samples, dt, noise, rho):
    # the paper's accuracy tooling compares three vectors, "the output for F, Fa, and Fb" (Fig. 4: L2
    # relative errors up to ~1e-5): 2F alone cannot see a slip that leaves the quadratic form of eq. 8 unchanged
    # (Fa <-> conj Fa, a phase common to Fa and Fb).  Signal-dominated (no noise) and noisy cases; the oracle and the
    # library share the SSB grid convention (index 0 at t_start - K_m dt), so the spectra compare directly.
    p = synth.small_problem(seed=300 + log_nfft, rho=rho, noise=noise, n_templates=2, n_samples=n_samples, dt=dt,
                            n_fft=1 << log_nfft, fddot=1e-16 if log_nfft == 17 else 0.0)
    with _plan(p) as plan:
        fa, fb = plan.debug_compute_fafb(p.templates)
        twoF = plan.compute(p.templates)
        plan.sync()
        fa, fb, twoF = fa.cpu().numpy(), fb.cpu().numpy(), twoF.cpu().numpy()
    for t in range(len(p.templates)):
        Fa, Fb, (A, B, C, D) = O.fstat_FaFb(p, p.templates[t])
        cpu2F = O.twoF_from_FaFb(Fa, Fb, A, B, C, D)
        for name, g, c in (("Fa", fa[t], Fa), ("Fb", fb[t], Fb), ("2F", twoF[t], cpu2F)):
            r1, r2, th = O.comparison_metrics(g.astype(np.complex128 if name != "2F" else np.float64), c)
            print(f"[parity] n_fft 2^{log_nfft}, template {t}, {name}: r1 = {r1:.2e}, r2 = {r2:.2e}, theta = {th:.2e} rad (eq. 9-10)")
            assert r2 <= 1e-5 and th <= 1e-3, (name, r1, r2, th)
        # bin by bin, against the largest magnitude of the row (fp32 FFT: errors scale with the row's norm, not the bin's)
        scale = max(np.abs(Fa).max(), np.abs(Fb).max())
        assert np.abs(fa[t] - Fa).max() <= 2e-5 * scale and np.abs(fb[t] - Fb).max() <= 2e-5 * scale
        # and eq. 8 applied to the library's own spectra reproduces its 2F (same registers, fp64 combination here)
        own = O.twoF_from_FaFb(fa[t].astype(np.complex128), fb[t].astype(np.complex128), A, B, C, D)
        assert rel_err(twoF[t], own).max() <= 1e-4


def test_two_live_topk_plans_of_different_size():
    # the dynamic shared memory attribute of the selection kernel is per function, not per plan
    big = synth.small_problem(seed=96, n_samples=int(0.7 * (1 << 20)), dt=0.5, n_fft=1 << 20, n_templates=2, rho=10.0)
    small = synth.small_problem(seed=97, n_samples=9000, n_fft=1 << 14, n_templates=2, rho=10.0)
    with _plan(big) as a, _plan(small) as b:
        for _ in range(2):
            for plan, prob in ((a, big), (b, small), (a, big)):
                val, idx = plan.compute_topk(prob.templates, 16)
                full = plan.compute(prob.templates)
                plan.sync()
                for t in range(2):
                    ev, ei = O.topk(full.cpu().numpy()[t], 16)
                    np.testing.assert_array_equal(idx.cpu().numpy()[t], ei)
                    np.testing.assert_array_equal(val.cpu().numpy()[t], ev)


def test_sky_major_bank_spanning_several_sky_batches():
    # more sky groups than resampled-series slots: slots are reused batch after batch (fstat_debug_set_max_sky_slots)
    p = synth.small_problem(seed=98, n_samples=20000, n_fft=1 << 15, n_templates=2, rho=None)
    sky = synth.disc_sky_points(11, seed=3)
    p.templates = np.array([(a, d, p.f_min, fd, 0.0) for (a, d) in sky for fd in (-3e-9, 0.0, -1e-9)])
    cpu = O.fstat_2F_bank(p)
    with _plan(p) as plan:
        ref = plan.compute(p.templates)
        plan.sync()
        ref = ref.cpu().numpy()
        assert rel_err(ref, cpu).max() <= TOL
        for slots in (1, 3, 4):
            plan.debug_set_max_sky_slots(slots)
            got = plan.compute(p.templates)
            val, idx = plan.compute_topk(p.templates, 3)
            plan.sync()
            np.testing.assert_array_equal(got.cpu().numpy(), ref)
            np.testing.assert_array_equal(idx.cpu().numpy()[:, 0], ref.argmax(axis=1))


@pytest.mark.parametrize("log_nfft,shapes", [
    (16, [(8, 11, 11, 16), (8, 12, 12, 16), (7, 11, 12, 16), (9, 11, 12, 16), (9, 11, 12, 32), (9, 12, 11, 16), (6, 11, 11, 16), (10, 11, 12, 32)]),
    (19, [(9, 11, 12, 32), (9, 12, 12, 16), (10, 11, 12, 32), (10, 11, 13, 32), (10, 11, 12, 16), (8, 11, 12, 16), (8, 12, 11, 16), (7, 12, 12, 16)]),
    (22, [(11, 11, 12, 16), (11, 12, 13, 16), (10, 12, 13, 32), (10, 13, 12, 16), (12, 11, 13, 16), (12, 11, 12, 16), (11, 13, 11, 16)]),
])
def test_every_instantiated_launch_shape_gives_the_same_answer(log_nfft, shapes):
    # fstat_debug_set_geometry: (log_n2, tile1, tile2, pass-2 elements); each shape against the oracle
    n = int(0.72 * (1 << log_nfft))
    p = synth.small_problem(seed=300 + log_nfft, n_samples=n, dt=0.5, n_fft=1 << log_nfft, n_templates=2, gap_frac=0.3, rho=11.0)
    sample = [p.injection_template]
    cpu = O.fstat_2F_bank(p, sample)
    from paper_2201_00451_b200.binding import FstatError
    with _plan(p) as plan:
        for (ln2, t1, t2, e) in shapes:
            plan.debug_set_geometry(ln2, t1, t2, e)
            gpu = plan.compute(p.templates[sample])
            val, idx = plan.compute_topk(p.templates[sample], 5)
            plan.sync()
            gpu = gpu.cpu().numpy()
            assert rel_err(gpu, cpu).max() <= TOL, (ln2, t1, t2, e)
            ev, ei = O.topk(gpu[0], 5)
            np.testing.assert_array_equal(idx.cpu().numpy()[0], ei)
        with pytest.raises(FstatError):
            plan.debug_set_geometry(5, 11, 11, 16)                # no 2^5-point kernel
        plan.debug_set_geometry()                                 # back to the default
        gpu = plan.compute(p.templates[sample])
        plan.sync()
        assert rel_err(gpu.cpu().numpy(), cpu).max() <= TOL


def _sky_bank(p, n_sky, fdots, seed, fddot=0.0):
    sky = synth.disc_sky_points(n_sky, seed=seed)
    rows = []
    for s, (a, d) in enumerate(sky):
        for fd in fdots[: 1 + (s % len(fdots))] if isinstance(fdots, tuple) else fdots:
            rows.append((a, d, p.f_min, fd, fddot))
    return np.array(rows)


@pytest.mark.parametrize("log_nfft,n_samples,dt,fddot", [(15, 20000, 1.0, 0.0), (17, 100003, 1.0, 2e-15), (18, 250000, 0.5, 0.0), (12, 1500, 1.0, 0.0)])
def test_fused_sky_pass1_matches_oracle_and_hoisted_path(log_nfft, n_samples, dt, fddot):
    # sky-varying bank: the per-sky work runs inside the FFT pass-1 prologue (no resampled series in
    # global memory).  Ragged bank: 1..3 spin-down templates per sky position; several launches (small in-flight count).
    p = synth.small_problem(seed=400 + log_nfft, n_samples=n_samples, dt=dt, n_fft=1 << log_nfft, n_templates=2, gap_frac=0.3, rho=None)
    p.templates = _sky_bank(p, 9, (-3e-9, 0.0, -1e-9), seed=5, fddot=fddot)
    cpu = O.fstat_2F_bank(p)
    with _plan(p) as plan:
        plan.debug_set_geometry(log_tile1=11)                 # the fused kernel's tile shape (16 elements per thread)
        plan.debug_set_paths(fused_sky=0)
        hoisted = plan.compute(p.templates)
        plan.sync()
        hoisted = hoisted.cpu().numpy()
        plan.debug_set_paths(fused_sky=1)
        l0 = plan.launch_count()
        plan.set_profile(True)
        fused = plan.compute(p.templates)
        plan.sync()
        prof = plan.get_profile()
        plan.set_profile(False)
        assert prof["fused_sky_pass1"][1] >= 1 and prof["fft_pass1"][1] == 0       # the fused kernel ran, the plain pass 1 did not
        fused = fused.cpu().numpy()
        assert rel_err(hoisted, cpu).max() <= TOL
        assert rel_err(fused, cpu).max() <= TOL
        np.testing.assert_allclose(fused, hoisted, rtol=0, atol=2e-5 * max(4.0, float(cpu.max())))
        plan.set_inflight(4)                                   # several launches, sky groups never split
        again = plan.compute(p.templates)
        val, idx = plan.compute_topk(p.templates, 4)
        per = plan.compute_per_detector(p.templates[:5])
        plan.sync()
        np.testing.assert_array_equal(again.cpu().numpy(), fused)
        np.testing.assert_array_equal(idx.cpu().numpy()[:, 0], fused.argmax(axis=1))
        cpu_per = np.stack([O.fstat_2F_per_detector(p, t) for t in p.templates[:5]], axis=1)
        assert rel_err(per.cpu().numpy(), cpu_per).max() <= TOL
        plan.debug_set_paths()                                 # automatic: the hoisted form (measured faster)
        plan.set_inflight(0)
        plan.set_profile(True)
        auto = plan.compute(p.templates)
        plan.sync()
        assert plan.get_profile()["fused_sky_pass1"][1] == 0
        np.testing.assert_array_equal(auto.cpu().numpy(), hoisted)


@pytest.mark.parametrize("log_nfft,n_samples,dt,n_t", [(12, 1500, 1.0, 5), (13, 5000, 1.0, 3), (14, 11000, 1.0, 3), (15, 20000, 1.0, 200),
                                                       (16, 50001, 1.0, 7), (17, 100003, 1.0, 40), (18, 250000, 0.5, 30)])
def test_single_kernel_form_matches_two_launch_form_and_oracle(log_nfft, n_samples, dt, n_t):
    # small transforms: both FFT passes in one cooperative kernel, groups of templates through an L2-resident buffer with a
    # grid-wide barrier per group (n_t is chosen so that 2^15, 2^17 and 2^18 need 2-3 groups)
    p = synth.small_problem(seed=500 + log_nfft, n_samples=n_samples, dt=dt, n_fft=1 << log_nfft, n_templates=n_t, gap_frac=0.3,
                            rho=11.0, fddot=3e-16 if log_nfft % 2 else 0.0)
    sample = sorted({0, p.injection_template, n_t - 1})
    cpu = O.fstat_2F_bank(p, sample)
    with _plan(p) as plan:
        # both passes on 2^11-element tiles and the split the single-kernel form is instantiated for
        plan.debug_set_geometry(log_n2={12: 6, 13: 6, 14: 7, 15: 6, 16: 6, 17: 7, 18: 8}[log_nfft], log_tile1=11, log_tile2=11)
        plan.debug_set_paths(single=0)
        plan.set_profile(True)
        two = plan.compute(p.templates)
        plan.sync()
        prof = plan.get_profile()
        assert prof["fft_single"][1] == 0 and prof["fft_pass1"][1] >= 1
        plan.debug_set_paths(single=1)
        one = plan.compute(p.templates)
        val, idx = plan.compute_topk(p.templates, 5)
        plan.sync()
        prof = plan.get_profile()
        plan.set_profile(False)
        assert prof["fft_single"][1] == 2 and prof["fft_pass1"][1] == 0 and prof["fft_pass2"][1] == 0
        two, one = two.cpu().numpy(), one.cpu().numpy()
        np.testing.assert_array_equal(one, two)                   # same tiles, same arithmetic, same order
        assert rel_err(one[sample], cpu).max() <= TOL
        for t in sample:
            ev, ei = O.topk(one[t], 5)
            np.testing.assert_array_equal(idx.cpu().numpy()[t], ei)
            np.testing.assert_array_equal(val.cpu().numpy()[t], ev)
        assert int(np.argmax(one.max(axis=1))) == p.injection_template or n_samples * dt < 50000
