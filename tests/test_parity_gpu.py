"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Tolerance (BASELINE.json north_star):
|2F_gpu - 2F_cpu| <= 1e-3 * max(2F_cpu, 4) per bin; loudest template identical."""
import math

import numpy as np
import pytest

from oracle import fstat_oracle as O
from paper_2201_00451_b200 import synth

pytestmark = pytest.mark.gpu

TOL = 1e-3


def _plan(prob, **kw):
    from paper_2201_00451_b200.binding import FstatPlan
    return FstatPlan(prob, **kw)


def _rel_err(gpu, cpu):
    return np.abs(gpu.astype(np.float64) - cpu) / np.maximum(cpu, 4.0)


def _check_bank(prob, idxs=None, tol=TOL):
    idxs = list(range(len(prob.templates))) if idxs is None else list(idxs)
    cpu = O.fstat_2F_bank(prob, idxs)
    with _plan(prob) as plan:
        gpu = plan.compute(prob.templates[idxs])
        plan.sync()
        gpu = gpu.cpu().numpy()
    assert gpu.shape == cpu.shape
    err = _rel_err(gpu, cpu)
    assert np.isfinite(gpu).all()
    assert err.max() <= tol, (err.max(), np.unravel_index(err.argmax(), err.shape))
    return gpu, cpu


# every sub-FFT length 2^6 .. 2^12 appears in one of these (n_fft = 2^12 .. 2^24 splits as L/2, L-L/2)
@pytest.mark.parametrize("log_nfft,n_samples,dt", [
    (12, 1500, 1.0), (13, 5000, 1.0), (14, 11000, 1.0), (15, 20000, 1.0), (16, 50001, 1.0),
    (17, 100003, 1.0), (18, 250000, 0.5), (19, 400001, 0.5),
])
def test_parity_small_all_bins(log_nfft, n_samples, dt):
    p = synth.small_problem(seed=log_nfft, n_samples=n_samples, dt=dt, n_fft=1 << log_nfft, n_templates=3,
                            gap_frac=0.3, rho=12.0, fddot=1e-16)
    gpu, cpu = _check_bank(p)
    assert int(np.argmax(gpu.max(axis=1))) == int(np.argmax(cpu.max(axis=1)))
    if n_samples * dt >= 50000:       # shorter spans cannot tell the fdot templates apart
        assert int(np.argmax(gpu.max(axis=1))) == p.injection_template


@pytest.mark.parametrize("log_nfft", [20, 21, 22])
def test_parity_large_fft_one_template(log_nfft):
    n = int(0.8 * (1 << log_nfft))
    p = synth.small_problem(seed=100 + log_nfft, n_samples=n, dt=0.5, n_fft=1 << log_nfft, n_templates=2,
                            gap_frac=0.4, rho=15.0)
    _check_bank(p, [p.injection_template])


def test_parity_maximum_fft_length():
    # n_fft = 2^24 = 2^12 x 2^12: the largest size fstat_setup accepts (both passes run their 2^12-point kernels)
    p = synth.small_problem(seed=124, n_det=1, n_samples=int(0.75 * (1 << 24)), dt=0.5, n_fft=1 << 24, n_templates=1,
                            gap_frac=0.4, rho=15.0)
    _check_bank(p, [0])


def test_parity_fs_equals_band_full_output():
    # config-4 shape: band = sample rate, every FFT output is a bin, f_het at band centre
    p = synth.small_problem(seed=3, n_samples=30000, dt=0.5, n_fft=1 << 16, n_templates=2, band=2.0, rho=10.0)
    assert p.n_bins == p.n_fft
    _check_bank(p)


def test_parity_dterms16_single_detector_no_gaps():
    p = synth.small_problem(seed=4, n_det=1, n_samples=40000, n_fft=1 << 16, dterms=16, gap_frac=0.0,
                            weights=False, n_templates=2, rho=20.0)
    _check_bank(p)


def test_parity_three_detectors():
    # odd detector count: the sky kernel takes detectors two at a time, the last one alone
    p = synth.small_problem(seed=5, n_det=3, n_samples=30000, n_fft=1 << 16, n_templates=2, gap_frac=0.35, rho=14.0)
    gpu, cpu = _check_bank(p)
    assert int(np.argmax(gpu.max(axis=1))) == int(np.argmax(cpu.max(axis=1))) == p.injection_template


@pytest.mark.parametrize("n_det", [4, 5])
def test_parity_four_and_five_detectors(n_det):
    # more than one full detector pair in the sky kernel's pair loop (4: two pairs; 5: two pairs and one alone)
    q = synth.small_problem(seed=50 + n_det, n_det=3, n_samples=30000, n_fft=1 << 16, n_templates=2, gap_frac=0.3, rho=14.0)
    extra = [dict(lat_rad=36.41 * synth.DEG, lon_east_rad=137.31 * synth.DEG, xarm_azimuth_rad=60.4 * synth.DEG),
             dict(lat_rad=19.61 * synth.DEG, lon_east_rad=77.03 * synth.DEG, xarm_azimuth_rad=207.0 * synth.DEG)]
    dets = (q.detectors + extra)[:n_det]
    p = synth.make_problem(f"det{n_det}", dets, q.n_samples, q.dt, q.f_min, q.band, q.f_het, q.n_fft, q.dterms, q.templates,
                           seed=q.seed, gap_frac=0.3, weight_range=(0.5, 2.0), injection=q.injection,
                           injection_template=q.injection_template, snap_injection_to_bin=True)
    assert p.n_det == n_det
    gpu, cpu = _check_bank(p)
    assert int(np.argmax(gpu.max(axis=1))) == int(np.argmax(cpu.max(axis=1))) == p.injection_template


@pytest.mark.parametrize("omega_rot", [1e-2, 0.5])
def test_parity_fast_rotation_ephemeris_without_orbit(omega_rot):
    # an ephemeris fstat_setup admits (omega * delay < 0.05 rad) that is nothing like the Earth: no orbit, a rotation
    # period of 10 minutes / 13 s.  The timing nodes (<= 256 s apart for the Earth) must move closer together for the
    # cubic Hermite interpolant of the delay to hold: fstat_setup bounds h^4/384 (re w_rot^4 + au w_orb^4) <= 1e-9 s
    # (at 0.5 rad/s every grid point becomes a node).  With 256 s nodes the delay would be off by milliseconds.
    eph = dict(synth.EPHEM_DEFAULT, au_over_c_s=0.0, omega_rot=omega_rot)
    p = synth.small_problem(seed=77, n_samples=20000, n_fft=1 << 15, n_templates=2, rho=12.0, ephem=eph)
    gpu, cpu = _check_bank(p)
    assert int(gpu[p.injection_template].argmax()) == int(cpu[p.injection_template].argmax())
    # and the resampled series itself (the delay enters through the sample index and the heterodyne phase)
    _check_resampled_series(p, float(p.templates[0, 0]), float(p.templates[0, 1]))


def _check_resampled_series(p, al, de):
    sky = O.per_sky(p, al, de)
    n_src = p.n_samples + 2 * O.k_margin(p)
    ya = np.zeros(n_src, dtype=np.complex128)
    yb = np.zeros(n_src, dtype=np.complex128)
    k = np.arange(n_src)
    for X in range(p.n_det):
        s = sky["det"][X]
        rot = np.exp(-2j * np.pi * np.mod(p.f_het * s["Delta"], 1.0))
        ya += s["wk"] * s["a"] * s["z"] * rot
        yb += s["wk"] * s["b"] * s["z"] * rot
    shift = np.exp(-2j * np.pi * O.band_shift_cycles(p, k))
    ya *= shift
    yb *= shift
    with _plan(p) as plan:
        S, abcd = plan.resample_sky(al, de)
        S = S.cpu().numpy().astype(np.float64)
    scale = np.abs(np.concatenate([ya, yb])).max()
    assert np.abs(S[:n_src, 0] + 1j * S[:n_src, 1] - ya).max() <= 2e-5 * scale
    assert np.abs(S[:n_src, 2] + 1j * S[:n_src, 3] - yb).max() <= 2e-5 * scale
    assert np.all(S[n_src:] == 0)
    np.testing.assert_allclose(abcd, np.array(sky["ABCD"]), rtol=2e-6)


def test_resampled_series_and_antenna_sums_match_oracle():
    p = synth.small_problem(seed=9, n_samples=30000, n_fft=1 << 15, n_templates=1)
    _check_resampled_series(p, *synth.SKY0)


def test_multiple_sky_positions_in_one_call():
    # config-5 shape: sky-major template order, sky-dependent work redone per sky position
    p = synth.small_problem(seed=12, n_samples=20000, n_fft=1 << 15, n_templates=2, rho=None)
    sky = synth.disc_sky_points(5, seed=1)
    rows = [(a, d, p.f_min, fd, 0.0) for (a, d) in sky for fd in (-3e-9, 0.0)]
    p.templates = np.array(rows)
    _check_bank(p)


def test_topk_matches_oracle_topk():
    p = synth.small_problem(seed=13, n_samples=30000, n_fft=1 << 15, n_templates=4, rho=14.0)
    k = 10
    cpu = O.fstat_2F_bank(p)
    with _plan(p) as plan:
        val, idx = plan.compute_topk(p.templates, k)
        full = plan.compute(p.templates)
        plan.sync()
        val, idx, full = val.cpu().numpy(), idx.cpu().numpy(), full.cpu().numpy()
        hv, hi = plan.compute_topk_host(p.templates, k)
    np.testing.assert_array_equal(hv, val)
    np.testing.assert_array_equal(hi, idx)
    for t in range(len(p.templates)):
        # bit-exact against the same selection rule applied to the GPU's own 2F row
        ev, ei = O.topk(full[t], k)
        np.testing.assert_array_equal(idx[t], ei)
        np.testing.assert_array_equal(val[t], ev)
        # and against the oracle: same loudest bin, values within tolerance
        cv, ci = O.topk(cpu[t], k)
        assert idx[t, 0] == ci[0]
        assert abs(val[t, 0] - cv[0]) <= TOL * max(cv[0], 4.0)
        assert np.all(np.diff(val[t]) <= 0)


def test_host_variant_equals_device_variant():
    p = synth.small_problem(seed=14, n_samples=20000, n_fft=1 << 15, n_templates=7)
    with _plan(p) as plan:
        dev = plan.compute(p.templates)
        plan.sync()
        host = plan.compute_host(p.templates)
        np.testing.assert_array_equal(host.numpy(), dev.cpu().numpy())
        plan.set_inflight(2)
        host2 = plan.compute_host(p.templates)
        np.testing.assert_array_equal(host2.numpy(), dev.cpu().numpy())
        assert plan.launch_count() > 0


def test_series_on_device_and_error_codes():
    from paper_2201_00451_b200.binding import FstatError, FSTAT_EDOM
    p = synth.small_problem(seed=15, n_samples=8000, n_fft=1 << 14, n_templates=2)
    with _plan(p) as a, _plan(p, series_on_device=True) as b:
        ra, rb = a.compute(p.templates), b.compute(p.templates)
        a.sync(); b.sync()
        np.testing.assert_array_equal(ra.cpu().numpy(), rb.cpu().numpy())
        bad = p.templates.copy()
        bad[0, 2] += 0.1
        with pytest.raises(FstatError) as ei:
            a.compute(bad)
        assert ei.value.code == FSTAT_EDOM
        a.compute(p.templates[:0])            # empty batch is a no-op


def test_empty_detector_gives_edom():
    from paper_2201_00451_b200.binding import FstatError, FSTAT_EDOM
    p = synth.small_problem(seed=16, n_det=1, n_samples=8000, n_fft=1 << 14, n_templates=1)
    p.timestamps = [p.timestamps[0][:0]]
    p.weights = [p.weights[0][:0]]
    with _plan(p) as plan:
        out = plan.compute(p.templates)
        with pytest.raises(FstatError) as ei:
            plan.sync()
        assert ei.value.code == FSTAT_EDOM
        assert np.isnan(out.cpu().numpy()).all()


@pytest.mark.parametrize("log_nfft,k", [(12, 3), (17, 1), (18, 64), (20, 16)])
def test_topk_select_matches_own_rows(log_nfft, k):
    # the fused selection (per-warp maxima from FFT pass 2 -> threshold -> hot groups) must reproduce,
    # bit for bit, the (2F desc, bin asc) selection applied to the full rows the same plan computes
    n = int(0.7 * (1 << log_nfft))
    p = synth.small_problem(seed=40 + log_nfft, n_samples=n, dt=0.5 if log_nfft > 17 else 1.0, n_fft=1 << log_nfft,
                            n_templates=3, gap_frac=0.3, rho=9.0)
    with _plan(p) as plan:
        val, idx = plan.compute_topk(p.templates, k)
        full = plan.compute(p.templates)
        plan.sync()
        val, idx, full = val.cpu().numpy(), idx.cpu().numpy(), full.cpu().numpy()
    for t in range(len(p.templates)):
        ev, ei = O.topk(full[t], k)
        np.testing.assert_array_equal(idx[t], ei)
        np.testing.assert_array_equal(val[t], ev)


def test_topk_degenerate_rows_take_the_exact_slow_path():
    # all-zero data: every bin ties at 2F = 0 -> bins 0..k-1 in order (S15)
    p = synth.small_problem(seed=41, n_samples=20000, n_fft=1 << 15, n_templates=2, rho=None, noise=False)
    with _plan(p) as plan:
        val, idx = plan.compute_topk(p.templates, 5)
        plan.sync()
        np.testing.assert_array_equal(idx.cpu().numpy(), np.tile(np.arange(5, dtype=np.int32), (2, 1)))
        np.testing.assert_array_equal(val.cpu().numpy(), np.zeros((2, 5), dtype=np.float32))
    # D <= 0 (no valid data): rows are NaN -> (-inf, -1)
    from paper_2201_00451_b200.binding import FstatError
    q = synth.small_problem(seed=16, n_det=1, n_samples=8000, n_fft=1 << 14, n_templates=1)
    q.timestamps = [q.timestamps[0][:0]]
    q.weights = [q.weights[0][:0]]
    with _plan(q) as plan:
        val, idx = plan.compute_topk(q.templates, 4)
        with pytest.raises(FstatError):
            plan.sync()
        assert np.all(idx.cpu().numpy() == -1) and np.all(np.isneginf(val.cpu().numpy()))


@pytest.mark.parametrize("thr,k", [(18.0, 16), (30.0, 4), (1e6, 3), (12.0, 64)])
def test_threshold_retention_matches_oracle_rule(thr, k):
    # keep 2F > threshold on the GPU.  Bit-exact against the same rule applied to the GPU's own rows;
    # the loudest candidate and the count agree with the oracle's rows up to bins within tolerance of the threshold.
    p = synth.small_problem(seed=50, n_samples=60000, n_fft=1 << 17, n_templates=3, gap_frac=0.3, rho=11.0)
    cpu = O.fstat_2F_bank(p)
    with _plan(p) as plan:
        val, idx, cnt = plan.compute_threshold(p.templates, thr, k)
        full = plan.compute(p.templates)
        plan.sync()
        val, idx, cnt, full = val.cpu().numpy(), idx.cpu().numpy(), cnt.cpu().numpy(), full.cpu().numpy()
    for t in range(len(p.templates)):
        ev, ei, ec = O.threshold_candidates(full[t], np.float32(thr), k)
        assert cnt[t] == ec
        n = len(ei)
        np.testing.assert_array_equal(idx[t, :n], ei)
        np.testing.assert_array_equal(val[t, :n], ev)
        assert np.all(idx[t, n:] == -1) and np.all(np.isneginf(val[t, n:]))
        # against the oracle: bins clearly above / below the threshold are counted alike
        lo = int(np.sum(cpu[t] > thr * (1 + 2 * TOL) + 8 * TOL)); hi = int(np.sum(cpu[t] > thr * (1 - 2 * TOL) - 8 * TOL))
        assert lo <= cnt[t] <= hi


def test_results_do_not_depend_on_templates_per_launch():
    # chunked launches (fstat_set_inflight) and a sky-major bank larger than one launch give the same bits
    p = synth.small_problem(seed=21, n_samples=9000, n_fft=1 << 14, n_templates=3, rho=None)
    sky = synth.disc_sky_points(7, seed=2)
    p.templates = np.array([(a, d, p.f_min, fd, 0.0) for (a, d) in sky for fd in (-2e-9, -1e-9, 0.0)])
    with _plan(p) as plan:
        full = plan.compute(p.templates)
        val, idx = plan.compute_topk(p.templates, 6)
        plan.sync()
        full, val, idx = full.cpu().numpy(), val.cpu().numpy(), idx.cpu().numpy()
        plan.set_inflight(4)
        full2 = plan.compute(p.templates)
        val2, idx2 = plan.compute_topk(p.templates, 6)
        tv, ti, tc = plan.compute_threshold(p.templates, 14.0, 6)
        plan.sync()
        np.testing.assert_array_equal(full2.cpu().numpy(), full)
        np.testing.assert_array_equal(val2.cpu().numpy(), val)
        np.testing.assert_array_equal(idx2.cpu().numpy(), idx)
        assert np.array_equal(tc.cpu().numpy(), (full > 14.0).sum(axis=1))


@pytest.mark.parametrize("case", range(10))
def test_parity_random_geometries(case):
    # unusual plans: Dterms 1..32, sample intervals that are not powers of two, narrow bands off the heterodyne
    # frequency, 1-3 detectors, heavy gaps, second spin-down
    rng = np.random.default_rng(1000 + case)
    dt = float(rng.choice([0.25, 0.5, 0.7, 1.0, 3.0]))
    log_nfft = int(rng.integers(12, 17))
    km2 = 2 * int(np.ceil(512.0 / dt))
    while (1 << log_nfft) < 2 * km2:               # room for data beside the 2 x 512 s margins
        log_nfft += 1
    n_samples = int(rng.uniform(0.35, 0.95) * ((1 << log_nfft) - km2))
    if n_samples * dt < 2 * 1800.0:                # at least two 1800 s slots of data
        n_samples = int(min(((1 << log_nfft) - km2), 2.5 * 1800.0 / dt))
    band = float(rng.choice([1.0, 0.5, 0.25, 0.1])) / dt
    p = synth.small_problem(seed=2000 + case, n_det=int(rng.integers(1, 4)), n_samples=n_samples, dt=dt, n_fft=1 << log_nfft,
                            dterms=int(rng.choice([1, 3, 8, 20, 32])), n_templates=3, gap_frac=0.0,
                            weights=bool(rng.integers(0, 2)), rho=float(rng.choice([6.0, 15.0])), f_min=float(rng.uniform(20.0, 900.0)),
                            band=band, fddot=float(rng.choice([0.0, 3e-15])))
    # heterodyne frequency away from the band centre (the plan shifts the band to FFT bin 0)
    p.f_het = p.f_min + float(rng.uniform(0.0, 1.0)) * band
    gap = 0.3 if n_samples * dt >= 8 * 1800.0 else 0.0          # keep at least a few data slots
    p = synth.make_problem(p.name, p.detectors, p.n_samples, p.dt, p.f_min, p.band, p.f_het, p.n_fft, p.dterms, p.templates,
                           seed=p.seed, gap_frac=gap, weight_range=(0.5, 2.0), injection=p.injection,
                           injection_template=p.injection_template, snap_injection_to_bin=True)
    _check_bank(p)
