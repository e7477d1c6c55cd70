"""CPU oracle for the resampling F-statistic hot path.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` legs may import this file.  The product path
(`paper_2201_00451_b200`) never does, and this file imports nothing from the
product: it only reads the attributes of a `Problem` object made by the shared
input generator `paper_2201_00451_b200.synth`.

Plain numpy, float64 / complex128 throughout.  The method (PAPER.md:77-87,
steps (iii)-(vii) of "Resamp") is an approximation scheme -- interpolation with
a truncated kernel and dt/dt_b ~ 1 -- so this file follows the
algorithm step by step in the paper's order with every free choice fixed as in
DESIGN.md "Readings" (G1-G6, S1-S19).  `numpy.fft.fft` is the one library
primitive used as a step ("computing the FFTs").  No blocking,
fusion or reordering: arrays are recomputed per call unless the caller passes
the per-sky cache explicitly (memoisation of identical values, not a
reordering).

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): P1 chi^2_4 noise statistics,
P2 noise-free 2F = rho^2, P3 E[2F]=4+rho^2, P4 brute-force detector-frame sum
(eq. 4-5) on tiny inputs, P5 antenna closed form vs tensor form, P6
invariances, P7 zero-delay special case = plain zero-padded numpy FFT, P8 the
chi^2_4 tail against the paper's printed false-alarm figure,
Fig. 1's code formula with E=0 against eq. 8; eq. 9-10 metrics on hand-computed
vectors; the semi-coherent sum (chi^2 with 4 N_seg dof, sum of rho^2_seg); the
single-detector statistic (sum_X rho_X^2 = rho^2).  No function is unpinned.
"""
from __future__ import annotations

import math
from typing import Dict, Optional, Tuple

import numpy as np


# ---------------------------------------------------------------------------
# Timing model (S3: analytic circular orbit + sidereal rotation,
# Roemer delay only).  t_m(t; alpha, delta) of PAPER.md:44-46 (eq. 3).
# ---------------------------------------------------------------------------
def ssb_delay(det: dict, eph: dict, alpha: float, delta: float, tp: np.ndarray) -> np.ndarray:
    """Delta_X(t') = n.(r_orb + r_X)/c  with t' = t - t_start  [seconds]."""
    nx = math.cos(delta) * math.cos(alpha)
    ny = math.cos(delta) * math.sin(alpha)
    nz = math.sin(delta)
    phi_o = eph["phi_orb0"] + eph["omega_orb"] * tp
    eps = eph["obliquity_rad"]
    theta = eph["gmst0_rad"] + eph["omega_rot"] * tp + det["lon_east_rad"]
    lam = det["lat_rad"]
    orb = eph["au_over_c_s"] * (nx * np.cos(phi_o) + ny * np.sin(phi_o) * math.cos(eps)
                                + nz * np.sin(phi_o) * math.sin(eps))
    rot = eph["re_over_c_s"] * (nx * math.cos(lam) * np.cos(theta) + ny * math.cos(lam) * np.sin(theta)
                                + nz * math.sin(lam))
    return orb + rot


# ---------------------------------------------------------------------------
# Antenna patterns a(t), b(t): eq. (12)-(13) of ref. [24], arms at
# 90 deg; gamma = x-arm azimuth (CCW from North) + 135 deg (S1, S2).
# ---------------------------------------------------------------------------
def antenna_ab(det: dict, eph: dict, alpha: float, delta: float, tp: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    lam = det["lat_rad"]
    gam = det["xarm_azimuth_rad"] + 0.75 * math.pi
    theta = eph["gmst0_rad"] + eph["omega_rot"] * tp + det["lon_east_rad"]
    h = alpha - theta
    s2g, c2g = math.sin(2 * gam), math.cos(2 * gam)
    a = (s2g * (3.0 - math.cos(2 * lam)) * (3.0 - math.cos(2 * delta)) / 16.0 * np.cos(2 * h)
         - 0.25 * c2g * math.sin(lam) * (3.0 - math.cos(2 * delta)) * np.sin(2 * h)
         + 0.25 * s2g * math.sin(2 * lam) * math.sin(2 * delta) * np.cos(h)
         - 0.5 * c2g * math.cos(lam) * math.sin(2 * delta) * np.sin(h)
         + 0.75 * s2g * math.cos(lam) ** 2 * math.cos(delta) ** 2)
    b = (c2g * math.sin(lam) * math.sin(delta) * np.cos(2 * h)
         + 0.25 * s2g * (3.0 - math.cos(2 * lam)) * math.sin(delta) * np.sin(2 * h)
         + c2g * math.cos(lam) * math.cos(delta) * np.cos(h)
         + 0.5 * s2g * math.sin(2 * lam) * math.cos(delta) * np.sin(h))
    return a, b


# ---------------------------------------------------------------------------
# Segment weights (S10): weight per (detector, 1800 s slot), 0 in gaps.
# ---------------------------------------------------------------------------
def slot_weights(prob, X: int) -> np.ndarray:
    n_slots = int(math.ceil(prob.n_samples * prob.dt / prob.t_sft - 1e-9))
    w = np.zeros(n_slots)
    idx = np.rint((np.asarray(prob.timestamps[X], dtype=np.float64) - prob.t_start) / prob.t_sft).astype(np.int64)
    w[idx] = np.asarray(prob.weights[X], dtype=np.float64)
    return w


def antenna_sums(prob, alpha: float, delta: float) -> Tuple[float, float, float, float]:
    """A, B, C, D = AB - C^2: sums of w a^2, w b^2, w a b over the valid
    DETECTOR-frame samples of all detectors (S11, G6)."""
    A = B = C = 0.0
    tp = np.arange(prob.n_samples, dtype=np.float64) * prob.dt
    for X, det in enumerate(prob.detectors):
        w = slot_weights(prob, X)
        slot = np.minimum(np.floor(tp / prob.t_sft).astype(np.int64), len(w) - 1)
        ws = w[slot]
        a, b = antenna_ab(det, prob.ephem, alpha, delta, tp)
        A += float(np.sum(ws * a * a))
        B += float(np.sum(ws * b * b))
        C += float(np.sum(ws * a * b))
    return A, B, C, A * B - C * C


# ---------------------------------------------------------------------------
# Steps 1-4 (per sky position): SSB grid, inverse timing, validity, interpolation
# PAPER.md:82-83 (steps iv, v).
# ---------------------------------------------------------------------------
def k_margin(prob) -> int:
    return int(math.ceil(512.0 / prob.dt))


def ssb_grid_timing(prob, X: int, alpha: float, delta: float, n_iter: int = 6):
    """tau'_k = (k - K_m) dt ; solve T' = tau' - Delta_X(T') by fixed-point
    iteration from T' = tau' (contraction factor <= 1e-4 per iteration).
    Returns (tau', T', Delta)."""
    km = k_margin(prob)
    n_src = prob.n_samples + 2 * km
    tau = (np.arange(n_src, dtype=np.float64) - km) * prob.dt
    T = tau.copy()
    for _ in range(n_iter):
        T = tau - ssb_delay(prob.detectors[X], prob.ephem, alpha, delta, T)
    return tau, T, tau - T


def windowed_sinc_interpolate(x: np.ndarray, u: np.ndarray, dterms: int) -> np.ndarray:
    """z(u) = sum_{m=-D..D} x[j0+m] sinc(d-m) W(d-m),  j0 = floor(u+1/2), d = u-j0,
    sinc(v) = sin(pi v)/(pi v),  W(v) = 0.54 + 0.46 cos(pi v/(D+1/2));
    terms with j0+m outside [0,N) are zero  (S6, S7)."""
    n = len(x)
    j0 = np.floor(u + 0.5).astype(np.int64)
    d = u - j0
    z = np.zeros(len(u), dtype=np.complex128)
    for m in range(-dterms, dterms + 1):
        v = d - m
        j = j0 + m
        ok = (j >= 0) & (j < n)
        coef = np.sinc(v) * (0.54 + 0.46 * np.cos(math.pi * v / (dterms + 0.5)))
        z += np.where(ok, x[np.clip(j, 0, n - 1)], 0.0) * coef
    return z


def per_sky(prob, alpha: float, delta: float) -> Dict[str, object]:
    """Everything that depends on (alpha, delta) only: per detector
    tau', T', Delta, validity weight w_k, z_k, a(T_k), b(T_k); and A, B, C, D."""
    out = {"det": []}
    for X in range(prob.n_det):
        tau, T, Delta = ssb_grid_timing(prob, X, alpha, delta)
        w = slot_weights(prob, X)
        inside = (T >= 0.0) & (T < prob.n_samples * prob.dt)
        slot = np.clip(np.floor(T / prob.t_sft).astype(np.int64), 0, len(w) - 1)
        wk = np.where(inside, w[slot], 0.0)
        x = prob.series[X].astype(np.complex128)
        z = windowed_sinc_interpolate(x, T / prob.dt, prob.dterms)
        a, b = antenna_ab(prob.detectors[X], prob.ephem, alpha, delta, T)
        out["det"].append(dict(tau=tau, T=T, Delta=Delta, wk=wk, z=z, a=a, b=b))
    out["ABCD"] = antenna_sums(prob, alpha, delta)
    return out


# ---------------------------------------------------------------------------
# Steps 5-8 (per template): phases, Fa(t), Fb(t), FFTs, 2F.  PAPER.md:81, :84-85,
# eq. 8 in the unit-free normalisation of DESIGN.md G5.
# ---------------------------------------------------------------------------
def band_shift_cycles(prob, k: np.ndarray) -> np.ndarray:
    """Phase ramp (cycles, reduced mod 1) that places output bin 0 exactly at f_min: FFT index m of the
    series sampled at (k - K_m) dt is frequency f_het + m df, so Fa(f_min + q df) = sum_k Ya_k
    exp(-2 pi i [(f_min - f_het) dt k + q k / n_fft])  ("Fa(f - f_h)"; S13).  When
    (f_min - f_het)/df is an integer s this is the index shift q -> (q + s) mod n_fft of the plain FFT."""
    x = (prob.f_min - prob.f_het) * prob.dt * np.asarray(k, dtype=np.float64)
    return x - np.floor(x)


def validate(prob) -> None:
    """The size rules of include/fstat.h (FSTAT_ESIZE / FSTAT_EINVAL)."""
    n_src = prob.n_samples + 2 * k_margin(prob)
    if prob.n_fft & (prob.n_fft - 1) or n_src > prob.n_fft:
        raise ValueError("n_fft must be a power of two >= n_samples + 2*ceil(512 s/dt)")
    if prob.band > 1.0 / prob.dt * (1 + 1e-12):
        raise ValueError("band wider than the sample rate")


def fstat_FaFb(prob, template, sky: Optional[dict] = None):
    validate(prob)
    alpha, delta, f0, fdot, fddot = [float(v) for v in template]
    if abs(f0 - prob.f_min) > 1e-9 * max(1.0, abs(prob.f_min)):
        raise ValueError("template f0 must equal the plan's f_min")
    if sky is None:
        sky = per_sky(prob, alpha, delta)
    n_src = prob.n_samples + 2 * k_margin(prob)
    Ya = np.zeros(prob.n_fft, dtype=np.complex128)
    Yb = np.zeros(prob.n_fft, dtype=np.complex128)
    for X in range(prob.n_det):
        s = sky["det"][X]
        tau = s["tau"]                                # tau_k - tau_ref, tau_ref = t_start (S9)
        p1 = prob.f_het * s["Delta"]                  # step (iii), sign per G3
        p2 = 0.5 * fdot * tau ** 2 + fddot * tau ** 3 / 6.0
        cyc = (p1 - np.floor(p1)) + (p2 - np.floor(p2))
        y = s["z"] * np.exp(-2j * math.pi * cyc)
        Ya[:n_src] += s["wk"] * s["a"] * y
        Yb[:n_src] += s["wk"] * s["b"] * y
    ramp = np.exp(-2j * math.pi * band_shift_cycles(prob, np.arange(n_src)))     # step 7: bin 0 at f_min (S13)
    Ya[:n_src] *= ramp
    Yb[:n_src] *= ramp
    Fa = np.fft.fft(Ya)
    Fb = np.fft.fft(Yb)
    return Fa[:prob.n_bins], Fb[:prob.n_bins], sky["ABCD"]


def twoF_from_FaFb(Fa, Fb, A, B, C, D):
    """eq. 8 with weights already carrying 1/sigma^2 (G5)."""
    return (B * np.abs(Fa) ** 2 + A * np.abs(Fb) ** 2 - 2.0 * C * np.real(Fa * np.conj(Fb))) / D


def fstat_2F(prob, template, sky: Optional[dict] = None) -> np.ndarray:
    Fa, Fb, (A, B, C, D) = fstat_FaFb(prob, template, sky)
    if not D > 0.0:
        raise ValueError("D <= 0")
    return twoF_from_FaFb(Fa, Fb, A, B, C, D)


def fstat_2F_bank(prob, template_indices=None) -> np.ndarray:
    """2F[len(indices)][n_bins] for the problem's template bank; per-sky work is
    memoised across consecutive templates that share (alpha, delta)."""
    idxs = range(len(prob.templates)) if template_indices is None else template_indices
    out = np.empty((len(idxs), prob.n_bins))
    cache_key, cache = None, None
    for r, i in enumerate(idxs):
        t = prob.templates[i]
        key = (float(t[0]), float(t[1]))
        if key != cache_key:
            cache_key, cache = key, per_sky(prob, key[0], key[1])
        out[r] = fstat_2F(prob, t, cache)
    return out


# ---------------------------------------------------------------------------
# Single-detector statistic and the semi-coherent sum over segments
# ---------------------------------------------------------------------------
def single_detector_view(prob, X: int):
    """The same problem restricted to detector X (a shallow copy with one-element lists)."""
    import copy
    q = copy.copy(prob)
    q.detectors = [prob.detectors[X]]
    q.series = [prob.series[X]]
    q.timestamps = [prob.timestamps[X]]
    q.weights = [prob.weights[X]]
    return q


def fstat_2F_per_detector(prob, template) -> np.ndarray:
    """2F_X[n_det][n_bins]: eq. 8 with every sum over detector X only -- the per-detector
    quantity the paper's accuracy tooling compares.  By definition: the whole path on the
    one-detector problem."""
    return np.stack([fstat_2F(single_detector_view(prob, X), template) for X in range(prob.n_det)])


def fstat_2F_semicoherent(probs, templates, bin_offsets=None) -> np.ndarray:
    """Semi-coherent statistic (section 6: "each segment is searched using the F-statistic, and
    results from all segments are summed"): out[q] = sum_s 2F_s[q + off_s], where segment s has its own problem
    (data, t_start = its reference time), its own template (the signal's parameters at that reference time) and a
    bin offset off_s (the signal's frequency drift since the search's reference time, in bins; default 0).
    Bins that fall outside a segment's band add nothing."""
    n_bins = probs[0].n_bins
    out = np.zeros(n_bins)
    for s, (prob, tmpl) in enumerate(zip(probs, templates)):
        assert prob.n_bins == n_bins
        row = fstat_2F(prob, tmpl)
        off = 0 if bin_offsets is None else int(bin_offsets[s])
        q = np.arange(n_bins)
        src = q + off
        ok = (src >= 0) & (src < n_bins)
        out[ok] += row[src[ok]]
    return out


def chi2_sf(x, dof: int):
    """Pr(chi^2_dof > x) for even dof: e^{-x/2} sum_{j < dof/2} (x/2)^j / j!  (dof = 4: chi2_4_sf)."""
    assert dof % 2 == 0 and dof > 0
    x = np.asarray(x, dtype=np.float64)
    term = np.ones_like(x)
    acc = np.ones_like(x)
    for j in range(1, dof // 2):
        term = term * (0.5 * x) / j
        acc = acc + term
    return np.exp(-0.5 * x) * acc


# ---------------------------------------------------------------------------
# Figure 1's code listing, restated.
# ---------------------------------------------------------------------------
def twoF_fig1(Fa, Fb, Ahat, Bhat, Chat, Ehat, Dinv):
    return 2.0 * Dinv * (Bhat * (Fa.real ** 2 + Fa.imag ** 2) + Ahat * (Fb.real ** 2 + Fb.imag ** 2)
                         - 2.0 * Chat * (Fa.real * Fb.real + Fa.imag * Fb.imag)
                         - 2.0 * Ehat * (-Fa.real * Fb.imag + Fa.imag * Fb.real))


# ---------------------------------------------------------------------------
# Brute-force detector-frame sum: eq. 4-5 discretised, no
# resampling and no FFT.  Exact definition; agrees with the method only within
# the method's own (interpolation, dt/dt_b ~ 1) error.
# ---------------------------------------------------------------------------
def direct_sum_2F(prob, template, bins: np.ndarray) -> np.ndarray:
    alpha, delta, f0, fdot, fddot = [float(v) for v in template]
    A, B, C, D = antenna_sums(prob, alpha, delta)
    tp = np.arange(prob.n_samples, dtype=np.float64) * prob.dt
    bins = np.asarray(bins, dtype=np.int64)
    foff = (prob.f_min - prob.f_het) + bins * prob.df          # f - f_het per requested bin
    Fa = np.zeros(len(bins), dtype=np.complex128)
    Fb = np.zeros(len(bins), dtype=np.complex128)
    for X, det in enumerate(prob.detectors):
        w = slot_weights(prob, X)
        ws = w[np.minimum(np.floor(tp / prob.t_sft).astype(np.int64), len(w) - 1)]
        Delta = ssb_delay(det, prob.ephem, alpha, delta, tp)
        tau = tp + Delta
        a, b = antenna_ab(det, prob.ephem, alpha, delta, tp)
        x = prob.series[X].astype(np.complex128)
        base = prob.f_het * Delta + 0.5 * fdot * tau ** 2 + fddot * tau ** 3 / 6.0
        rot = np.exp(-2j * math.pi * (base - np.floor(base)))
        xa = ws * x * a * rot
        xb = ws * x * b * rot
        for i, fo in enumerate(foff):
            ph = fo * tau
            e = np.exp(-2j * math.pi * (ph - np.floor(ph)))
            Fa[i] += np.sum(xa * e)
            Fb[i] += np.sum(xb * e)
    return twoF_from_FaFb(Fa, Fb, A, B, C, D)


# ---------------------------------------------------------------------------
# Post-processing: chi^2_4 tail, top-k (S15)
# ---------------------------------------------------------------------------
def chi2_4_sf(x):
    """Pr(2F > x) for a chi-squared variable with 4 degrees of freedom."""
    x = np.asarray(x, dtype=np.float64)
    return np.exp(-0.5 * x) * (1.0 + 0.5 * x)


def topk(twoF_row: np.ndarray, k: int):
    """k largest values, descending; ties -> lower bin index first."""
    order = np.lexsort((np.arange(len(twoF_row)), -twoF_row))[:k]
    return twoF_row[order], order.astype(np.int32)


def threshold_candidates(twoF_row: np.ndarray, threshold: float, k: int):
    """Candidate retention of PAPER.md:307: the (at most k) loudest bins with 2F > threshold, ordered like topk(),
    and the number of bins above the threshold."""
    above = np.nonzero(twoF_row > threshold)[0]
    order = above[np.lexsort((above, -twoF_row[above]))][:k]
    return twoF_row[order], order.astype(np.int32), int(len(above))


def comparison_metrics(x: np.ndarray, y: np.ndarray):
    """The paper's vector comparison metrics: relative errors
    r_p(x, y) = 2 ||x - y||_p / (||x||_p + ||y||_p) for p = 1, 2 (eq. 9) and the angle
    theta = arccos( Re(x^* . y) / (||x||_2 ||y||_2) ) (eq. 10), for real or complex vectors."""
    x = np.asarray(x).ravel()
    y = np.asarray(y).ravel()
    r1 = 2.0 * np.sum(np.abs(x - y)) / (np.sum(np.abs(x)) + np.sum(np.abs(y)))
    r2 = 2.0 * np.linalg.norm(x - y) / (np.linalg.norm(x) + np.linalg.norm(y))
    c = np.real(np.vdot(x, y)) / (np.linalg.norm(x) * np.linalg.norm(y))
    return float(r1), float(r2), math.acos(min(1.0, max(-1.0, c)))
