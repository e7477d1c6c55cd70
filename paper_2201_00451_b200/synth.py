"""Seeded synthetic inputs for the resampling F-statistic hot path.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2201_00451_b200/csrc`).  It produces the *inputs* -- detector
geometry, the heterodyned complex64 series x_h(t^k) of PAPER.md:80 (step ii),
segment timestamps / noise weights and the template bank -- and none of the
method's arithmetic (no resampling, no FFT, no 2F).

The injected signal needs the detector response and the SSB delay.  They are
written here *geometrically* (detector tensor contracted with polarisation
tensors; dot product of position vectors), on purpose different from the
closed trigonometric forms the oracle and the kernels use, so that the
noise-free pin "2F == rho^2" (pin P2) also cross-checks those
formulas instead of sharing them.

The configs stand in for the paper's Makefakedata_v4 Gaussian-noise study
 and for the shape of its O2 pilot search;
no LIGO data and no LALSuite output is used or reproduced.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Sequence

import numpy as np

DEG = math.pi / 180.0

# Analytic ephemeris constants (reading S3; all are plan inputs).
EPHEM_DEFAULT = dict(
    au_over_c_s=499.004783836,
    omega_orb=2.0 * math.pi / (365.256363004 * 86400.0),
    phi_orb0=0.0,
    obliquity_rad=23.4392911 * DEG,
    re_over_c_s=6378137.0 / 299792458.0,
    omega_rot=2.0 * math.pi / 86164.0905,
    gmst0_rad=0.0,
)

H1 = dict(lat_rad=46.455 * DEG, lon_east_rad=-119.408 * DEG, xarm_azimuth_rad=36.0 * DEG)
L1 = dict(lat_rad=30.563 * DEG, lon_east_rad=-90.774 * DEG, xarm_azimuth_rad=108.0 * DEG)

V1 = dict(lat_rad=43.631 * DEG, lon_east_rad=10.504 * DEG, xarm_azimuth_rad=341.0 * DEG)   # a third, Virgo-like site (tests)

T_SFT = 1800.0
T_START = 1.0e9  # arbitrary epoch; every formula uses t' = t - t_start


@dataclasses.dataclass
class Injection:
    rho: float
    cosi: float
    psi: float
    phi0: float
    f: float
    fdot: float
    fddot: float
    alpha: float
    delta: float


@dataclasses.dataclass
class Problem:
    """Everything `fstat_setup` needs, plus the template bank."""
    name: str
    detectors: List[dict]
    ephem: dict
    series: List[np.ndarray]          # per detector complex64[n_samples]
    n_samples: int
    t_start: float
    dt: float
    f_het: float
    timestamps: List[np.ndarray]      # per detector float64[n_seg]: start of each listed slot
    weights: List[np.ndarray]         # per detector float32[n_seg]: 1/sigma_c^2 of that slot
    t_sft: float
    dterms: int
    f_min: float
    band: float
    n_fft: int
    templates: np.ndarray             # float64[n_tmpl,5]: alpha, delta, f0, fdot, fddot
    injection: Optional[Injection] = None
    injection_template: Optional[int] = None
    seed: int = 0

    @property
    def n_det(self) -> int:
        return len(self.detectors)

    @property
    def n_bins(self) -> int:
        return int(round(self.band * self.n_fft * self.dt))

    @property
    def df(self) -> float:
        return 1.0 / (self.n_fft * self.dt)


# --------------------------------------------------------------------------
# Geometry used only for the injection (vector / tensor form)
# --------------------------------------------------------------------------
def _sky_vector(alpha: float, delta: float) -> np.ndarray:
    return np.array([math.cos(delta) * math.cos(alpha),
                     math.cos(delta) * math.sin(alpha),
                     math.sin(delta)])


def _earth_frames(det: dict, eph: dict, tp: np.ndarray):
    """Unit vectors (zenith, east, north) of the site in the equatorial frame."""
    th = eph["gmst0_rad"] + eph["omega_rot"] * tp + det["lon_east_rad"]
    lat = det["lat_rad"]
    c, s = np.cos(th), np.sin(th)
    zen = np.stack([math.cos(lat) * c, math.cos(lat) * s, np.full_like(tp, math.sin(lat))])
    east = np.stack([-s, c, np.zeros_like(tp)])
    north = np.stack([-math.sin(lat) * c, -math.sin(lat) * s, np.full_like(tp, math.cos(lat))])
    return zen, east, north


def geometric_delay(det: dict, eph: dict, alpha: float, delta: float, tp: np.ndarray) -> np.ndarray:
    """Roemer delay n.(r_orbit + r_site)/c at detector time t' (seconds)."""
    n = _sky_vector(alpha, delta)
    ph = eph["phi_orb0"] + eph["omega_orb"] * tp
    eps = eph["obliquity_rad"]
    r_orb = eph["au_over_c_s"] * np.stack([np.cos(ph), np.sin(ph) * math.cos(eps), np.sin(ph) * math.sin(eps)])
    zen, _, _ = _earth_frames(det, eph, tp)
    r_site = eph["re_over_c_s"] * zen
    return n @ (r_orb + r_site)


def geometric_antenna(det: dict, eph: dict, alpha: float, delta: float, tp: np.ndarray):
    """a(t), b(t) as contractions of the detector tensor d = (uu - vv)/2 with the
    polarisation basis of the wave frame (xi, eta)."""
    _, east, north = _earth_frames(det, eph, tp)
    az = det["xarm_azimuth_rad"]  # x-arm, counter-clockwise from local North
    u = math.cos(az) * north - math.sin(az) * east
    v = -math.sin(az) * north - math.cos(az) * east   # y-arm, 90 deg further CCW
    xi = np.array([math.sin(alpha), -math.cos(alpha), 0.0])
    eta = np.array([-math.sin(delta) * math.cos(alpha), -math.sin(delta) * math.sin(alpha), math.cos(delta)])
    uxi, ueta, vxi, veta = xi @ u, eta @ u, xi @ v, eta @ v
    a = 0.5 * ((uxi * uxi - vxi * vxi) - (ueta * ueta - veta * veta))
    b = 0.5 * 2.0 * (uxi * ueta - vxi * veta)
    return a, b


def _jks_amplitudes(h0: float, cosi: float, psi: float, phi0: float):
    ap = 0.5 * h0 * (1.0 + cosi * cosi)
    ax = h0 * cosi
    c2, s2 = math.cos(2 * psi), math.sin(2 * psi)
    cp, sp = math.cos(phi0), math.sin(phi0)
    a1 = ap * cp * c2 - ax * sp * s2
    a2 = ap * cp * s2 + ax * sp * c2
    a3 = -ap * sp * c2 - ax * cp * s2
    a4 = -ap * sp * s2 + ax * cp * c2
    return a1, a2, a3, a4


# --------------------------------------------------------------------------
# Series generator
# --------------------------------------------------------------------------
def make_problem(name: str, detectors: Sequence[dict], n_samples: int, dt: float,
                 f_min: float, band: float, f_het: float, n_fft: int, dterms: int,
                 templates: np.ndarray, seed: int, gap_frac: float = 0.0,
                 weight_range: Optional[Sequence[float]] = None,
                 injection: Optional[Injection] = None, injection_template: Optional[int] = None,
                 noise: bool = True, ephem: Optional[dict] = None,
                 snap_injection_to_bin: bool = False) -> Problem:
    eph = dict(EPHEM_DEFAULT if ephem is None else ephem)
    rng = np.random.default_rng(seed)
    n_slots = int(math.ceil(n_samples * dt / T_SFT - 1e-9))
    tp = np.arange(n_samples, dtype=np.float64) * dt
    slot_of = np.minimum((tp / T_SFT).astype(np.int64), n_slots - 1)

    series, stamps, weights, slotw = [], [], [], []
    for _ in detectors:
        w = np.ones(n_slots) if weight_range is None else rng.uniform(weight_range[0], weight_range[1], n_slots)
        keep = np.ones(n_slots, dtype=bool)
        n_gap = int(round(gap_frac * n_slots))
        if n_gap > 0:
            keep[rng.choice(n_slots, size=n_gap, replace=False)] = False
        wfull = np.where(keep, w, 0.0)
        slotw.append(wfull)
        stamps.append(T_START + T_SFT * np.nonzero(keep)[0].astype(np.float64))
        weights.append(w[keep].astype(np.float32))
        if noise:
            x = (rng.standard_normal(n_samples) + 1j * rng.standard_normal(n_samples))
            x /= np.sqrt(np.where(keep, w, 1.0))[slot_of]
        else:
            x = np.zeros(n_samples, dtype=np.complex128)
        series.append(x)

    inj = injection
    if inj is not None:
        if snap_injection_to_bin:
            df = 1.0 / (n_fft * dt)
            inj = dataclasses.replace(inj, f=f_min + round((inj.f - f_min) / df) * df)
        # weights seen by the statistic are the float32 values handed to fstat_setup
        a1, a2, a3, a4 = _jks_amplitudes(1.0, inj.cosi, inj.psi, inj.phi0)
        amp_a, amp_b = complex(a1, -a3), complex(a2, -a4)
        A = B = C = 0.0
        resp = []
        for X, det in enumerate(detectors):
            a, b = geometric_antenna(det, eph, inj.alpha, inj.delta, tp)
            w32 = np.zeros(n_slots)
            w32[np.nonzero(slotw[X])[0]] = weights[X].astype(np.float64)
            ws = w32[slot_of]
            A += float(np.sum(ws * a * a)); B += float(np.sum(ws * b * b)); C += float(np.sum(ws * a * b))
            resp.append((a, b))
        rho2_unit = A * abs(amp_a) ** 2 + B * abs(amp_b) ** 2 + 2.0 * C * (amp_a * amp_b.conjugate()).real
        scale = inj.rho / math.sqrt(rho2_unit)
        for X, det in enumerate(detectors):
            a, b = resp[X]
            tau = tp + geometric_delay(det, eph, inj.alpha, inj.delta, tp)   # SSB time - t_start
            cyc = np.mod(inj.f * tau, 1.0) + 0.5 * inj.fdot * tau * tau + inj.fddot * tau ** 3 / 6.0 \
                - np.mod(f_het * tp, 1.0)
            cyc -= np.floor(cyc)
            series[X] = series[X] + scale * (amp_a * a + amp_b * b) * np.exp(2j * math.pi * cyc)

    out = []
    for X in range(len(detectors)):
        x = series[X]
        x[slotw[X][slot_of] == 0.0] = 0.0
        out.append(np.ascontiguousarray(x.astype(np.complex64)))

    return Problem(name=name, detectors=[dict(d) for d in detectors], ephem=eph, series=out,
                   n_samples=n_samples, t_start=T_START, dt=dt, f_het=f_het,
                   timestamps=stamps, weights=weights, t_sft=T_SFT, dterms=dterms,
                   f_min=f_min, band=band, n_fft=n_fft,
                   templates=np.ascontiguousarray(templates, dtype=np.float64),
                   injection=inj, injection_template=injection_template, seed=seed)


def _fdot_bank(alpha, delta, f0, fdots, fddots=(0.0,)):
    """Template bank, fddot-major (outer) / fdot-minor (inner)."""
    rows = [(alpha, delta, f0, fd, fdd) for fdd in fddots for fd in fdots]
    return np.array(rows, dtype=np.float64)


def next_pow2(n: int) -> int:
    p = 1
    while p < n:
        p *= 2
    return p


SKY0 = (3.52, -0.83)


# --------------------------------------------------------------------------
# The five BASELINE.json configs and small variants
# --------------------------------------------------------------------------
def config1(n_templates: int = 16) -> Problem:
    inj = Injection(rho=20.0, cosi=0.3, psi=0.4, phi0=1.0, f=100.2, fdot=-1e-10, fddot=0.0,
                    alpha=SKY0[0], delta=SKY0[1])
    tm = _fdot_bank(SKY0[0], SKY0[1], 100.0, np.linspace(-2e-10, 2e-10, n_templates))
    return make_problem("config1", [H1], 86400, 1.0, 100.0, 0.5, 100.25, 1 << 18, 8, tm, seed=0, injection=inj)


def config2(n_templates: int = 1024, days: float = 10.0) -> Problem:
    fdots = np.linspace(-1e-9, 0.0, n_templates)
    it = min(300, n_templates - 1)
    inj = Injection(rho=15.0, cosi=0.3, psi=0.4, phi0=1.0, f=200.37, fdot=float(fdots[it]), fddot=0.0,
                    alpha=SKY0[0], delta=SKY0[1])
    n = int(round(days * 86400 * 2))
    tm = _fdot_bank(SKY0[0], SKY0[1], 200.0, fdots)
    kpad = 2 * int(math.ceil(512.0 / 0.5))
    return make_problem("config2", [H1, L1], n, 0.5, 200.0, 1.0, 200.5, next_pow2(n + kpad), 8, tm, seed=1,
                        gap_frac=0.30, weight_range=(0.5, 2.0), injection=inj, injection_template=it,
                        snap_injection_to_bin=True)


CONFIG3_DAYS = (1, 2, 5, 10, 20)
CONFIG3_BANDS = (0.1, 0.5, 1.0, 2.0)


def config3(days: float, band: float, n_templates: int = 256) -> Problem:
    cell = CONFIG3_DAYS.index(days) * len(CONFIG3_BANDS) + CONFIG3_BANDS.index(band) \
        if days in CONFIG3_DAYS and band in CONFIG3_BANDS else 99
    fs = 2.0 * band
    dt = 1.0 / fs
    n = int(round(days * 86400 * fs))
    kpad = 2 * int(math.ceil(512.0 / dt))
    tm = _fdot_bank(SKY0[0], SKY0[1], 150.0, np.linspace(-1e-9, 0.0, n_templates))
    return make_problem(f"config3_T{days}d_B{band}", [H1, L1], n, dt, 150.0, band, 150.0 + band / 2,
                        next_pow2(n + kpad), 8, tm, seed=100 + cell, gap_frac=0.5)


CONFIG4_TARGETS = (320.0, 480.0, 550.0, 680.0)


def config4(target: int, n_fdot: int = 4096, n_fddot: int = 4, days: float = 10.0) -> Problem:
    F = CONFIG4_TARGETS[target]
    fdots = np.linspace(-5e-9, 5e-9, n_fdot)
    fddots = np.linspace(-1e-17, 2e-17, n_fddot)
    tm = _fdot_bank(SKY0[0], SKY0[1], F - 1.0, fdots, fddots)
    inj, it = None, None
    if target in (0, 2):
        i_fd, i_fdd = (n_fdot * 3) // 8, min(1, n_fddot - 1)
        it = i_fdd * n_fdot + i_fd
        inj = Injection(rho=8.0 if target == 0 else 12.0, cosi=0.3, psi=0.4, phi0=1.0,
                        f=F - 0.23, fdot=float(fdots[i_fd]), fddot=float(fddots[i_fdd]),
                        alpha=SKY0[0], delta=SKY0[1])
    n = int(round(days * 86400 * 2))
    kpad = 2 * int(math.ceil(512.0 / 0.5))
    return make_problem(f"config4_target{target}", [H1, L1], n, 0.5, F - 1.0, 2.0, F,
                        max(next_pow2(n + kpad), 1 << 22) if days == 10.0 else next_pow2(n + kpad),
                        8, tm, seed=200 + target, gap_frac=0.40, injection=inj,
                        injection_template=it, snap_injection_to_bin=True)


def disc_sky_points(n_sky: int, seed: int, centre=SKY0, radius: float = 0.05) -> np.ndarray:
    """n_sky points uniform in solid angle within `radius` of `centre`."""
    rng = np.random.default_rng(seed)
    cosr = 1.0 - rng.uniform(0.0, 1.0, n_sky) * (1.0 - math.cos(radius))
    r = np.arccos(cosr)
    phi = rng.uniform(0.0, 2.0 * math.pi, n_sky)
    a0, d0 = centre
    n0 = _sky_vector(a0, d0)
    e1 = np.array([-math.sin(a0), math.cos(a0), 0.0])
    e2 = np.cross(n0, e1)
    v = (np.cos(r)[:, None] * n0 + np.sin(r)[:, None] * (np.cos(phi)[:, None] * e1 + np.sin(phi)[:, None] * e2))
    alpha = np.mod(np.arctan2(v[:, 1], v[:, 0]), 2.0 * math.pi)
    delta = np.arcsin(np.clip(v[:, 2], -1.0, 1.0))
    return np.stack([alpha, delta], axis=1)


def config5(n_sky: int = 4096, n_fdot: int = 4, days: float = 2.0) -> Problem:
    sky = disc_sky_points(n_sky, seed=300)
    fdots = np.linspace(-1e-9, 0.0, n_fdot)
    rows = [(a, d, 300.0, fd, 0.0) for (a, d) in sky for fd in fdots]   # sky-major, fdot inner
    tm = np.array(rows, dtype=np.float64)
    i_sky, i_fd = min(1234, n_sky - 1), min(2, n_fdot - 1)
    it = i_sky * n_fdot + i_fd
    inj = Injection(rho=10.0, cosi=0.3, psi=0.4, phi0=1.0, f=300.21, fdot=float(fdots[i_fd]), fddot=0.0,
                    alpha=float(sky[i_sky, 0]), delta=float(sky[i_sky, 1]))
    n = int(round(days * 86400))
    kpad = 2 * 512
    return make_problem("config5", [H1, L1], n, 1.0, 300.0, 0.5, 300.25, next_pow2(n + kpad), 16, tm,
                        seed=300, injection=inj, injection_template=it, snap_injection_to_bin=True)


def small_problem(seed: int = 7, n_det: int = 2, n_samples: int = 20000, dt: float = 1.0,
                  n_fft: int = 1 << 15, dterms: int = 8, n_templates: int = 4, gap_frac: float = 0.3,
                  weights: bool = True, rho: Optional[float] = 12.0, noise: bool = True,
                  f_min: float = 120.0, band: Optional[float] = None, fddot: float = 0.0,
                  ephem: Optional[dict] = None, f_het: Optional[float] = None) -> Problem:
    """A seconds-scale problem with the structure of config 2 (ragged length,
    gaps, weights, two detectors) used by the parity tests and smoke()."""
    band = 0.5 / dt if band is None else band
    fdots = np.linspace(-8e-9, 0.0, n_templates)
    it = n_templates // 2
    inj = None
    if rho is not None:
        inj = Injection(rho=rho, cosi=-0.4, psi=1.1, phi0=2.0, f=f_min + 0.31 * band, fdot=float(fdots[it]),
                        fddot=fddot, alpha=SKY0[0], delta=SKY0[1])
    tm = _fdot_bank(SKY0[0], SKY0[1], f_min, fdots, (fddot,))
    dets = [H1, L1, V1][:n_det]
    return make_problem(f"small_s{seed}", dets, n_samples, dt, f_min, band, f_min + band / 2 if f_het is None else f_het, n_fft, dterms, tm,
                        seed=seed, gap_frac=gap_frac, weight_range=(0.5, 2.0) if weights else None,
                        injection=inj, injection_template=it if inj else None, noise=noise, ephem=ephem,
                        snap_injection_to_bin=True)
