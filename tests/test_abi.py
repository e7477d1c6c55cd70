"""CPU-side checks of the boundary: the C-ABI library builds, loads without a GPU and
exports every symbol include/fstat.h declares; argument validation that needs no device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2201_00451_b200 import binding, build, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    syms = set()
    for h in ("fstat.h", "fstat_debug.h"):
        text = open(os.path.join(ROOT, "include", h)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        syms |= set(re.findall(r"\b(fstat_[a-z_]+)\s*\(", text))
    return sorted(syms)


def test_library_builds_loads_and_exports_header_symbols():
    build.build_library()
    lib = C.CDLL(build.LIB_PATH)
    syms = _declared_symbols()
    assert set(syms) == set(binding.EXPORTS), (syms, binding.EXPORTS)
    for s in syms:
        assert hasattr(lib, s), s


def test_strerror_and_codes():
    lib = binding.load_library()
    assert lib.fstat_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -5):
        assert len(lib.fstat_strerror(code)) > 0


def _setup_raw(lib, prob, **over):
    n_det = prob.n_det
    dets = (binding.Detector * n_det)(*[binding.Detector(d["lat_rad"], d["lon_east_rad"], d["xarm_azimuth_rad"]) for d in prob.detectors])
    eph = binding.Ephem(**{k: prob.ephem[k] for k, _ in binding.Ephem._fields_})
    ser = [np.ascontiguousarray(x) for x in prob.series]
    ts = [np.ascontiguousarray(over.get("timestamps", prob.timestamps)[X], dtype=np.float64) for X in range(n_det)]
    ws = [np.ascontiguousarray(w, dtype=np.float32) for w in prob.weights]
    sptr = (C.c_void_p * n_det)(*[x.ctypes.data for x in ser])
    tptr = (C.c_void_p * n_det)(*[t.ctypes.data for t in ts])
    wptr = (C.c_void_p * n_det)(*[w.ctypes.data for w in ws])
    nseg = (C.c_int32 * n_det)(*[len(t) for t in ts])
    h = C.c_void_p()
    rc = lib.fstat_setup(C.byref(h), n_det, dets, sptr, prob.n_samples, prob.t_start, prob.dt, prob.f_het, tptr, wptr, nseg,
                         prob.t_sft, C.byref(eph), over.get("dterms", prob.dterms), prob.f_min, over.get("band", prob.band),
                         over.get("n_fft", prob.n_fft), None)
    return rc, h


def test_setup_argument_validation_without_gpu():
    """Validation runs before any CUDA call, so these codes are observable on a CPU box."""
    lib = binding.load_library()
    p = synth.small_problem(n_samples=5000, n_fft=1 << 13, rho=None)
    assert _setup_raw(lib, p, n_fft=(1 << 13) + 2)[0] == binding.FSTAT_ESIZE          # not a power of two
    assert _setup_raw(lib, p, n_fft=1 << 12)[0] == binding.FSTAT_ESIZE                # n_samples + 2 K_m > n_fft
    assert _setup_raw(lib, p, band=1.5 / p.dt)[0] == binding.FSTAT_ESIZE              # band > sample rate
    assert _setup_raw(lib, p, dterms=0)[0] == binding.FSTAT_ESIZE
    assert _setup_raw(lib, p, dterms=33)[0] == binding.FSTAT_ESIZE
    bad = [t.copy() for t in p.timestamps]
    bad[0][0] += 7.0                                                                   # off the slot grid
    assert _setup_raw(lib, p, timestamps=bad)[0] == binding.FSTAT_EINVAL
    bad = [t[::-1].copy() for t in p.timestamps]                                       # unsorted
    assert _setup_raw(lib, p, timestamps=bad)[0] == binding.FSTAT_EINVAL
    assert len(lib.fstat_last_error(None)) > 0


def test_oracle_validate_and_fstat_setup_reject_the_same_sizes():
    """Pin of `O.validate` (the oracle's only function without one): it raises on exactly the size rules of the method that
    fstat_setup answers with FSTAT_ESIZE -- n_fft a power of two, n_samples + 2 ceil(512 s/dt) <= n_fft (the zero-padded
    transform must hold the resampled series, S7), band <= 1/dt -- and accepts what fstat_setup
    accepts, on both sides of every boundary.  (Dterms outside [1, 32] is a limit of the CUDA library only: the oracle's
    windowed sinc is defined for any D.)"""
    import copy
    from oracle import fstat_oracle as O
    lib = binding.load_library()
    p = synth.small_problem(n_samples=5000, n_fft=1 << 13, rho=None)
    km2 = 2 * O.k_margin(p)

    def both(**over):
        q = copy.copy(p)
        for k, v in over.items():
            setattr(q, k, v)
        try:
            O.validate(q)
            oracle_ok = True
        except ValueError:
            oracle_ok = False
        rc, h = _setup_raw(lib, p, **over)
        if rc == binding.FSTAT_OK:
            lib.fstat_destroy(h)
        lib_ok = rc != binding.FSTAT_ESIZE               # valid sizes end in FSTAT_OK (GPU box) or FSTAT_ECUDA (no device)
        assert rc in (binding.FSTAT_OK, binding.FSTAT_ECUDA, binding.FSTAT_ESIZE), rc
        assert oracle_ok == lib_ok, (over, oracle_ok, rc)
        return oracle_ok

    assert both() is True
    assert both(n_fft=(1 << 13) + 2) is False                       # not a power of two
    assert both(n_fft=1 << 12) is False                             # 5000 + 1024 > 4096
    assert both(n_fft=1 << 14) is True
    assert both(band=1.5 / p.dt) is False                           # wider than the sample rate
    assert both(band=1.0 / p.dt) is True                            # exactly the sample rate: every FFT output is a bin
    # the boundary of the padding rule, on a series cut to fit / not to fit exactly
    for n_samples, ok in (((1 << 13) - km2, True), ((1 << 13) - km2 + 1, False)):
        q = synth.small_problem(n_samples=n_samples, n_fft=1 << 13, rho=None)
        try:
            O.validate(q)
            oracle_ok = True
        except ValueError:
            oracle_ok = False
        rc, h = _setup_raw(lib, q)
        if rc == binding.FSTAT_OK:
            lib.fstat_destroy(h)
        assert oracle_ok == ok and (rc != binding.FSTAT_ESIZE) == ok, (n_samples, oracle_ok, rc)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    lib = binding.load_library()
    p = synth.small_problem(n_samples=5000, n_fft=1 << 13, rho=None)
    rc, _ = _setup_raw(lib, p)
    assert rc == binding.FSTAT_ECUDA                      # valid arguments, but no device: fails loudly
    with pytest.raises(RuntimeError):
        binding.FstatPlan(p)
