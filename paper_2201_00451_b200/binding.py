"""Thin Python binding over the C ABI of include/fstat.h.

Argument marshalling only: every step of the path runs in the CUDA kernels behind
`libfstat_b200.so`.  torch is used for device memory and streams (tensor.data_ptr(),
torch.cuda.current_stream().cuda_stream) and nothing else.  There is no fallback:
if the library is missing or no GPU is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence, Tuple

import numpy as np

from . import build as _build

FSTAT_OK, FSTAT_EINVAL, FSTAT_ESIZE, FSTAT_EDOM, FSTAT_ECUDA, FSTAT_ENOMEM = 0, -1, -2, -3, -4, -5

EXPORTS = [
    "fstat_setup", "fstat_get_layout", "fstat_compute", "fstat_compute_topk", "fstat_compute_threshold", "fstat_compute_host",
    "fstat_compute_topk_host", "fstat_compute_accumulate", "fstat_compute_per_detector", "fstat_select_topk",
    "fstat_select_threshold", "fstat_select_topk_noalloc", "fstat_resample_sky", "fstat_sync", "fstat_destroy", "fstat_strerror", "fstat_last_error",
    # include/fstat_debug.h: measurement / experiment hooks
    "fstat_launch_count", "fstat_set_inflight", "fstat_set_profile", "fstat_get_profile",
    "fstat_debug_set_geometry", "fstat_debug_set_max_sky_slots", "fstat_debug_set_paths", "fstat_debug_compute_fafb",
]


class Detector(C.Structure):
    _fields_ = [("lat_rad", C.c_double), ("lon_east_rad", C.c_double), ("xarm_azimuth_rad", C.c_double)]


class Ephem(C.Structure):
    _fields_ = [("au_over_c_s", C.c_double), ("omega_orb", C.c_double), ("phi_orb0", C.c_double),
                ("obliquity_rad", C.c_double), ("re_over_c_s", C.c_double), ("omega_rot", C.c_double),
                ("gmst0_rad", C.c_double)]


class FstatError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"fstat error {code}: {text}")
        self.code = code


_lib = None


def load_library(build_if_missing: bool = True) -> C.CDLL:
    """dlopen the in-tree library; build it with nvcc first if it is missing or stale."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB_PATH
    if build_if_missing and _build.is_stale():
        if _build.have_nvcc():
            _build.build_library()             # a compile error must surface, never run stale kernels silently
        elif os.path.exists(path):
            import warnings
            warnings.warn(f"{path} is older than its sources and nvcc is not available: loading the stale binary")
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not built: run `python -m paper_2201_00451_b200.build`")
    lib = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.fstat_setup.restype = C.c_int
    lib.fstat_setup.argtypes = [C.POINTER(vp), i32, C.POINTER(Detector), C.POINTER(vp), i64, dbl, dbl, dbl,
                                C.POINTER(vp), C.POINTER(vp), C.POINTER(i32), dbl, C.POINTER(Ephem),
                                i32, dbl, dbl, i64, vp]
    lib.fstat_get_layout.restype = C.c_int
    lib.fstat_get_layout.argtypes = [vp, C.POINTER(i64), C.POINTER(dbl)]
    lib.fstat_compute.restype = C.c_int
    lib.fstat_compute.argtypes = [vp, vp, i32, vp]
    lib.fstat_compute_topk.restype = C.c_int
    lib.fstat_compute_topk.argtypes = [vp, vp, i32, i32, vp, vp]
    lib.fstat_compute_threshold.restype = C.c_int
    lib.fstat_compute_threshold.argtypes = [vp, vp, i32, C.c_float, i32, vp, vp, vp]
    lib.fstat_compute_host.restype = C.c_int
    lib.fstat_compute_host.argtypes = [vp, vp, i32, vp]
    lib.fstat_compute_topk_host.restype = C.c_int
    lib.fstat_compute_topk_host.argtypes = [vp, vp, i32, i32, vp, vp]
    lib.fstat_compute_accumulate.restype = C.c_int
    lib.fstat_compute_accumulate.argtypes = [vp, vp, i32, vp, vp]
    lib.fstat_compute_per_detector.restype = C.c_int
    lib.fstat_compute_per_detector.argtypes = [vp, vp, i32, vp]
    lib.fstat_select_topk.restype = C.c_int
    lib.fstat_select_topk.argtypes = [vp, vp, i32, i32, vp, vp]
    lib.fstat_select_threshold.restype = C.c_int
    lib.fstat_select_threshold.argtypes = [vp, vp, i32, C.c_float, i32, vp, vp, vp]
    lib.fstat_select_topk_noalloc.restype = C.c_int
    lib.fstat_select_topk_noalloc.argtypes = [vp, i64, i32, i32, vp, vp, vp]
    lib.fstat_resample_sky.restype = C.c_int
    lib.fstat_resample_sky.argtypes = [vp, dbl, dbl, vp, C.POINTER(dbl)]
    lib.fstat_sync.restype = C.c_int
    lib.fstat_sync.argtypes = [vp]
    lib.fstat_launch_count.restype = C.c_int
    lib.fstat_launch_count.argtypes = [vp, C.POINTER(i64)]
    lib.fstat_set_inflight.restype = C.c_int
    lib.fstat_set_inflight.argtypes = [vp, i32]
    lib.fstat_set_profile.restype = C.c_int
    lib.fstat_set_profile.argtypes = [vp, i32]
    lib.fstat_get_profile.restype = C.c_int
    lib.fstat_get_profile.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
    lib.fstat_debug_set_geometry.restype = C.c_int
    lib.fstat_debug_set_geometry.argtypes = [vp, i32, i32, i32, i32]
    lib.fstat_debug_set_max_sky_slots.restype = C.c_int
    lib.fstat_debug_set_max_sky_slots.argtypes = [vp, i32]
    lib.fstat_debug_set_paths.restype = C.c_int
    lib.fstat_debug_set_paths.argtypes = [vp, i32, i32]
    lib.fstat_debug_compute_fafb.restype = C.c_int
    lib.fstat_debug_compute_fafb.argtypes = [vp, vp, i32, vp]
    lib.fstat_destroy.restype = None
    lib.fstat_destroy.argtypes = [vp]
    lib.fstat_strerror.restype = C.c_char_p
    lib.fstat_strerror.argtypes = [C.c_int]
    lib.fstat_last_error.restype = C.c_char_p
    lib.fstat_last_error.argtypes = [vp]
    _lib = lib
    return lib


NOALLOC_MAX_GROUPS = 262144          # FSTAT_NOALLOC_MAX_GROUPS of include/fstat.h


def select_topk_noalloc(rows, k: int, out: Tuple, stream=None):
    """fstat_select_topk_noalloc: the k loudest bins of every row of `rows` (float32[n_rows][n_bins] on the GPU), written
    into the caller's `out = (val float32[n_rows][k], bin int32[n_rows][k])` device tensors.

    For callers that cannot allocate device memory -- a pipeline whose own arena already owns the whole GPU, or a
    latency-bound loop that cannot take the device-wide stall of cudaMalloc -- so, unlike `FstatPlan.select_topk`, it
    takes no plan, creates no tensor and the library allocates nothing: the per-group maxima it needs live in a fixed
    1 MiB array inside the library.  Hence `n_rows * ceil(n_bins / 512) <= NOALLOC_MAX_GROUPS` per call (FSTAT_ESIZE
    otherwise), and calls whose GPU work overlaps race on that array: keep them on one stream.  The first call on a
    device does a one-time set-up and should come before any stream capture.  Returns `out`."""
    import torch
    val, idx = out
    assert rows.is_cuda and rows.dtype == torch.float32 and rows.is_contiguous() and rows.dim() == 2
    assert val.is_cuda and val.dtype == torch.float32 and val.is_contiguous() and tuple(val.shape) == (rows.shape[0], k)
    assert idx.is_cuda and idx.dtype == torch.int32 and idx.is_contiguous() and tuple(idx.shape) == (rows.shape[0], k)
    lib = load_library()
    s = torch.cuda.current_stream() if stream is None else stream
    rc = lib.fstat_select_topk_noalloc(rows.data_ptr(), rows.shape[1], rows.shape[0], k, val.data_ptr(), idx.data_ptr(),
                                       C.c_void_p(s.cuda_stream))
    if rc != 0:
        raise FstatError(rc, (lib.fstat_last_error(None) or lib.fstat_strerror(rc)).decode())
    return out


def _templates_array(templates) -> np.ndarray:
    t = np.ascontiguousarray(np.asarray(templates, dtype=np.float64))
    if t.ndim != 2 or t.shape[1] != 5:
        raise ValueError("templates must be [n, 5]: alpha, delta, f0, fdot, fddot")
    return t


class FstatPlan:
    """fstat_setup / fstat_compute* / fstat_destroy for one `synth.Problem`-like object."""

    def __init__(self, prob, stream=None, series_on_device: bool = False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2201_00451_b200 needs a CUDA device; there is no CPU fallback")
        self._torch = torch
        self.lib = load_library()
        self.prob = prob
        self.stream = torch.cuda.current_stream() if stream is None else stream
        n_det = prob.n_det
        dets = (Detector * n_det)(*[Detector(d["lat_rad"], d["lon_east_rad"], d["xarm_azimuth_rad"])
                                    for d in prob.detectors])
        eph = Ephem(**{k: prob.ephem[k] for k, _ in Ephem._fields_})
        keep = []
        if series_on_device:
            dev = [torch.from_numpy(x.view(np.float32)).cuda() for x in prob.series]
            keep.append(dev)
            sptr = (C.c_void_p * n_det)(*[t.data_ptr() for t in dev])
        else:
            host = [np.ascontiguousarray(x, dtype=np.complex64) for x in prob.series]
            keep.append(host)
            sptr = (C.c_void_p * n_det)(*[x.ctypes.data for x in host])
        ts = [np.ascontiguousarray(t, dtype=np.float64) for t in prob.timestamps]
        ws = [np.ascontiguousarray(w, dtype=np.float32) for w in prob.weights]
        tptr = (C.c_void_p * n_det)(*[t.ctypes.data for t in ts])
        wptr = (C.c_void_p * n_det)(*[w.ctypes.data for w in ws])
        nseg = (C.c_int32 * n_det)(*[len(t) for t in ts])
        handle = C.c_void_p()
        rc = self.lib.fstat_setup(C.byref(handle), n_det, dets, sptr, prob.n_samples, prob.t_start, prob.dt,
                                  prob.f_het, tptr, wptr, nseg, prob.t_sft, C.byref(eph), prob.dterms,
                                  prob.f_min, prob.band, prob.n_fft, C.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            raise FstatError(rc, (self.lib.fstat_last_error(None) or b"").decode())
        self.handle = handle
        nb, df = C.c_int64(), C.c_double()
        self._check(self.lib.fstat_get_layout(self.handle, C.byref(nb), C.byref(df)))
        self.n_bins, self.df = int(nb.value), float(df.value)
        self.n_fft = int(prob.n_fft)

    # -- helpers ----------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            raise FstatError(rc, (self.lib.fstat_last_error(self.handle) or self.lib.fstat_strerror(rc)).decode())

    def close(self):
        if getattr(self, "handle", None):
            self.lib.fstat_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the C-ABI calls -----------------------------------------------------------
    def compute(self, templates, out=None):
        """fstat_compute: 2F[n_tmpl][n_bins] in device memory (a torch tensor)."""
        t = _templates_array(templates)
        torch = self._torch
        if out is None:
            out = torch.empty((t.shape[0], self.n_bins), dtype=torch.float32, device="cuda")
        assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.numel() == t.shape[0] * self.n_bins
        self._check(self.lib.fstat_compute(self.handle, t.ctypes.data, t.shape[0], out.data_ptr()))
        return out

    def compute_topk(self, templates, k: int, out: Optional[Tuple] = None):
        t = _templates_array(templates)
        torch = self._torch
        if out is None:
            out = (torch.empty((t.shape[0], k), dtype=torch.float32, device="cuda"),
                   torch.empty((t.shape[0], k), dtype=torch.int32, device="cuda"))
        val, idx = out
        self._check(self.lib.fstat_compute_topk(self.handle, t.ctypes.data, t.shape[0], k, val.data_ptr(), idx.data_ptr()))
        return val, idx

    def compute_threshold(self, templates, threshold: float, k: int):
        """fstat_compute_threshold: (val[n,k], bin[n,k], count[n]) device tensors."""
        t = _templates_array(templates)
        torch = self._torch
        val = torch.empty((t.shape[0], k), dtype=torch.float32, device="cuda")
        idx = torch.empty((t.shape[0], k), dtype=torch.int32, device="cuda")
        cnt = torch.empty((t.shape[0],), dtype=torch.int32, device="cuda")
        self._check(self.lib.fstat_compute_threshold(self.handle, t.ctypes.data, t.shape[0], float(threshold), k,
                                                     val.data_ptr(), idx.data_ptr(), cnt.data_ptr()))
        return val, idx, cnt

    def compute_accumulate(self, templates, out, bin_offsets=None):
        """fstat_compute_accumulate: out[t][q - off_t] += 2F_t[q] (semi-coherent sum over segment plans)."""
        t = _templates_array(templates)
        torch = self._torch
        assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.numel() == t.shape[0] * self.n_bins
        off = None if bin_offsets is None else np.ascontiguousarray(bin_offsets, dtype=np.int32)
        assert off is None or off.shape == (t.shape[0],)
        self._check(self.lib.fstat_compute_accumulate(self.handle, t.ctypes.data, t.shape[0],
                                                      None if off is None else off.ctypes.data, out.data_ptr()))
        return out

    def compute_per_detector(self, templates, out=None):
        """fstat_compute_per_detector: 2F_X[n_det][n_tmpl][n_bins] device tensor."""
        t = _templates_array(templates)
        torch = self._torch
        if out is None:
            out = torch.empty((self.prob.n_det, t.shape[0], self.n_bins), dtype=torch.float32, device="cuda")
        assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous()
        self._check(self.lib.fstat_compute_per_detector(self.handle, t.ctypes.data, t.shape[0], out.data_ptr()))
        return out

    def select_topk(self, rows, k: int):
        torch = self._torch
        assert rows.is_cuda and rows.dtype == torch.float32 and rows.is_contiguous() and rows.shape[1] == self.n_bins
        val = torch.empty((rows.shape[0], k), dtype=torch.float32, device="cuda")
        idx = torch.empty((rows.shape[0], k), dtype=torch.int32, device="cuda")
        self._check(self.lib.fstat_select_topk(self.handle, rows.data_ptr(), rows.shape[0], k, val.data_ptr(), idx.data_ptr()))
        return val, idx

    def select_threshold(self, rows, threshold: float, k: int):
        torch = self._torch
        assert rows.is_cuda and rows.dtype == torch.float32 and rows.is_contiguous() and rows.shape[1] == self.n_bins
        val = torch.empty((rows.shape[0], k), dtype=torch.float32, device="cuda")
        idx = torch.empty((rows.shape[0], k), dtype=torch.int32, device="cuda")
        cnt = torch.empty((rows.shape[0],), dtype=torch.int32, device="cuda")
        self._check(self.lib.fstat_select_threshold(self.handle, rows.data_ptr(), rows.shape[0], float(threshold), k,
                                                    val.data_ptr(), idx.data_ptr(), cnt.data_ptr()))
        return val, idx, cnt

    def compute_host(self, templates, out=None):
        """fstat_compute_host: 2F rows land in HOST memory (pinned torch tensor by default)."""
        t = _templates_array(templates)
        torch = self._torch
        if out is None:
            out = torch.empty((t.shape[0], self.n_bins), dtype=torch.float32, pin_memory=True)
        assert (not out.is_cuda) and out.dtype == torch.float32 and out.is_contiguous()
        self._check(self.lib.fstat_compute_host(self.handle, t.ctypes.data, t.shape[0], out.data_ptr()))
        return out

    def compute_topk_host(self, templates, k: int):
        t = _templates_array(templates)
        val = np.empty((t.shape[0], k), dtype=np.float32)
        idx = np.empty((t.shape[0], k), dtype=np.int32)
        self._check(self.lib.fstat_compute_topk_host(self.handle, t.ctypes.data, t.shape[0], k, val.ctypes.data, idx.ctypes.data))
        return val, idx

    def resample_sky(self, alpha: float, delta: float):
        torch = self._torch
        S = torch.empty((self.n_fft, 4), dtype=torch.float32, device="cuda")
        abcd = (C.c_double * 4)()
        self._check(self.lib.fstat_resample_sky(self.handle, alpha, delta, S.data_ptr(), abcd))
        return S, np.array(list(abcd))

    def sync(self):
        self._check(self.lib.fstat_sync(self.handle))

    def launch_count(self) -> int:
        n = C.c_int64()
        self._check(self.lib.fstat_launch_count(self.handle, C.byref(n)))
        return int(n.value)

    PROFILE_CLASSES = ("sky", "fft_pass1", "fft_pass2", "topk", "fused_sky_pass1", "fft_single")

    def set_profile(self, enable: bool):
        self._check(self.lib.fstat_set_profile(self.handle, 1 if enable else 0))

    def get_profile(self):
        """{class: (milliseconds, launches)} since the last call."""
        ms = (C.c_double * len(self.PROFILE_CLASSES))()
        n = (C.c_int64 * len(self.PROFILE_CLASSES))()
        self._check(self.lib.fstat_get_profile(self.handle, ms, n))
        return {c: (float(ms[i]), int(n[i])) for i, c in enumerate(self.PROFILE_CLASSES)}

    def set_inflight(self, n: int):
        self._check(self.lib.fstat_set_inflight(self.handle, n))

    def debug_set_geometry(self, log_n2: int = -1, log_tile1: int = -1, log_tile2: int = -1, p2_elems: int = -1):
        self._check(self.lib.fstat_debug_set_geometry(self.handle, log_n2, log_tile1, log_tile2, p2_elems))

    def debug_set_max_sky_slots(self, n: int):
        self._check(self.lib.fstat_debug_set_max_sky_slots(self.handle, n))

    def debug_compute_fafb(self, templates):
        """fstat_debug_compute_fafb: (Fa, Fb) as two complex64 device tensors [n_tmpl][n_bins]."""
        t = _templates_array(templates)
        torch = self._torch
        out = torch.empty((t.shape[0], self.n_bins, 4), dtype=torch.float32, device="cuda")
        self._check(self.lib.fstat_debug_compute_fafb(self.handle, t.ctypes.data, t.shape[0], out.data_ptr()))
        return torch.complex(out[..., 0], out[..., 1]), torch.complex(out[..., 2], out[..., 3])

    def debug_set_paths(self, fused_sky: int = -1, single: int = -1):
        self._check(self.lib.fstat_debug_set_paths(self.handle, fused_sky, single))
