"""Helpers of the GPU parity tests: oracle rows on a thread pool (numpy releases the GIL in its FFT and array
kernels), compared with the GPU rows as they are produced so that no float64 row is kept, and the paper's
comparison metrics (eq. 9-10) printed for every case."""
import concurrent.futures
import os

import numpy as np

from oracle import fstat_oracle as O

TOL = 1e-3      # BASELINE.json north_star: |2F_gpu - 2F_cpu| <= 1e-3 * max(2F_cpu, 4) per bin


def rel_err(gpu, cpu):
    return np.abs(np.asarray(gpu, dtype=np.float64) - cpu) / np.maximum(cpu, 4.0)


def compare_rows(prob, idxs, gpu_rows, sky=None, workers=None, label=""):
    """Oracle 2F row of every template in idxs against gpu_rows[r] (same order), bin by bin.
    Returns a list of dicts (err, cpu_max, cpu_argmax, r1, r2, theta) and prints one summary line."""
    idxs = list(idxs)
    if sky is None:
        al, de = float(prob.templates[idxs[0], 0]), float(prob.templates[idxs[0], 1])
        assert np.all(prob.templates[idxs, 0] == al) and np.all(prob.templates[idxs, 1] == de)
        sky = O.per_sky(prob, al, de)

    def one(r):
        cpu = O.fstat_2F(prob, prob.templates[idxs[r]], sky)
        g = np.asarray(gpu_rows[r], dtype=np.float64)
        r1, r2, th = O.comparison_metrics(g, cpu)
        return dict(err=float(rel_err(g, cpu).max()), cpu_max=float(cpu.max()), cpu_argmax=int(cpu.argmax()),
                    r1=r1, r2=r2, theta=th, finite=bool(np.isfinite(g).all()))

    workers = workers or max(1, min(8, (os.cpu_count() or 2) // 2, len(idxs)))
    with concurrent.futures.ThreadPoolExecutor(max_workers=workers) as ex:
        out = list(ex.map(one, range(len(idxs))))
    print(f"[parity] {label or prob.name}: {len(idxs)} templates x {prob.n_bins} bins: max |d2F|/max(2F,4) = "
          f"{max(o['err'] for o in out):.2e}, r1 = {max(o['r1'] for o in out):.2e}, r2 = {max(o['r2'] for o in out):.2e}, "
          f"theta = {max(o['theta'] for o in out):.2e} rad (eq. 9-10)")
    return out
