"""The oracle over a WHOLE template bank, on all host cores, keeping only what a full-bank parity test needs: the three
loudest bins of every template's 2F row (value and bin) and the complete rows of a few named templates.

    python tests/oracle_bank_maxima.py <synth config function, e.g. config5> <out.npz> [--rows 0,5,17] [--limit N]

Test infrastructure ("the oracle runs all templates of configs 1, 2 and 5"): calls only `oracle/` and the
seeded input generators of `synth.py`; run by tests/test_configs_gpu.py as a separate process, started before the GPU
work, so that the fork pool never shares a process with a CUDA context.  Nothing here is tuned: every template goes
through `O.fstat_2F` exactly as in the small parity tests; templates of one sky position share `O.per_sky`.

Output arrays: val float64[n_t][3], bin int64[n_t][3] (descending 2F, ties by ascending bin: `O.topk`), row_idx int64[r],
rows float64[r][n_bins]."""
import argparse
import multiprocessing as mp
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import fstat_oracle as O                      # noqa: E402
from paper_2201_00451_b200 import synth                   # noqa: E402

_STATE = {}
PIECE = 64        # templates of one sky position handled by one worker call (each call prepares the sky position once)


def _unit(args):
    first, count = args
    p, keep = _STATE["p"], _STATE["keep"]
    sky = O.per_sky(p, float(p.templates[first, 0]), float(p.templates[first, 1]))
    out = []
    for t in range(first, first + count):
        row = O.fstat_2F(p, p.templates[t], sky)
        v, b = O.topk(row, 3)
        out.append((t, np.asarray(v, dtype=np.float64), np.asarray(b, dtype=np.int64), row if t in keep else None))
    return out


def sky_pieces(templates, limit=None):
    """Consecutive templates with the same (alpha, delta), cut into pieces of at most PIECE templates."""
    n_t = len(templates) if limit is None else min(limit, len(templates))
    units, first = [], 0
    while first < n_t:
        end = first + 1
        while end < n_t and end - first < PIECE and templates[end, 0] == templates[first, 0] and templates[end, 1] == templates[first, 1]:
            end += 1
        units.append((first, end - first))
        first = end
    return units


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config")
    ap.add_argument("out")
    ap.add_argument("--rows", default="")
    ap.add_argument("--limit", type=int, default=None)
    a = ap.parse_args()
    p = getattr(synth, a.config)()
    keep = {int(x) for x in a.rows.split(",") if x != ""}
    units = sky_pieces(p.templates, a.limit)
    n_t = sum(c for _, c in units)
    _STATE.update(p=p, keep=keep)
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    val = np.full((n_t, 3), -np.inf)
    bins = np.full((n_t, 3), -1, dtype=np.int64)
    rows = {}
    t0 = time.perf_counter()
    with mp.get_context("fork").Pool(cores) as pool:
        for out in pool.imap_unordered(_unit, units, chunksize=1):
            for t, v, b, row in out:
                val[t, :len(v)], bins[t, :len(b)] = v, b
                if row is not None:
                    rows[t] = row
    row_idx = np.array(sorted(rows), dtype=np.int64)
    tmp = a.out + ".tmp.npz"
    np.savez(tmp, val=val, bin=bins, row_idx=row_idx,
             rows=np.stack([rows[t] for t in row_idx]) if len(rows) else np.zeros((0, p.n_bins)))
    os.replace(tmp, a.out)
    print(f"oracle maxima of {n_t} {a.config} templates ({len(units)} sky pieces) on {cores} cores in {time.perf_counter() - t0:.1f} s")


if __name__ == "__main__":
    main()
