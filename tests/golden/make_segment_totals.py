#!/usr/bin/env python
"""Writes tests/golden/segment_totals.txt: the exact number of positive-length (ray, cell) segments of one
sweep (per frequency bin) for the five BASELINE.json configs, from the CPU oracle alone.

The count is a property of the integer traversal (readings O3/O4: PAPER.md:86, 150, 177), not of
the fields, so the oracle is run on a unit medium with one bin; the GPU tests compare rt_total_segments
and the sum of rt_segment_counts against these integers at the full benchmark sizes, where running the
full oracle sweep inside the test would take minutes.  Next to each total it writes the SHA-256 of the
oracle's per-cell count array summed over the directions (uint32 little-endian, [nz][ny][nx]): the GPU
tests hash rt_segment_counts(-1) the same way, which makes the integer gate bit-exact on EVERY cell of
the full-size configs, not only on the sampled ones.

    python tests/golden/make_segment_totals.py [C1 C2 ...]      (calls only oracle/ and rt_inputs/)
"""
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle                      # noqa: E402
from rt_inputs import CONFIGS                  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "segment_totals.txt")


def main():
    names = sys.argv[1:] or ["C1", "C2", "C3", "C4", "C5"]
    have = {}
    if os.path.exists(OUT):
        for line in open(OUT):
            if line.strip() and not line.startswith("#"):
                w = line.split()
                have[w[0]] = (int(w[1]), w[4] if len(w) > 4 else "-")
    for name in names:
        spec = CONFIGS[name]
        nx, ny, nz = spec.dims
        kap = np.ones((1, nz, ny, nx), dtype=np.float32)
        S = np.zeros((1, nz, ny, nx), dtype=np.float32)
        dirs = oracle.healpix_dirs(spec.nside)
        t0 = time.time()
        r = oracle.sweep(kap, S, dirs, want_counts=True)
        assert int(r["cnt_sum"].astype(np.uint64).sum()) == r["seg_total"]
        sha = hashlib.sha256(np.ascontiguousarray(r["cnt_sum"], dtype="<u4").tobytes()).hexdigest()
        have[name] = (r["seg_total"], sha)
        print(name, r["seg_total"], sha, "%.0f s" % (time.time() - t0), flush=True)
        with open(OUT, "w") as f:
            f.write("# exact segments per sweep and bin (oracle/oracle.c orc_sweep, readings O3/O4); written by make_segment_totals.py\n")
            f.write("# config  segments  mesh  directions  sha256 of the per-cell counts summed over directions (uint32 LE, [nz][ny][nx])\n")
            for k in sorted(have):
                sp = CONFIGS[k]
                f.write("%s %d %dx%dx%d %d %s\n" % (k, have[k][0], sp.dims[0], sp.dims[1], sp.dims[2], sp.ndirs, have[k][1]))


if __name__ == "__main__":
    main()
