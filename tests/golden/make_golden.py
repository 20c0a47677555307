#!/usr/bin/env python
"""Write tests/golden/<config>_oracle.npz: the CPU oracle's zeta and pair counts of a full-size config.

    python tests/golden/make_golden.py c4 [c2 c3 c5 table2_4pcf_lmax10 ...]

Calls ONLY `oracle/` (eq. 34/35 written out) and `workloads/` (seeded input generators); nothing
from the CUDA package is imported, so no stored value comes from the GPU path.  The file holds
  zeta        [n_Lambda, n_B] float64   oracle.zeta(...)["zeta"]
  bin_counts  [nbins] uint64            accepted ordered pairs per radial bin
  max_imag    float                     largest |Im zeta| the oracle met (~0 for even parity)
  digest      str                       workloads.digest(pos, w): sha256 of the input bytes
  seconds, threads                      oracle wall time and OpenMP threads of the run that wrote the file
The GPU parity test regenerates the inputs, checks the digest (a stale fixture fails loudly) and compares element by
element.  c4 (1.6e6 particles, 2.54e10 pairs) took the oracle 3978 s on 8 threads, which is why it is stored; c2, c3
and c5 are recomputed inside the test run.  table2_4pcf_lmax10 (workloads.EXTRA: the input of the paper's Table 2, 4PCF at
lmax = 10, 45 720 outputs) is stored because its contraction takes the oracle minutes.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import workloads as W  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def main(names):
    oracle.build()
    for name in names:
        cfg = W.CONFIGS[name] if name in W.CONFIGS else W.EXTRA[name]
        pos, w = W.make(cfg)
        t0 = time.perf_counter()
        o = oracle.zeta(cfg.order, pos, w, cfg.box, cfg.rmin, cfg.rmax, cfg.nbins, cfg.lmax)
        dt = time.perf_counter() - t0
        out = os.path.join(HERE, f"{name}_oracle.npz")
        np.savez(out, zeta=o["zeta"], bin_counts=o["bin_counts"], max_imag=o["max_imag"], digest=W.digest(pos, w),
                 seconds=dt, threads=oracle.num_threads())
        print(f"{name}: {out}  {dt:.1f} s on {oracle.num_threads()} threads, max|zeta|={np.abs(o['zeta']).max():.6e}, "
              f"pairs={int(o['bin_counts'].sum())}", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or ["c4"])
