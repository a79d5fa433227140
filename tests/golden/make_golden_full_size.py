#!/usr/bin/env python
"""Writes tests/golden/tau00_full_size_*.txt: tau00 of single items of the largest workloads computed by the CPU
oracle alone (oracle.assemble_M + oracle.tau00_refined: FP64 LU of [M | E] with unrestricted partial pivoting and
three steps of iterative refinement with the residual in long double), so that the GPU path can
be compared element by element at full size where the oracle needs minutes per item (H: cond_1 up to 1.6e6).

    python tests/golden/make_golden_full_size.py            # ~10 min on 4 cores; calls nothing but oracle/ and synth_liz/
    python tests/golden/make_golden_full_size.py NC:5       # only the named workload:item cases (NC: ~1 h on one core)

Format: line 1 '# workload item n k', then k*k lines 'row col re im' with 17 significant digits.
"""
from __future__ import annotations

import os
import sys
from concurrent.futures import ProcessPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

CASES = (("H", 0), ("H", 23), ("N", 23), ("C", 24), ("NC", 5), ("P", 24))


def one(case):
    import oracle
    import synth_liz as sl
    key, item = case
    batch = sl.make_batch(key).select([item])
    cfg = batch.cfg
    M = oracle.assemble_M(cfg.n_sites, cfg.lmax, cfg.spin_canted, batch.site_pos[0], batch.species[0], batch.delta,
                          batch.moment_dir[0], batch.z[0])
    tau = oracle.tau00_refined(M, cfg.k, 3)
    path = os.path.join(ROOT, "tests", "golden", f"tau00_full_size_{key}_{item}.txt")
    with open(path, "w") as f:
        f.write(f"# {key} {item} {cfg.n} {cfg.k}\n")
        for r in range(cfg.k):
            for c in range(cfg.k):
                f.write(f"{r} {c} {tau[r, c].real:.17e} {tau[r, c].imag:.17e}\n")
    return path


if __name__ == "__main__":
    os.environ.setdefault("OMP_NUM_THREADS", "1")
    cases = tuple((a.split(":")[0], int(a.split(":")[1])) for a in sys.argv[1:]) or CASES
    with ProcessPoolExecutor(max_workers=min(4, len(cases))) as ex:
        for p in ex.map(one, cases):
            print("wrote", p)
