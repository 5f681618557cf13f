"""Writes tests/golden/oracle_c0.json: oracle output for config c0 (all 4 points, all 4 pairs),
sampled.  Calls only oracle/ and workloads/ (never the CUDA path).  Run from the repo root:
    python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.collide import collide_pairs          # noqa: E402
from oracle.tables import precompute              # noqa: E402
from workloads import get_config, make_points     # noqa: E402


def main():
    cfg = get_config("c0")
    tab = precompute(cfg.N, cfg.N_rho, cfg.M, cfg.L, cfg.mass, cfg.omega, cfg.alpha)
    f = make_points(cfg, range(cfg.nx))
    Qpq = collide_pairs(tab, f)
    N3 = cfg.N ** 3
    samples = []
    for x in range(cfg.nx):
        for p in range(cfg.ns):
            for q in range(cfg.ns):
                for z in (0, 73, (4 * 8 + 4) * 8 + 4, (3 * 8 + 5) * 8 + 2, N3 - 1):
                    samples.append({"x": x, "p": p, "q": q, "z": z, "Q": float(Qpq[x, p, q, z])})
    out = {
        "config": "c0",
        "source": "oracle/collide.py via tests/golden/make_golden.py",
        "maxabs": np.abs(Qpq).max(axis=3).tolist(),
        "sum": Qpq.sum(axis=3).tolist(),
        "samples": samples,
    }
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_c0.json"), "w") as fh:
        json.dump(out, fh, indent=1)


if __name__ == "__main__":
    main()
