"""Writes the stored oracle outputs under tests/golden/ — calls ONLY oracle/ and the input generators.

    python tests/golden/make_golden.py cpa64     # 64^3 CPA wave, one full period  (~7 min, 1 core)
    python tests/golden/make_golden.py cpa128    # 128^3 CPA wave, one full period (~2 h, 1 core)

Each .npz holds: the flat indices of a deterministic cell sample (inputs.sample_cells), the oracle's 8
cell-centred primitives + 3 staggered B at those cells after the run, per-variable max|q| over the full field
(denominators of the S16 norm), the L1 errors against the exact solution, and the diagnostics vector.
No value in these files comes from the CUDA path.
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle.binding import Oracle  # noqa: E402
from paper_2401_03008_b200 import inputs  # noqa: E402

G = 4.0 / 3.0
NAMES = "rho vx vy vz p bx by bz bxf byf bzf".split()


def cpa_period(n, direction="diag"):
    w = inputs.cpa_wave(n, n, n, direction=direction)
    o = Oracle(n, n, n, G, 0.3)
    o.set_primitives(*[w[k] for k in "rho vx vy vz p bxf byf bzf".split()])
    d0 = o.diagnostics()
    t0 = time.time()
    steps = o.step(10 ** 9, w["T"])
    wall = time.time() - t0
    d1 = o.diagnostics()
    q = o.get_primitives()
    ex = inputs.cpa_wave(n, n, n, t=d1["t"], direction=direction)
    idx = inputs.sample_cells((n, n, n), 4096, seed=7)
    out = {"n": n, "steps": steps, "t": d1["t"], "idx": idx, "diag0": d0["raw"], "diag1": d1["raw"],
           "wall_s": wall, "names": np.array(NAMES)}
    out["values"] = np.stack([q[k].ravel()[idx] for k in NAMES])
    out["maxabs"] = np.array([np.abs(q[k]).max() for k in NAMES])
    out["l1"] = np.array([np.abs(q[k] - ex[k]).mean() for k in NAMES[:8]])
    return out


if __name__ == "__main__":
    what = sys.argv[1]
    n = {"cpa64": 64, "cpa128": 128, "cpa32": 32}[what]
    res = cpa_period(n)
    np.savez_compressed(os.path.join(HERE, "oracle_%s_period.npz" % what), **res)
    print(what, "steps", res["steps"], "t", res["t"], "wall", res["wall_s"], "L1", res["l1"])
