"""Writes oracle_small_configs.json from the fp64 oracle ONLY (never from the CUDA path).

    python tests/golden/make_golden.py

Small instances of configs 1-4 (same generators, same solver parameters, reduced size so the oracle
takes seconds).  Stored per case: shape, solver parameters, |S|, the validity count, mean/rms of u and
v over S = {det > 1e-3 max det}, and (u, v) at 12 fixed pixels printed with 17 significant digits.
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle                                   # noqa: E402
from paper_1306_2461_b200 import synthetic as syn           # noqa: E402  (input generators only)

CASES = {"config1": (syn.config1, (256, 256)), "config2": (syn.config2, (320, 256)),
         "config3": (syn.config3, (352, 288)), "config4": (syn.config4, (384, 320))}


def sample_points(W, H, n=12):
    rng = np.random.default_rng(20130613)
    return [(int(x), int(y)) for x, y in zip(rng.integers(0, W, n), rng.integers(0, H, n))]


def describe(name):
    gen, (W, H) = CASES[name]
    c = gen(W, H)
    ref = oracle.solve(c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type)
    S = ref["det"] > 1e-3 * ref["det"].max()
    pts = sample_points(W, H)
    return {"width": W, "height": H, "levels": c.levels, "window_radius": c.window_radius,
            "iterations": c.iterations, "window_type": c.window_type,
            "n_S": int(S.sum()), "n_valid": int(ref["valid"].sum()),
            "mean_u": float(ref["u"][S].mean()), "mean_v": float(ref["v"][S].mean()),
            "rms_u": float(np.sqrt((ref["u"][S] ** 2).mean())), "rms_v": float(np.sqrt((ref["v"][S] ** 2).mean())),
            "points": [[x, y, float(ref["u"][y, x]), float(ref["v"][y, x]), bool(S[y, x])] for x, y in pts]}


if __name__ == "__main__":
    out = {k: describe(k) for k in CASES}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_small_configs.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path)
