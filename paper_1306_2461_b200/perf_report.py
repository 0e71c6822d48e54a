"""Per-config throughput and in-kernel pass timeline of the solve (CUDA path only).

    python -m paper_1306_2461_b200.perf_report [--configs 1 2 3 4] [--reps 50] [--masks] [--hoist]

For every config of BASELINE.json: frame pairs/s with device-resident inputs (CUDA events over `reps`
solves), the persistent solve kernel alone (of_run_solve), its algorithmic GB/s on the 72 B per
pixel-iteration basis, and per level the median K2 pass / barrier / K3 pass / barrier times from
of_solve_timeline (SM cycles, maximum over CTAs).  Inputs are the seeded synthetic pairs of synthetic.py.
--masks repeats config 3 with no mask, the backward-step obstacle mask and the right half of the frame masked
(of_set_mask).
"""
from __future__ import annotations

import argparse
import json

import numpy as np


def report(index: int, reps: int, sm_mhz: float, mask=None, mask_name=None, hoist=False):
    import torch
    from . import binding as B, synthetic as syn
    c = syn.make_case(index)
    to_dev = (lambda a: torch.from_numpy(a.view(np.int16)).cuda()) if c.I1.dtype == np.uint16 else (lambda a: torch.from_numpy(a).cuda())
    d1, d2 = to_dev(c.I1), to_dev(c.I2)
    W, H, L, it = c.width, c.height, c.levels, c.iterations
    out = {"config": index, "size": [W, H], "levels": L, "window_radius": c.window_radius, "iterations": it,
           "window": "gaussian" if c.window_type == B.OF_WINDOW_GAUSSIAN else "box", "dtype": str(c.I1.dtype)}
    if mask_name is not None:
        out["mask"] = mask_name
        out["mask_obstacle_share"] = 0.0 if mask is None else float(1.0 - (np.asarray(mask) != 0).mean())
    with B.OpticalFlow(*c.create_args) as of:
        if mask is not None:
            of.set_mask(mask)
        of.set_hoist(hoist)
        out["hoist"] = bool(hoist)
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            u, v = of.compute(d1, d2)
            for _ in range(3):
                of.compute(d1, d2, u, v)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(reps):
                of.compute(d1, d2, u, v)
            b.record()
            b.synchronize()
            pair_us = a.elapsed_time(b) / reps * 1e3
            of.run_solve(3)
            a.record()
            of.run_solve(reps)
            b.record()
            b.synchronize()
            solve_us = a.elapsed_time(b) / reps * 1e3
        of.solve_timeline(True)
        with torch.cuda.stream(s):
            of.compute(d1, d2, u, v)
        s.synchronize()
        tl = of.solve_timeline(False).astype(np.float64)
    px = [((W + (1 << l) - 1) >> l) * ((H + (1 << l) - 1) >> l) for l in range(L)]
    nbytes = 72.0 * sum(px) * it
    out.update({"pair_us": pair_us, "pairs_per_s": 1e6 / pair_us, "solve_kernel_us": solve_us,
                "algorithmic_MB": nbytes / 1e6, "algorithmic_GBps": nbytes / solve_us / 1e3,
                "mpixel_iterations_per_s": sum(px) * it / pair_us})
    d = np.diff(tl) / sm_mhz
    i, levels = 0, []
    for l in range(L - 1, -1, -1):
        if l < L - 1:
            i += 2
        seg = d[i:i + 4 * it].reshape(it, 4)
        i += 4 * it
        med = np.median(seg[:-1] if it > 1 else seg, axis=0)
        if l < L - 1:
            levels.append({"level": l, "hand_down_us": float(d[i - 4 * it - 2]), "hand_down_barrier_us": float(d[i - 4 * it - 1])})
        levels.append({"level": l, "pixels": px[l], "k2_pass_us": float(med[0]), "barrier_us": float(med[1]),
                       "k3_pass_us": float(med[2]), "barrier2_us": float(med[3]), "iteration_us": float(med.sum()),
                       "iteration_GBps": 72.0 * px[l] / med.sum() / 1e3})
    out["levels_timeline"] = levels
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="*", default=[1, 2, 3, 4])
    ap.add_argument("--reps", type=int, default=50)
    ap.add_argument("--sm-mhz", type=float, default=1965.0, help="SM clock used to convert cycle stamps")
    ap.add_argument("--hoist", action="store_true", help="of_set_hoist(1): IxIx, IxIy, IyIy planes formed once per level (60 B basis; "
                                                          "the GB/s figures printed here stay on the 72 B basis)")
    ap.add_argument("--masks", action="store_true", help="config 3 without a mask, with the step mask, with the right half masked")
    args = ap.parse_args()
    if args.masks:
        from . import synthetic as syn
        half = np.ones((1024, 1280), dtype=np.uint8)
        half[:, 640:] = 0
        for name, m in (("none", None), ("backward_step", syn.mask_backward_step(1280, 1024)), ("right_half", half)):
            print(json.dumps(report(3, args.reps, args.sm_mhz, m, name, args.hoist)))
        return
    for k in args.configs:
        print(json.dumps(report(k, args.reps, args.sm_mhz, hoist=args.hoist)))


if __name__ == "__main__":
    main()
