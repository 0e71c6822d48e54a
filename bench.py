#!/usr/bin/env python
"""bench.py -- dense-flow frame pairs/s at 1280x1024 (BASELINE.json `metric`) on N GPUs of one node.

    python bench.py --gpus 1 --steps 200 --warmup 10
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W
    python bench.py --impl reference ...      # the fp64 oracle on the host cores (slow on purpose)

A "step" is one pass of the whole hot path (convert, pyramid, then the persistent solve kernel: 3 levels
x 10 iterations x {K2 pass, K3 pass} + flow hand-down) over one frame pair of the workload `config3` (BASELINE.json:9; 1280x1024 uint8, 3 levels,
Gaussian window sigma 4 = radius 12, 10 iterations).  Frame pairs are independent, so
N > 1 runs N replicas with no data-path collective ("replicas only", weak scaling).

One JSON line is printed by rank 0: value (device-resident inputs), e2e (host buffers through the
frame pipeline), roofline of the dominant kernel, cpu_baseline (the oracle, bounded sample), clocks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "dense-flow frame pairs/s at 1280x1024"
UNIT = "pairs/s"
WORKLOAD = "config3: 1280x1024 uint8 particle pair, backward-facing-step-like field, 3 levels, Gaussian window sigma 4 (R=12), 10 iterations"
BYTES_PER_PX = {"k2_products_hsum": 16 + 20, "k3_vsum_solve": 28 + 8}    # 72 B per pixel-iteration
NCU_DRAM_BYTES_PER_SOLVE = 13.85e6 + 11.26e6   # dram__bytes_read.sum + dram__bytes_write.sum, one of_solve_pair launch (profiles/)
RING = 16          # default: distinct input pairs + output buffers cycled through: 16*(2.6+10.5) MB = 210 MB > 126 MB L2


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def shard_pairs(n_pairs, rank, world):
    """Round-robin frame pairs over ranks (independent fields -> replicas)."""
    return list(range(rank, n_pairs, world))


def reduce_max_time(ms, dist, device=None):
    """Max over ranks of a per-rank duration (gloo or nccl)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return ms
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def make_ring(n, rank):
    from paper_1306_2461_b200 import synthetic as syn
    pairs = []
    for i in range(n):
        c = syn.config3(seed_offset=i + 100 * rank)
        pairs.append((c.I1, c.I2))
    return pairs, syn.config3(seed_offset=0)


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the fp64 oracle as it stands on the host cores.  Each step = one full
    config-3 pair (about 1-2 s on 8 cores)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import oracle
    from paper_1306_2461_b200 import synthetic as syn
    oracle.build()
    c = syn.config3()
    for _ in range(max(0, min(args.warmup, 1))):
        oracle.solve(c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type)
    steps = max(1, min(args.steps, 20))
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.solve(c.I1, c.I2, c.levels, c.window_radius, c.iterations, c.window_type)
    dt = time.perf_counter() - t0
    val = steps / dt
    cores = oracle.num_threads()
    sample = "%d full 1280x1024 config3 pairs, one oracle solve each (steps capped at 20)" % steps
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": min(args.warmup, 1), "ms_per_step": dt / steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "note": "fp64 CPU oracle (oracle/optflow_oracle.c), OpenMP over rows"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))
    return 0


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_1306_2461_b200 import binding as B
    B.lib()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback "
                         "(use --impl reference for the oracle)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    RING = max(1, args.ring)
    pairs, c0 = make_ring(RING, rank)
    W, H = c0.width, c0.height
    d_in = [(torch.from_numpy(a).to(dev), torch.from_numpy(b).to(dev)) for a, b in pairs]
    d_out = [(torch.empty((H, W), dtype=torch.float32, device=dev), torch.empty((H, W), dtype=torch.float32, device=dev))
             for _ in range(RING)]
    of = B.OpticalFlow(*c0.create_args)
    stream = torch.cuda.Stream(device=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---------------- device-resident throughput (value)
    with torch.cuda.stream(stream):
        for i in range(max(args.warmup, 3) + RING):        # also captures one graph per ring slot
            of.compute(d_in[i % RING][0], d_in[i % RING][1], d_out[i % RING][0], d_out[i % RING][1])
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record()
        for i in range(args.steps):
            of.compute(d_in[i % RING][0], d_in[i % RING][1], d_out[i % RING][0], d_out[i % RING][1])
        e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = of.last_launch_count() * args.steps

    # ---------------- dominant kernel = the persistent solve kernel (all levels x iterations of a pair in one
    # launch): CUDA events on the launching stream around `rep` back-to-back launches of that kernel alone
    with torch.cuda.stream(stream):
        of.run_solve(5)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        rep = 100
        a.record()
        of.run_solve(rep)
        b.record()
        b.synchronize()
        solve_us = a.elapsed_time(b) / rep * 1e3
    # stand-alone K2 / K3 launches at level 0 (each includes a kernel boundary, which the persistent kernel avoids)
    kt = {}
    with torch.cuda.stream(stream):
        for which, name in ((0, "k2_products_hsum"), (1, "k3_vsum_solve")):
            of.run_step(0, which, 20)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            rep = 200
            a.record()
            of.run_step(0, which, rep)
            b.record()
            b.synchronize()
            kt[name] = a.elapsed_time(b) / rep * 1e3      # us per launch
    # in-kernel timeline (SM cycles at every pass boundary, max over CTAs) of one more solve
    of.solve_timeline(True)
    with torch.cuda.stream(stream):
        of.compute(d_in[0][0], d_in[0][1], d_out[0][0], d_out[0][1])
    stream.synchronize()
    tl = of.solve_timeline(False).astype(np.float64)

    # ---------------- the same job with of_set_hoist(1) (opt-in; bit-identical results; reported beside the headline, which
    # stays the five-plane form BASELINE.json's north_star states)
    hoist = None
    if not args.no_hoist:
        of.set_hoist(True)
        with torch.cuda.stream(stream):
            for i in range(3 + RING):
                of.compute(d_in[i % RING][0], d_in[i % RING][1], d_out[i % RING][0], d_out[i % RING][1])
            h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            h0.record()
            for i in range(args.steps):
                of.compute(d_in[i % RING][0], d_in[i % RING][1], d_out[i % RING][0], d_out[i % RING][1])
            h1.record()
            h1.synchronize()
            h_ms = h0.elapsed_time(h1)
            of.run_solve(5)
            h0.record()
            of.run_solve(100)
            h1.record()
            h1.synchronize()
            h_solve_us = h0.elapsed_time(h1) / 100 * 1e3
        of.solve_timeline(True)
        with torch.cuda.stream(stream):
            of.compute(d_in[0][0], d_in[0][1], d_out[0][0], d_out[0][1])
        stream.synchronize()
        h_tl = of.solve_timeline(False).astype(np.float64)
        of.set_hoist(False)
        h_ms = reduce_max_time(h_ms, dist, dev)
        hoist = (h_ms, h_solve_us, h_tl)
    clocks = sampler.stop()
    ms = reduce_max_time(ms, dist, dev)

    # ---------------- end to end through the public pipeline API, host buffers (PAIRS mode)
    e2e_steps = max(args.steps // 2, 10)
    checksum = 0.0

    def pump(n, timed):
        nonlocal checksum
        pending = 0
        for i in range(n):
            slot = of.stream_acquire()
            np.copyto(slot[0], pairs[i % RING][0])
            np.copyto(slot[1], pairs[i % RING][1])
            of.stream_submit()
            pending += 1
            if pending == 2:
                _, u, v = of.stream_result()
                checksum += float(u[H // 2, W // 2]) + float(v[H // 2, W // 2])
                pending -= 1
        while pending:
            _, u, v = of.stream_result()
            checksum += float(u[H // 2, W // 2]) + float(v[H // 2, W // 2])
            pending -= 1

    e2e_ms = float("nan")
    if not args.no_e2e:
        of.stream_open(B.OF_DTYPE_U8, B.OF_STREAM_PAIRS, True)
        pump(4, False)
        barrier()
        t0 = time.perf_counter()
        pump(e2e_steps, True)
        torch.cuda.synchronize(dev)
        e2e_ms = (time.perf_counter() - t0) * 1e3
        of.stream_close()
        e2e_ms = reduce_max_time(e2e_ms, dist, dev)

    # ---------------- oracle timed beside it (rank 0, N = 1 only): bounded sample
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle
        oracle.build()
        n, t0 = 0, time.perf_counter()
        while n < 2 or (time.perf_counter() - t0 < 12.0 and n < 16):
            oracle.solve(pairs[n % RING][0], pairs[n % RING][1], c0.levels, c0.window_radius, c0.iterations, c0.window_type)
            n += 1
        dt = time.perf_counter() - t0
        cpu = {"value": n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": "%d full config3 pairs (1280x1024, 3 levels, R=12 Gaussian, 10 it), %.1f s" % (n, dt)}

    if rank == 0:
        peak, peak_src = measured_peaks()
        px = W * H
        level_px = [((W + (1 << l) - 1) >> l) * ((H + (1 << l) - 1) >> l) for l in range(c0.levels)]
        solve_bytes = 72.0 * sum(level_px) * c0.iterations
        ach = solve_bytes / (solve_us * 1e-6) / 1e9
        # level-0 iteration from the in-kernel timeline: {K2 pass, barrier, K3 pass, barrier} medians
        mhz = clocks.get("sm_mhz") or 1965.0
        L, it = c0.levels, c0.iterations
        d = np.diff(tl) / mhz                                  # us per phase
        i0 = 2 * (L - 1) + 4 * it * (L - 1)                    # first phase of level 0's iterations
        seg = d[i0:i0 + 4 * it].reshape(it, 4)
        med = np.median(seg[:-1], axis=0)
        iter_us = float(med.sum())
        iter_gbs = 72.0 * px / (iter_us * 1e-6) / 1e9
        pix_iters = sum(((W + (1 << l) - 1) >> l) * ((H + (1 << l) - 1) >> l) for l in range(c0.levels)) * c0.iterations
        value = world * args.steps / (ms * 1e-3)
        hoist_out = None
        if hoist is not None:
            h_ms, h_solve_us, h_tl = hoist
            hd = np.diff(h_tl) / mhz
            hseg = hd[i0:i0 + 4 * it].reshape(it, 4)
            hmed = np.median(hseg[1:-1], axis=0)               # iterations 2 .. it-1 of level 0 (the first one forms all five planes)
            h_iter_us = float(hmed.sum())
            # bytes moved with hoisting: first iteration of a level 72 + 12 (a, b, c written), later ones K2 16 R + 8 W, K3 28 R + 8 W
            h_bytes = (84.0 + 60.0 * (it - 1)) * sum(level_px)
            hoist_out = {"api": "of_set_hoist(handle, 1): IxIx, IxIy, IyIy and their window sums formed in the first iteration of a "
                                "level only (SURVEY.md 8(f) note f5); results bit-identical to the headline run "
                                "(tests/test_gpu_parity.py::test_hoisted_invariant_planes_agree_bitwise); opt-in",
                         "value": world * args.steps / (h_ms * 1e-3), "unit": UNIT, "ms_per_step": h_ms / args.steps,
                         "kernel": "of_solve_pair<12, false, true>", "us_per_launch": h_solve_us,
                         "bytes_per_launch": h_bytes, "achieved_GB/s": h_bytes / (h_solve_us * 1e-6) / 1e9,
                         "frac": h_bytes / (h_solve_us * 1e-6) / 1e9 / peak,
                         "iteration_level0": {"us": h_iter_us, "bytes": 60 * px, "GB/s": 60.0 * px / (h_iter_us * 1e-6) / 1e9,
                                              "frac_of_peak": 60.0 * px / (h_iter_us * 1e-6) / 1e9 / peak,
                                              "frac_of_peak_on_72B_basis": 72.0 * px / (h_iter_us * 1e-6) / 1e9 / peak,
                                              "phases_us": {"k2_pass": float(hmed[0]), "barrier_1": float(hmed[1]),
                                                            "k3_pass": float(hmed[2]), "barrier_2": float(hmed[3])}}}
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "levels": c0.levels, "window_radius": c0.window_radius, "iterations": c0.iterations,
                       "window": "gaussian", "parallelism": "replicas only x%d" % world,
                       "l2": "inputs and outputs rotate over a ring of %d distinct pairs (%.0f MB > 126 MB L2); the 47 MB of "
                             "internal planes are L2-resident by construction at this size" % (RING, RING * (2 * px + 8 * px) / 1e6)},
            "mpixel_iterations_per_s": value * pix_iters / 1e6,
            "clocks": clocks,
            "e2e": {"value": world * e2e_steps / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 2 * px,
                    "d2h_bytes_per_step": 8 * px, "steps": e2e_steps,
                    "api": "of_stream_open(PAIRS, host results) / acquire+fill / submit / result", "checksum": checksum},
            "gpu_launches": launches,
            "roofline": {"bound": "hbm", "kernel": "of_solve_pair<12, false, false> (persistent: K2 pass + K3 pass + hand-down, all levels and iterations)",
                         "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                         "traffic": NCU_DRAM_BYTES_PER_SOLVE, "traffic_source": "profiles/r1_persistent_solve.md, final-build addendum (ncu --set full, dram read + write of one launch; the 47 MB of planes are L2 resident)",
                         "peak_source": peak_src, "bytes_per_launch": solve_bytes,
                         "bytes_basis": "72 B per pixel-iteration (K2 16 R + 20 W, K3 28 R + 8 W) x %d pixel-iterations" % (sum(level_px) * c0.iterations),
                         "us_per_launch": solve_us},
            "iteration_level0": {"bytes": 72 * px, "us": iter_us, "GB/s": iter_gbs, "frac_of_peak": iter_gbs / peak,
                                 "phases_us": {"k2_pass": float(med[0]), "barrier_1": float(med[1]), "k3_pass": float(med[2]), "barrier_2": float(med[3])},
                                 "how": "in-kernel SM cycle stamps (of_solve_timeline, max over CTAs) / sampled SM clock; median over iterations"},
            "kernels_level0_standalone_us": kt,
            "variant_hoist": hoist_out,
            "cpu_baseline": cpu,
        }
        print(json.dumps(out))
    of.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer pipeline leg (profiling runs)")
    ap.add_argument("--no-hoist", action="store_true", help="skip the of_set_hoist(1) variant leg (profiling runs)")
    ap.add_argument("--ring", type=int, default=RING, help="distinct input pairs / output buffers cycled through")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
