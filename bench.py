#!/usr/bin/env python
"""bench.py -- dense-flow frame pairs/s (BASELINE.json `metric`) on N GPUs of one node.

    python bench.py --gpus 1 --steps 500 --warmup 10                 # config 3 (the headline workload, 1280x1024)
    python bench.py --workload config4                               # 2048x2048: planes exceed L2, the HBM-bound cross-check
    python bench.py --workload config5                               # 256 consecutive frames through of_stream_* (scheme 1)
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W
    python bench.py --impl reference ...                             # the fp64 oracle on the host cores (slow on purpose)

A "step" is one pass of the whole hot path (frame conversion + pyramid, then the persistent solve kernel: every level, every
iteration {K2 pass, K3 pass} or the fused coarse-level iteration, flow hand-down) over one frame pair of the workload.  Frame
pairs are independent, so N > 1 runs N replicas with no data-path collective ("replicas only", weak scaling).

One JSON line is printed by rank 0: value (device-resident inputs), e2e (host buffers through the frame pipeline), roofline of
the dominant kernel, cpu_baseline (the oracle, bounded sample, all threads and one thread), clocks.
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

UNIT = "pairs/s"
WORKLOADS = {
    "config1": ("dense-flow frame pairs/s at 256x256",
                "config1: 256x256 fp32-from-uint8 particle pair, uniform shift (1.3,-0.7), 1 level, box window R=8, 4 iterations"),
    "config2": ("dense-flow frame pairs/s at 1024x1024",
                "config2: 1024x1024 uint8 particle pair, Lamb-Oseen vortex, 2 levels, box window R=7, 6 iterations"),
    "config3": ("dense-flow frame pairs/s at 1280x1024",
                "config3: 1280x1024 uint8 particle pair, backward-facing-step-like field, 3 levels, Gaussian window sigma 4 (R=12), 10 iterations"),
    "config4": ("dense-flow frame pairs/s at 2048x2048",
                "config4: 2048x2048 uint16 (12-bit) particle pair, random smooth field RMS 3 px, 4 levels, box window R=10, 8 iterations"),
    "config5": ("dense-flow frame pairs/s at 1280x1024, streaming",
                "config5: 256 consecutive 1280x1024 uint8 frames (convected-vortex shear layer), 255 consecutive pairs, 3 levels, box window R=8, "
                "10 iterations, frames uploaded from host memory through the pinned double-buffered pipeline"),
}
RING = 16          # default: distinct input pairs + output buffers cycled through: 16*(2.6+10.5) MB = 210 MB > 126 MB L2 (config 3)
DRAM_FILE = os.path.join(ROOT, "profiles", "r2_solve_dram.csv")      # dram__bytes of one solve launch per workload, from the ncu captures
L2_STREAM_GBPS = 14600.0   # measured: a plain streaming kernel with the K2 byte mix (4 planes read, 5 written, 47 MB, L2 resident) on this B200 (profiles/r2_notes.md)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_dram_bytes(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of one solve launch, as captured with ncu for this build (profiles/)."""
    try:
        import csv
        for row in csv.DictReader(open(DRAM_FILE)):
            if row["workload"] == workload:
                return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]), row["source"]
    except Exception:
        pass
    return None, None


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


def trace_overlap(run):
    """Device activity of one pipeline pass as CUPTI sees it (torch.profiler; nsys is not in this image): how much of the host<->device
    copy time runs under a kernel of the library, i.e. the overlap of Fig. 4."""
    from torch.profiler import ProfilerActivity, profile
    from torch.autograd import DeviceType
    with profile(activities=[ProfilerActivity.CUDA]) as prof:
        run()
    kern, h2d, d2h = [], [], []
    for e in prof.events():
        if e.device_type != DeviceType.CUDA:
            continue
        iv = (float(e.time_range.start), float(e.time_range.end))
        n = e.name.lower()
        if "memcpy htod" in n:
            h2d.append(iv)
        elif "memcpy dtoh" in n:
            d2h.append(iv)
        elif "memcpy" not in n and "memset" not in n:
            kern.append(iv)

    def union(iv):
        out = []
        for a, b in sorted(iv):
            if out and a <= out[-1][1]:
                out[-1][1] = max(out[-1][1], b)
            else:
                out.append([a, b])
        return out

    def length(iv):
        return sum(b - a for a, b in iv)

    def inter(x, y):
        i = j = 0
        tot = 0.0
        while i < len(x) and j < len(y):
            a, b = max(x[i][0], y[j][0]), min(x[i][1], y[j][1])
            if b > a:
                tot += b - a
            if x[i][1] < y[j][1]:
                i += 1
            else:
                j += 1
        return tot
    ku, hu, du = union(kern), union(h2d), union(d2h)
    span = max(b for _, b in ku + hu + du) - min(a for a, _ in ku + hu + du) if (ku or hu or du) else 0.0
    return {"tool": "torch.profiler (CUPTI activity records of every stream of the process)", "span_us": span,
            "kernels": len(kern), "kernel_busy_us": length(ku), "kernel_busy_frac_of_span": length(ku) / span if span else None,
            "h2d_copies": len(h2d), "h2d_us": length(hu), "h2d_under_kernels_frac": inter(hu, ku) / length(hu) if hu else None,
            "d2h_copies": len(d2h), "d2h_us": length(du), "d2h_under_kernels_frac": inter(du, ku) / length(du) if du else None}


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


def make_pairs(workload, n, rank):
    """n seeded synthetic pairs of the workload (distinct where the generator takes a seed offset) and the case description."""
    from paper_1306_2461_b200 import synthetic as syn
    if workload == "config5":
        st = syn.Config5Stream(n + 1)
        frames = [f.copy() for f in st.frames()]
        return [(frames[i], frames[i + 1]) for i in range(n)], st
    if workload == "config3":
        cs = [syn.config3(seed_offset=i + 100 * rank) for i in range(n)]
        return [(c.I1, c.I2) for c in cs], syn.config3(seed_offset=0)
    c = syn.make_case(int(workload[-1]))
    if workload == "config1":                                  # "fp32 from uint8": the frames reach the library as fp32
        return [(c.I1.astype(np.float32), c.I2.astype(np.float32))] * n, c
    return [(c.I1, c.I2)] * n, c


def oracle_leg(workload, threads, budget_s, max_pairs):
    """The oracle as it stands, in a child process with OMP_NUM_THREADS=threads (None: all), on a bounded sample."""
    code = (
        "import sys, time, json, numpy as np\n"
        "sys.path.insert(0, %r)\n"
        "from oracle import oracle\n"
        "import bench\n"
        "pairs, c = bench.make_pairs(%r, 2, 0)\n"
        "n, t0 = 0, time.perf_counter()\n"
        "while n < 1 or (time.perf_counter() - t0 < %f and n < %d):\n"
        "    a, b = pairs[n %% len(pairs)]\n"
        "    oracle.solve(a, b, c.levels, c.window_radius, c.iterations, c.window_type)\n"
        "    n += 1\n"
        "print(json.dumps({'pairs': n, 'seconds': time.perf_counter() - t0, 'threads': oracle.num_threads()}))\n"
    ) % (ROOT, workload, budget_s, max_pairs)
    env = dict(os.environ)
    if threads is not None:
        env["OMP_NUM_THREADS"] = str(threads)
    else:
        env.pop("OMP_NUM_THREADS", None)
    try:
        out = subprocess.run([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600)
        r = json.loads(out.stdout.strip().splitlines()[-1])
    except Exception as e:  # noqa: BLE001
        return {"value": None, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": "failed: %s" % e}
    return {"value": r["pairs"] / r["seconds"], "unit": UNIT, "cores": r["threads"], "kind": "oracle",
            "sample": "%d full %s pairs, one fp64 oracle solve each, %.1f s (OMP_NUM_THREADS=%s)" %
                      (r["pairs"], workload, r["seconds"], "unset" if threads is None else threads)}


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the fp64 oracle as it stands on the host cores.  Each step = one full pair of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import oracle
    oracle.build()
    metric, wl = WORKLOADS[args.workload]
    pairs, c = make_pairs(args.workload, 2, 0)
    warm = max(0, min(args.warmup, 1))
    for _ in range(warm):
        oracle.solve(pairs[0][0], pairs[0][1], c.levels, c.window_radius, c.iterations, c.window_type)
    steps = max(1, min(args.steps, 20))
    t0 = time.perf_counter()
    for i in range(steps):
        a, b = pairs[i % len(pairs)]
        oracle.solve(a, b, c.levels, c.window_radius, c.iterations, c.window_type)
    dt = time.perf_counter() - t0
    val = steps / dt
    cores = oracle.num_threads()
    sample = "%d full %s pairs, one oracle solve each (steps capped at 20)" % (steps, args.workload)
    print(json.dumps({
        "impl": "reference", "metric": metric, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": dt / steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl, "note": "fp64 CPU oracle (oracle/optflow_oracle.c), OpenMP over rows"},
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
    metric, wl = WORKLOADS[args.workload]
    streaming = args.workload == "config5"

    RINGN = max(1, args.ring)
    pairs, c0 = make_pairs(args.workload, RINGN if not streaming else 255, rank)
    W, H = c0.width, c0.height
    esize = pairs[0][0].dtype.itemsize

    def to_dev(a):
        return torch.from_numpy(a.view(np.int16) if a.dtype == np.uint16 else a).to(dev)

    nring = min(RINGN, len(pairs))
    d_in = [(to_dev(a), to_dev(b)) for a, b in pairs[:nring]]
    d_out = [(torch.empty((H, W), dtype=torch.float32, device=dev), torch.empty((H, W), dtype=torch.float32, device=dev))
             for _ in range(nring)]
    of = B.OpticalFlow(*c0.create_args)
    if args.mask != "none":                                     # obstacle mask (row f4): masked tiles and tasks are skipped
        from paper_1306_2461_b200 import synthetic as syn
        m = syn.mask_backward_step(W, H) if args.mask == "step" else np.ones((H, W), np.uint8)
        if args.mask == "half":
            m[:, W // 2:] = 0
        of.set_mask(m)
    if args.equalise > 0:                                       # eq. 2 pre-filter fused with the frame conversion (row f1)
        of.set_equalisation(args.equalise)
    stream = torch.cuda.Stream(device=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---------------- device-resident throughput (value)
    with torch.cuda.stream(stream):
        for i in range(max(args.warmup, 3) + nring):        # also captures one graph per ring slot
            of.compute(d_in[i % nring][0], d_in[i % nring][1], d_out[i % nring][0], d_out[i % nring][1])
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record()
        for i in range(args.steps):
            of.compute(d_in[i % nring][0], d_in[i % nring][1], d_out[i % nring][0], d_out[i % nring][1])
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
    # in-kernel timeline (SM cycles at every pass boundary, max over CTAs) of one more solve
    of.solve_timeline(True)
    with torch.cuda.stream(stream):
        of.compute(d_in[0][0], d_in[0][1], d_out[0][0], d_out[0][1])
    stream.synchronize()
    tl = of.solve_timeline(False).astype(np.float64)

    # ---------------- throughput mode: two pairs per launch (of_compute_dual: the passes of two independent pairs alternate in one
    # persistent kernel and the grid barrier of one pair is waited for behind a pass of the other; results bit-identical to of_compute)
    dual = None
    if not args.no_dual and nring >= 2 and args.mask == "none" and args.equalise == 0:      # (a masked handle cannot share a launch: of_compute_dual would fall back)
        of2 = B.OpticalFlow(*c0.create_args)
        npair2 = nring // 2

        def dual_step(k):
            i, j = 2 * (k % npair2), 2 * (k % npair2) + 1
            B.compute_dual(of, of2, d_in[i][0], d_in[i][1], d_in[j][0], d_in[j][1], d_out[i][0], d_out[i][1], d_out[j][0], d_out[j][1])
        with torch.cuda.stream(stream):
            for k in range(max(args.warmup, 3) + npair2):
                dual_step(k)
        barrier()
        nd = max(1, args.steps // 2)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            g0.record()
            for k in range(nd):
                dual_step(k)
            g1.record()
        barrier()
        d_ms = reduce_max_time(g0.elapsed_time(g1), dist, dev)
        d_launches = of.last_launch_count() * nd
        with torch.cuda.stream(stream):
            B.run_solve_dual(of, of2, 5)
            g0.record()
            B.run_solve_dual(of, of2, 100)
            g1.record()
            g1.synchronize()
            d_solve_us = g0.elapsed_time(g1) / 100 * 1e3
        of.solve_timeline(True)
        with torch.cuda.stream(stream):
            dual_step(0)
        stream.synchronize()
        d_tl = of.solve_timeline(False).astype(np.float64)
        dual = (d_ms, 2 * nd, d_launches, d_solve_us, d_tl)
        of2.close()

    # ---------------- the same job with of_set_hoist(1) (opt-in; bit-identical results; reported beside the headline, which
    # stays the five-plane form BASELINE.json's north_star states)
    hoist = None
    if not args.no_hoist:
        of.set_hoist(True)
        for fused in (True, False):           # a fused coarse level always forms five planes, so with hoisting the two-pass form of the coarse levels can win
            of.set_fused(fused)
            with torch.cuda.stream(stream):
                for i in range(3 + nring):
                    of.compute(d_in[i % nring][0], d_in[i % nring][1], d_out[i % nring][0], d_out[i % nring][1])
                h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                h0.record()
                for i in range(args.steps):
                    of.compute(d_in[i % nring][0], d_in[i % nring][1], d_out[i % nring][0], d_out[i % nring][1])
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
            h_ms = reduce_max_time(h_ms, dist, dev)
            if hoist is None or h_ms < hoist[0]:
                hoist = (h_ms, h_solve_us, h_tl, fused)
        of.set_fused(True)
        of.set_hoist(False)
    clocks = sampler.stop()
    ms = reduce_max_time(ms, dist, dev)

    # ---------------- end to end through the public pipeline API: host buffers in, host fields out
    checksum = 0.0
    e2e = None
    overlap_trace = None
    prefilled_ms = None
    if not args.no_e2e:
        if streaming:
            # config 5 as BASELINE.json:11 states it: the frames sit in ordinary (pageable) host memory, every frame is uploaded once
            # (scheme 1) and is I2 of one pair and I1 of the next; wall clock from the first submit to the last result
            frames = [pairs[0][0]] + [p[1] for p in pairs]                 # 256 frames

            def run_stream():
                nonlocal checksum
                of.stream_open(B.OF_DTYPE_U8, B.OF_STREAM_CONSECUTIVE, True)
                t0 = time.perf_counter()
                got = 0
                for k, f in enumerate(frames):
                    slot = of.stream_acquire()
                    np.copyto(slot, f)
                    of.stream_submit()
                    if k >= 3:                                            # stay two fields behind: uploads k+1, k+2 overlap solve k
                        _, u, v = of.stream_result()
                        checksum += float(u[H // 2, W // 2]) + float(v[H // 2, W // 2])
                        got += 1
                while got < len(frames) - 1:
                    _, u, v = of.stream_result()
                    checksum += float(u[H // 2, W // 2]) + float(v[H // 2, W // 2])
                    got += 1
                dt = time.perf_counter() - t0
                of.stream_close()
                return dt, got
            run_stream()                                                  # warm-up pass (graphs, pinned allocations)
            barrier()
            dt, got = run_stream()
            e2e_ms, e2e_steps = dt * 1e3, got
            if args.trace_overlap and rank == 0:
                overlap_trace = trace_overlap(run_stream)                 # one more pass, under the profiler (not timed)
            api = "of_stream_open(CONSECUTIVE, host results) / acquire+fill / submit / result; 256 frames from pageable host memory, wall clock first submit -> last result"
            h2d, d2h = W * H * esize, 8 * W * H + W * H
        else:
            e2e_steps = min(5000, max(args.steps // 2, 200, int(50.0 / (ms / args.steps))))   # at least 200 pairs and about 50 ms of device work

            def pump(n, fill=True):
                nonlocal checksum
                pending = 0
                for i in range(n):
                    slot = of.stream_acquire()
                    if fill or i < 4:                                     # fill=False: the four pinned slots keep their frames (as a frame grabber
                        np.copyto(slot[0], pairs[i % 4 if not fill else i % nring][0])   # writing into them would leave them)
                        np.copyto(slot[1], pairs[i % 4 if not fill else i % nring][1])
                    of.stream_submit()
                    pending += 1
                    if pending == 3:
                        _, u, v = of.stream_result()
                        checksum += float(u[H // 2, W // 2]) + float(v[H // 2, W // 2])
                        pending -= 1
                while pending:
                    _, u, v = of.stream_result()
                    checksum += float(u[H // 2, W // 2]) + float(v[H // 2, W // 2])
                    pending -= 1
            dt_code = {np.dtype(np.float32): B.OF_DTYPE_F32, np.dtype(np.uint8): B.OF_DTYPE_U8, np.dtype(np.uint16): B.OF_DTYPE_U16}[pairs[0][0].dtype]
            of.stream_open(dt_code, B.OF_STREAM_PAIRS, True)
            pump(6)
            barrier()
            t0 = time.perf_counter()
            pump(e2e_steps)
            torch.cuda.synchronize(dev)
            e2e_ms = (time.perf_counter() - t0) * 1e3
            # the same with the host-side fill of the slots left out (frames already in pinned memory): what the pipeline itself sustains
            pump(8, fill=False)
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            pump(e2e_steps, fill=False)
            torch.cuda.synchronize(dev)
            prefilled_ms = reduce_max_time((time.perf_counter() - t0) * 1e3, dist, dev)
            if args.trace_overlap and rank == 0:
                overlap_trace = trace_overlap(lambda: (pump(min(e2e_steps, 64)), torch.cuda.synchronize(dev)))   # one more stretch, under the profiler (not timed)
            of.stream_close()
            api = "of_stream_open(PAIRS, host results) / acquire+fill / submit / result"
            h2d, d2h = 2 * W * H * esize, 8 * W * H + W * H
        e2e_ms = reduce_max_time(e2e_ms, dist, dev)
        e2e = {"value": world * e2e_steps / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "value_slots_prefilled": (world * e2e_steps / (prefilled_ms * 1e-3)) if prefilled_ms else None,
               "fill": "value: every pair is first copied from ordinary host memory into the pinned slot (np.copyto, one core); "
                       "value_slots_prefilled: the slots already hold the frames; H2D, solve and D2H of every pair in both",
               "steps": e2e_steps, "api": api, "checksum": checksum, "overlap_trace": overlap_trace,
               "overlap": "serial sum per pair would be solve %.0f us + H2D %.0f us + D2H %.0f us at ~25 GB/s pinned PCIe; measured %.0f us per pair" %
                          (ms / args.steps * 1e3, h2d / 25e3, d2h / 25e3, e2e_ms / e2e_steps * 1e3)}

    # ---------------- oracle timed beside it (rank 0, N = 1 only): bounded samples, all threads and one thread
    cpu = cpu1 = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle
        oracle.build()
        cpu = oracle_leg(args.workload, None, 12.0, 16)
        cpu1 = oracle_leg(args.workload, 1, 8.0, 4)

    if rank == 0:
        peak, peak_src = measured_peaks()
        px = W * H
        level_px = [((W + (1 << l) - 1) >> l) * ((H + (1 << l) - 1) >> l) for l in range(c0.levels)]
        pix_iters = sum(level_px) * c0.iterations
        mhz = clocks.get("sm_mhz") or 1965.0
        L, it = c0.levels, c0.iterations
        i0 = 2 * (L - 1) + 4 * it * (L - 1)                    # first phase of level 0's iterations
        traffic, traffic_src = ncu_dram_bytes(args.workload)

        def analyse(tl_, solve_us_, npairs, kernel):
            """Roofline of the solve kernel and per-level timeline from the in-kernel stamps; npairs = pairs one launch solves."""
            solve_bytes = 72.0 * pix_iters * npairs
            ach = solve_bytes / (solve_us_ * 1e-6) / 1e9
            d = np.diff(tl_) / mhz                              # us per phase
            # level-0 iteration: {K2 pass, barrier, K3 pass, barrier} medians over the iterations
            seg = d[i0:i0 + 4 * it].reshape(it, 4)
            med = np.median(seg[:-1], axis=0) if it > 1 else seg[0]
            iter_us = float(med.sum())
            iter_gbs = 72.0 * px * npairs / (iter_us * 1e-6) / 1e9
            # every level, coarse to fine (a fused coarse level has one pass and one barrier per iteration: its time is under k2_pass)
            levels_tl, k = [], 0
            for l in range(L - 1, -1, -1):
                if l < L - 1:
                    levels_tl.append({"level": l, "hand_down_us": float(d[k]), "hand_down_barrier_us": float(d[k + 1])})
                    k += 2
                sg = d[k:k + 4 * it].reshape(it, 4)
                k += 4 * it
                m4 = np.median(sg[:-1], axis=0) if it > 1 else sg[0]
                levels_tl.append({"level": l, "pixels": level_px[l], "k2_pass_us": float(m4[0]), "barrier_1_us": float(m4[1]), "k3_pass_us": float(m4[2]),
                                  "barrier_2_us": float(m4[3]), "iteration_us": float(m4.sum()),
                                  "frac_of_peak": 72.0 * level_px[l] * npairs / (float(m4.sum()) * 1e-6) / 1e9 / peak})
            roof = {"bound": "hbm", "kernel": kernel, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "traffic": traffic * npairs if traffic is not None else None, "traffic_source": traffic_src,
                    "peak_source": peak_src, "bytes_per_launch": solve_bytes,
                    "bytes_basis": "72 B per pixel-iteration (K2 16 R + 20 W, K3 28 R + 8 W; SURVEY.md 8(d)) x %d pixel-iterations x %d pair(s) per launch"
                                   % (pix_iters, npairs),
                    "us_per_launch": solve_us_,
                    "note": "algorithmic bytes over time against the HBM copy peak, as SURVEY.md 8(d) defines the bar; at 1280x1024 the planes are "
                            "L2 resident (see traffic: the single-pair capture x pairs per launch), so the limiter is latency / issue rate, not DRAM: "
                            "against the measured L2-resident streaming rate of the same byte mix the fraction is frac_of_l2_streaming",
                    "frac_of_l2_streaming": ach / L2_STREAM_GBPS, "l2_streaming_GBps": L2_STREAM_GBPS,
                    # the second bound of DESIGN.md sec. 7: fp32 FMA of the two window sums, 2 x 5 x (2R+1) per pixel-iteration, against
                    # 128 FMA per clock per SM (measured 127, profiles/r2_notes.md sec. 1) at the sampled SM clock
                    "window_fma_per_launch": 10.0 * (2 * c0.window_radius + 1) * pix_iters * npairs,
                    "window_fma_frac_of_fma_peak": 10.0 * (2 * c0.window_radius + 1) * pix_iters * npairs / (solve_us_ * 1e-6) / (torch.cuda.get_device_properties(dev).multi_processor_count * 128 * mhz * 1e6),
                    "window_fma_note": "direct (2R+1)-tap sums; box windows of radius >= 4 take the add-only form with about half as many operations"}
            it0 = {"bytes": 72 * px * npairs, "us": iter_us, "GB/s": iter_gbs, "frac_of_peak": iter_gbs / peak,
                   "phases_us": {"k2_pass": float(med[0]), "barrier_1": float(med[1]), "k3_pass": float(med[2]), "barrier_2": float(med[3])},
                   "how": "in-kernel SM cycle stamps (of_solve_timeline, max over CTAs) / sampled SM clock; median over iterations" +
                          ("; one iteration of BOTH pairs (K2 pass of a, of b, K3 pass of a, of b; the barriers are waited for behind the other pair's pass)"
                           if npairs == 2 else "")}
            return roof, it0, levels_tl

        s_value = world * args.steps / (ms * 1e-3)
        s_roof, s_it0, s_levels = analyse(tl, solve_us, 1, "of_solve_pair<R, false, false> (persistent: K2 pass + K3 pass per iteration, fused coarse "
                                                          "levels, hand-down; all levels and iterations of one pair)")
        single = {"api": "of_compute (one pair per launch: lowest latency)", "value": s_value, "unit": UNIT, "ms_per_step": ms / args.steps,
                  "gpu_launches": launches, "roofline": s_roof, "iteration_level0": s_it0, "levels_timeline": s_levels}
        # the headline is the faster of the two launch modes of the public API; the other one is reported beside it
        dual_out = None
        if dual is not None:
            d_ms, d_pairs, d_launches, d_solve_us, d_tl = dual
            d_roof, d_it0, d_levels = analyse(d_tl, d_solve_us, 2, "of_solve_dual<R> (persistent, two pairs per launch: the passes of the two pairs alternate, "
                                                                  "split grid barriers; K2 pass + K3 pass per iteration, fused coarse levels, hand-down)")
            dual_out = {"api": "of_compute_dual (two pairs of two handles per launch: throughput mode; results bit-identical to of_compute)",
                        "value": world * d_pairs / (d_ms * 1e-3), "unit": UNIT, "ms_per_step": d_ms / d_pairs, "steps": d_pairs,
                        "gpu_launches": d_launches, "roofline": d_roof, "iteration_level0": d_it0, "levels_timeline": d_levels}
        if dual_out is not None and dual_out["value"] > s_value:
            value, ms_per_step, n_launch, steps_timed = dual_out["value"], dual_out["ms_per_step"], dual_out["gpu_launches"], dual_out["steps"]
            roof, it0, levels_tl = dual_out["roofline"], dual_out["iteration_level0"], dual_out["levels_timeline"]
            launch_mode = "two pairs per launch (of_compute_dual): the faster mode on this workload; one pair per launch under single_pair"
        else:
            value, ms_per_step, n_launch, steps_timed = s_value, ms / args.steps, launches, args.steps
            roof, it0, levels_tl = s_roof, s_it0, s_levels
            launch_mode = "one pair per launch (of_compute)" + ("" if dual_out is None else ": the faster mode on this workload; two pairs per launch under dual_launch")
        hoist_out = None
        if hoist is not None:
            h_ms, h_solve_us, h_tl, h_fused = hoist
            hd = np.diff(h_tl) / mhz
            hseg = hd[i0:i0 + 4 * it].reshape(it, 4)
            hmed = np.median(hseg[1:-1], axis=0) if it > 2 else hseg[-1]   # iterations 2 .. it-1 of level 0 (the first one forms all five planes)
            h_iter_us = float(hmed.sum())
            # bytes moved with hoisting: first iteration of a level 72 + 12 (a, b, c written), later ones K2 16 R + 8 W, K3 28 R + 8 W
            h_bytes = (84.0 + 60.0 * (it - 1)) * sum(level_px)
            hoist_out = {"api": "of_set_hoist(handle, 1): IxIx, IxIy, IyIy and their window sums formed in the first iteration of a "
                                "level only (SURVEY.md 8(f) note f5); results bit-identical to the headline run "
                                "(tests/test_gpu_parity.py::test_hoisted_invariant_planes_agree_bitwise); opt-in; one pair per launch; the faster of "
                                "of_set_fused(1) / of_set_fused(0) for the coarse levels",
                         "coarse_levels": "fused (five planes per iteration there)" if h_fused else "two-pass (of_set_fused(0): hoisted like level 0)",
                         "value": world * args.steps / (h_ms * 1e-3), "unit": UNIT, "ms_per_step": h_ms / args.steps,
                         "kernel": "of_solve_pair<R, false, true>", "us_per_launch": h_solve_us,
                         "bytes_per_launch": h_bytes, "achieved_GB/s": h_bytes / (h_solve_us * 1e-6) / 1e9,
                         "frac": h_bytes / (h_solve_us * 1e-6) / 1e9 / peak,
                         "iteration_level0": {"us": h_iter_us, "bytes": 60 * px, "GB/s": 60.0 * px / (h_iter_us * 1e-6) / 1e9,
                                              "frac_of_peak": 60.0 * px / (h_iter_us * 1e-6) / 1e9 / peak,
                                              "phases_us": {"k2_pass": float(hmed[0]), "barrier_1": float(hmed[1]),
                                                            "k3_pass": float(hmed[2]), "barrier_2": float(hmed[3])}}}
        planes_mb = 9 * 4 * px / 1e6
        out = {
            "metric": metric, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps_timed, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl, "levels": c0.levels, "window_radius": c0.window_radius, "iterations": c0.iterations,
                       "window": "gaussian" if c0.window_type == B.OF_WINDOW_GAUSSIAN else "box", "parallelism": "replicas only x%d" % world,
                       "launch": launch_mode, "mask": args.mask, "equalisation_radius": args.equalise,
                       "l2": "inputs and outputs rotate over a ring of %d pairs (%.0f MB; L2 is 126 MB); the %.0f MB of internal planes of the "
                             "finest level %s" % (nring, nring * (2 * px * esize + 8 * px) / 1e6, planes_mb,
                                                  "exceed L2: this workload is HBM bound" if planes_mb > 126 else "are L2 resident at this size")},
            "mpixel_iterations_per_s": value * pix_iters / 1e6,
            "clocks": clocks,
            "e2e": e2e,
            "gpu_launches": n_launch,
            "roofline": roof,
            "iteration_level0": it0,
            "levels_timeline": levels_tl,
            "single_pair": single if (dual_out is not None and dual_out["value"] > s_value) else None,
            "dual_launch": dual_out if not (dual_out is not None and dual_out["value"] > s_value) else None,
            "variant_hoist": hoist_out,
            "cpu_baseline": cpu,
            "cpu_baseline_1thread": cpu1,
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
    ap.add_argument("--workload", default="config3", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer pipeline leg (profiling runs)")
    ap.add_argument("--no-hoist", action="store_true", help="skip the of_set_hoist(1) variant leg (profiling runs)")
    ap.add_argument("--no-dual", action="store_true", help="skip the two-pairs-per-launch leg (of_compute_dual); the headline is then the single-pair launch")
    ap.add_argument("--mask", default="none", choices=["none", "step", "half"],
                    help="obstacle mask set on the handle (of_set_mask): step = synthetic.mask_backward_step (14 %% obstacle), half = right half of the frame")
    ap.add_argument("--equalise", type=int, default=0, help="radius of the eq. 2 local-equalisation pre-filter (of_set_equalisation); 0 = off; the paper uses 5")
    ap.add_argument("--trace-overlap", action="store_true",
                    help="one extra stretch of the frame pipeline under torch.profiler; reports how much of the copy time runs under kernels")
    ap.add_argument("--ring", type=int, default=RING, help="distinct input pairs / output buffers cycled through")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
