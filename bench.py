#!/usr/bin/env python
"""bench.py -- X-engine throughput on B200 (complex MACs/s) and fraction of the relevant roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c2] [--no-sweep] [--impl reference]

One "step" = one corr_xengine call (the whole hot path: fused corner turn, CMAC, epilogue) over one
integration of the named config's seeded synthetic input.  The headline
workload is BASELINE.json configs[1] (c2: N_I=64, 768 channels, T=10000; 6x the paper's one-second
workload).  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "xengine_complex_macs_per_s"
UNIT = "CMAC/s"
L2_BYTES = 126 * 1024 * 1024
# FP32 FMA peak: measured live by the library's FFMA issue-rate probe (corr_probe_ffma); this derived figure
# (148 SMs x 128 lanes x 2 flops x max clock) is printed beside it and used only if the probe cannot run
FP32_PEAK_DERIVED = 148 * 128 * 2 * 1.965e9


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


def fp32_peak_flops(peaks, pkg=None):
    """FP32 FMA peak in FLOP/s: the best of the scalar and packed issue-rate probes, else the derived figure."""
    if "fp32_flops" not in peaks:
        peaks["fp32_flops"], peaks["fp32_source"] = FP32_PEAK_DERIVED, "derived: 148 SM x 128 lanes x 2 x 1.965 GHz"
        if pkg is not None:
            try:
                r = {k: max(pkg.probe_ffma(packed=(k == "packed"), iters=8192)["tflops"] for _ in range(3)) for k in ("scalar", "packed")}
                peaks["fp32_probe"] = r
                peaks["fp32_flops"] = max(r.values()) * 1e12
                peaks["fp32_source"] = "measured: corr_probe_ffma (register-resident FMA chains, best of scalar FFMA / packed FFMA2)"
            except Exception:
                pass
    return peaks["fp32_flops"]


def int8_peak_tops(peaks, pkg=None):
    """Dense int8 tensor peak in TOP/s: measured live by the library's tcgen05 issue-rate probe
    (M=128, N=256, K=32, MN-major operands, pseudo-random bytes); else 2 x measured bf16."""
    if "int8_tops" not in peaks:
        peaks["int8_tops"], peaks["int8_source"] = 2.0 * peaks["bf16_tflops"], "2 x bf16 of " + peaks["source"]
        if pkg is not None:
            try:
                best = max(pkg.probe_mma(128, 256, True, 16384, random_fill=True)["tops"] for _ in range(3))
                peaks["int8_tops"], peaks["int8_source"] = best, "measured: corr_probe_mma (tcgen05 kind::i8 issue loop)"
            except Exception:
                pass
    return peaks["int8_tops"]


def roofline_times(w, peaks):
    """(t_hbm, t_alu) seconds per integration: north_star's lower-of-two roofline."""
    t_a = w.in_bytes / (peaks["hbm_gbs"] * 1e9)
    ops = 8.0 * w.cmacs
    peak_ops = int8_peak_tops(peaks) * 1e12 if w.dtype == "ci8" else fp32_peak_flops(peaks)
    return t_a, ops / peak_ops


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index=0, period=0.01):
        super().__init__(daemon=True)
        self.period, self.samples, self.reasons, self.stop_flag = period, [], set(), False
        self.power_w = []
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {getattr(nv, k): k for k in dir(nv) if k.startswith("nvmlClocksEventReason") or
                 k.startswith("nvmlClocksThrottleReason")}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM))
                try:
                    self.power_w.append(nv.nvmlDeviceGetPowerUsage(self.dev) / 1000.0)
                except Exception:
                    pass
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.dev)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev)
                for bit, name in names.items():
                    if isinstance(bit, int) and bit and (r & bit) and bit & (bit - 1) == 0:
                        self.reasons.add(name.replace("nvmlClocksEventReason", "").replace("nvmlClocksThrottleReason", ""))
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        s = sorted(self.samples)
        busy = [x for x in s if self.max_mhz is None or x > 0.3 * self.max_mhz] or s
        out = {"sm_mhz": busy[len(busy) // 2] if busy else None, "sm_max_mhz": self.max_mhz,
               "reasons": sorted(r for r in self.reasons if r not in ("GpuIdle", "None", "All"))}
        if self.power_w:
            out["power_w_max"] = round(max(self.power_w), 1)
        return out


def make_inputs(w, n_buffers, torch, rank=0):
    """n_buffers distinct device-resident integrations (rotated when one buffer fits in L2)."""
    return [torch.from_numpy(w.generate(integration=k + 1000 * rank)).cuda() for k in range(n_buffers)]


def shard_plan(w, world, rank):
    """Strong scaling: rank `rank` of `world` owns the channel window
    [c0, c1) of the ONE seeded cube every rank holds; returns (c0, c1, arguments of corr_create for the window,
    arguments of corr_set_chan_window)."""
    c0, c1 = shard_channels(w.n_chan, world, rank)
    return c0, c1, (w.n_inputs, c1 - c0, w.n_time, w.dtype), (w.n_chan, c0)


def time_config(pkg, torch, w, steps, warmup, rank=0, sampler=None, window=None):
    """Device-resident timing of `steps` corr_xengine calls.  Returns dict with per-step seconds.  window = (c0, c1):
    the handle correlates that channel window of the full cube in place (strong scaling)."""
    if window is None:
        h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, w.dtype)
    else:
        h = pkg.corr_create(w.n_inputs, window[1] - window[0], w.n_time, w.dtype)
        h.set_chan_window(w.n_chan, window[0])
    n_buf = 1 if w.in_bytes > 2 * L2_BYTES else min(64, -(-3 * L2_BYTES // w.in_bytes))
    if w.in_bytes <= (64 << 20) and w.dtype == "ci8":
        n_buf = 64  # two batched launches of 32 integrations on distinct buffers
    bufs = make_inputs(w, n_buf, torch, 0 if window is not None else rank)  # strong scaling: the same cube on every rank
    vis = h.empty_vis()
    stream = torch.cuda.current_stream()
    for k in range(warmup):
        h.xengine(bufs[k % n_buf], vis, stream)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    ev[0].record(stream)
    for k in range(steps):
        h.xengine(bufs[k % n_buf], vis, stream)
        ev[k + 1].record(stream)
    torch.cuda.synchronize()
    if sampler:
        sampler.stop_flag = True
    total = ev[0].elapsed_time(ev[steps]) * 1e-3
    per = sorted(ev[k].elapsed_time(ev[k + 1]) * 1e-3 for k in range(steps))
    out = {"total_s": total, "mean_s": total / steps, "median_s": per[len(per) // 2], "best_s": per[0],
           "launches": steps * h.launches_per_call, "n_buffers": n_buf, "handle": h, "bufs": bufs, "vis": vis}
    if n_buf == 1 and not sampler and window is None:
        # one call on an idle, cooled-down device (the "kernel timed alone" regime of the burst peaks): input > L2
        lone = []
        for k in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            time.sleep(0.02)
            e0.record(stream)
            h.xengine(bufs[0], vis, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            lone.append(e0.elapsed_time(e1) * 1e-3)
        out["isolated_s"] = sorted(lone)[len(lone) // 2]
    if n_buf > 1 and not sampler and window is None:
        # isolated latency of one call (device idle before and after), SURVEY H3
        lone = []
        for k in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record(stream)
            h.xengine(bufs[k % n_buf], vis, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            lone.append(e0.elapsed_time(e1) * 1e-3)
        out["isolated_s"] = sorted(lone)[len(lone) // 2]
        # an integration that fits in L2 is launch-bound when enqueued call by call from Python: the steady
        # state is one CUDA graph of n_buf calls (one per rotating buffer, > 2x L2 in total), replayed
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                for k in range(n_buf):
                    h.xengine(bufs[k], vis, side)
            for _ in range(2):
                g.replay()
            torch.cuda.synchronize()
            reps = []
            for _ in range(max(3, -(-steps // n_buf))):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(side)
                g.replay()
                e1.record(side)
                torch.cuda.synchronize()
                reps.append(e0.elapsed_time(e1) * 1e-3 / n_buf)
        out["graph_s"] = sorted(reps)[len(reps) // 2]
        del g
        # independent integrations may also overlap: the small-input plan leaves SMs idle (c1: 64 of 148), so the
        # same n_buf calls spread over 4 streams inside one graph run two to three at a time
        if w.in_bytes <= (64 << 20):
            n_str = 4
            hs = [pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, w.dtype) for _ in range(n_str)]
            vs = [h.empty_vis() for _ in range(n_str)]
            lanes = [torch.cuda.Stream() for _ in range(n_str)]
            with torch.cuda.stream(side):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=side):
                    for st in lanes:
                        st.wait_stream(side)
                    for k in range(n_buf):
                        hs[k % n_str].xengine(bufs[k], vs[k % n_str], lanes[k % n_str])
                    for st in lanes:
                        side.wait_stream(st)
                for _ in range(2):
                    g.replay()
                torch.cuda.synchronize()
                reps = []
                for _ in range(max(3, -(-steps // n_buf))):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(side)
                    g.replay()
                    e1.record(side)
                    torch.cuda.synchronize()
                    reps.append(e0.elapsed_time(e1) * 1e-3 / n_buf)
            out["graph4_s"] = sorted(reps)[len(reps) // 2]
            del g
            for hh in hs:
                hh.destroy()
            # the batched entry point (corr_xengine_batch): ONE launch per `nb` integrations, ONE
            # stream; a graph of n_buf / nb launches over the n_buf distinct buffers (> 2 x L2 in total), replayed
            for nb in (32, 64):
                if n_buf % nb:
                    continue
                vs = [h.empty_vis() for _ in range(nb)]
                with torch.cuda.stream(side):
                    h.xengine_batch(bufs[:nb], vs, side)
                    torch.cuda.synchronize()
                    g = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(g, stream=side):
                        for c in range(n_buf // nb):
                            h.xengine_batch(bufs[c * nb:(c + 1) * nb], vs, side)
                    for _ in range(2):
                        g.replay()
                    torch.cuda.synchronize()
                    reps = []
                    for _ in range(max(5, -(-steps // n_buf))):
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record(side)
                        g.replay()
                        e1.record(side)
                        torch.cuda.synchronize()
                        reps.append(e0.elapsed_time(e1) * 1e-3 / n_buf)
                out[f"batch{nb}_s"] = sorted(reps)[len(reps) // 2]
                if nb == 32:
                    out["batch_vis"], out["batch_bufs"] = vs, bufs[n_buf - nb:]
                del g
    return out


def time_e2e(pkg, torch, w, h, steps, rank=0):
    """Same metric through the public call with HOST buffers: per step, H2D of the integration from
    pinned memory, corr_xengine, D2H of the visibilities -- all inside the timed region."""
    n_host = 2 if w.in_bytes > (1 << 28) else 4
    host = [torch.from_numpy(w.generate(integration=50 + k + 1000 * rank)).pin_memory() for k in range(n_host)]
    d_in = torch.empty_like(host[0], device="cuda")
    vis = h.empty_vis()
    h_vis = torch.empty(vis.shape, dtype=vis.dtype).pin_memory()
    stream = torch.cuda.current_stream()
    for k in range(2):
        d_in.copy_(host[k % n_host], non_blocking=True)
        h.xengine(d_in, vis, stream)
        h_vis.copy_(vis, non_blocking=True)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for k in range(steps):
        d_in.copy_(host[k % n_host], non_blocking=True)
        h.xengine(d_in, vis, stream)
        h_vis.copy_(vis, non_blocking=True)
    e1.record(stream)
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3 / steps
    return {"value": w.cmacs / sec, "unit": UNIT, "h2d_bytes_per_step": w.in_bytes, "d2h_bytes_per_step": w.vis_bytes,
            "ms_per_step": sec * 1e3, "steps": steps, "h2d_gbs": w.in_bytes / sec / 1e9}


def cpu_baseline(w, target_s=12.0, gpu_vis=None):
    """The oracle as it stands, timed on this box's host cores on a bounded sample of the SAME
    workload: the first k channels over the full integration (channels are independent,
    PAPER.md:115).  Also compares those channels with the GPU output of the timed run."""
    import numpy as np
    import oracle
    cores = oracle.host_threads()
    fn = oracle.xengine_ci8 if w.dtype == "ci8" else oracle.xengine_cf32
    x = w.generate()
    t0 = time.perf_counter()
    fn(x, 0, 1, threads=1)
    one = max(time.perf_counter() - t0, 1e-4)            # one channel, one thread
    # (i) the plain single-threaded oracle -- the paper's comparator was single-threaded C -- on the
    # first k1 channels (about 2 s; work is exactly linear and independent in the channel)
    k1 = int(min(w.n_chan, max(1, 2.0 / one)))
    t0 = time.perf_counter()
    fn(x, 0, k1, threads=1)
    sec1 = time.perf_counter() - t0
    # (ii) the same loops under OpenMP over channels on all cores
    k = int(max(cores, min(w.n_chan, target_s * cores / one)))
    k = min(w.n_chan, k)
    t0 = time.perf_counter()
    ref = fn(x, 0, k, threads=cores)
    sec = time.perf_counter() - t0
    out = {"value": w.n_time * k * w.n_baselines / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"channels 0..{k - 1} of {w.n_chan}, all T={w.n_time} samples, {sec:.1f} s, OpenMP over channels",
           "single_thread": {"value": w.n_time * k1 * w.n_baselines / sec1, "unit": UNIT, "cores": 1,
                             "sample": f"channels 0..{k1 - 1} of {w.n_chan}, all T={w.n_time} samples, {sec1:.1f} s, one thread"}}
    if gpu_vis is not None:
        k = min(k, len(gpu_vis))   # a channel-sharded rank holds its window only (rank 0: channels 0 .. c1-1)
        g, ref = gpu_vis[:k], ref[:k]
        if w.dtype == "ci8":
            out["parity"] = "bit-exact" if np.array_equal(g, ref) else "MISMATCH"
        else:
            N = w.n_inputs
            ii, jj = np.tril_indices(N)
            sc = np.sqrt(np.abs(ref[:, ii * (ii + 1) // 2 + ii, 0] * ref[:, jj * (jj + 1) // 2 + jj, 0]))
            err = np.hypot(g[..., 0] - ref[..., 0], g[..., 1] - ref[..., 1])
            worst = float(np.max(err / np.maximum(sc, 1e-300)))
            out["parity"] = f"max err/scale {worst:.2e} (tol 1e-5)" if worst <= 1e-5 else f"OUT OF TOLERANCE {worst:.2e}"
    return out


def cpu_baseline_stream_parity(w, ring, d_vis, n_integrations, per_integration=2):
    """The streamed run of config 5 checked against the float64 oracle: for EACH of the integrations, a few sampled
    channels at north_star's tolerance |dV| <= 1e-5 sqrt(|V_ii V_jj|) (V_ii, V_jj from the oracle).  `ring` holds
    the distinct pinned host inputs; integration k streamed ring[k % len(ring)]."""
    import numpy as np
    import oracle
    rng = np.random.default_rng(2024)
    N = w.n_inputs
    ii, jj = np.tril_indices(N)
    worst, checked = 0.0, 0
    cache = {}
    for k in range(n_integrations):
        chans = sorted(int(c) for c in rng.choice(w.n_chan, size=per_integration, replace=False))
        for c in chans:
            key = (k % len(ring), c)
            if key not in cache:
                cache[key] = oracle.xengine_cf32(ring[key[0]].numpy(), c, c + 1, threads=1)[0]
            ref = cache[key]
            g = d_vis[k, c].cpu().numpy().astype(np.float64)
            sc = np.sqrt(np.abs(ref[ii * (ii + 1) // 2 + ii, 0] * ref[jj * (jj + 1) // 2 + jj, 0]))
            err = np.hypot(g[:, 0] - ref[:, 0], g[:, 1] - ref[:, 1])
            worst = max(worst, float(np.max(err / np.maximum(sc, 1e-300))))
            checked += 1
    verdict = "within tolerance" if worst <= 1e-5 else "OUT OF TOLERANCE"
    return {"result": verdict, "max_err_over_scale": worst, "tolerance": 1e-5, "integrations": n_integrations,
            "channels_checked": checked, "sample": f"{per_integration} seeded random channels of every integration, all 2080 baselines each"}


def run_reference(args, w):
    """--impl reference: the oracle on the host cores; each step a bounded sample of the workload."""
    import oracle
    cores = oracle.host_threads()
    fn = oracle.xengine_ci8 if w.dtype == "ci8" else oracle.xengine_cf32
    x = w.generate()
    t0 = time.perf_counter()
    fn(x, 0, 1, threads=1)
    one = max(time.perf_counter() - t0, 1e-4)
    # bounded sample: about 2 s of work per step, less when many steps are asked for, so that the whole
    # --steps K --warmup W run stays within ~2 minutes
    step_s = min(2.0, 120.0 / max(1, args.steps + args.warmup))
    k = int(min(w.n_chan, max(1, step_s * cores / one)))
    for _ in range(args.warmup):
        fn(x, 0, k, threads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        fn(x, 0, k, threads=cores)
    sec = (time.perf_counter() - t0) / args.steps
    val = w.n_time * k * w.n_baselines / sec
    sample = f"channels 0..{k - 1} of {w.n_chan}, all T={w.n_time} samples per step"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int64" if w.dtype == "ci8" else "f64", "data": "synthetic",
            "config": product_config(w, 1, "weak", 1),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def product_config(w, world, scaling, n_buffers):
    """The `config` object of the JSON line; both arms (--impl b200 / reference) print the same one for the same command."""
    return {"workload": workload_name(w), "n_inputs": w.n_inputs, "n_chan": w.n_chan, "n_time": w.n_time,
            "parallelism": (f"channels sharded over {world} GPUs, each reading its window of the one cube in place (corr_set_chan_window)"
                            if (world > 1 and scaling == "strong") else
                            f"channel-independent replicas x{world}" if world > 1 else "single GPU"),
            "l2": (f"input {w.in_bytes / 1e6:.0f} MB per step > 126 MB L2, no flush needed" if n_buffers == 1
                   else f"rotating {n_buffers} distinct input buffers ({n_buffers * w.in_bytes / 1e6:.0f} MB > L2)")}


def workload_name(w):
    return (f"{w.name}: N_I={w.n_inputs}, {w.n_chan} channels, T={w.n_time}, "
            f"{'complex int8 -> int32' if w.dtype == 'ci8' else 'complex float32'}, 1 integration per step")


def shard_channels(n_chan, world, rank):
    """Channel range [c0, c1) of `rank`: the products are independent per frequency channel, so
    channels shard across GPUs with no exchange; the first n_chan % world ranks get one
    channel more."""
    base, extra = divmod(n_chan, world)
    c0 = rank * base + min(rank, extra)
    return c0, c0 + base + (1 if rank < extra else 0)


def dist_setup(n_gpus):
    """One process per GPU under torchrun; returns (rank, world, dist or None)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world == 1:
        return 0, 1, None
    import torch
    import torch.distributed as dist
    rank, local = int(os.environ["RANK"]), int(os.environ.get("LOCAL_RANK", "0"))
    if torch.cuda.is_available():
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        dist.init_process_group("gloo")
    return rank, world, dist


def reduce_max(dist, value, device):
    """Max over ranks of a python float (the job is as slow as its slowest rank)."""
    if dist is None:
        return value
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def tensor_fracs(w, sec, peaks):
    """A tensor-bound int8 config against BOTH int8 denominators: the library's issue-rate probe and the guide's rule
    (another dtype's measured peak x the nominal ratio = 2 x measured bf16 burst)."""
    ops = 8.0 * w.cmacs
    sus = 2.0 * peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])
    return {"frac_probe_peak": ops / (int8_peak_tops(peaks) * 1e12) / sec, "int8_probe_tops": int8_peak_tops(peaks),
            "frac_2xbf16": ops / (2.0 * peaks["bf16_tflops"] * 1e12) / sec, "int8_2xbf16_tops": 2.0 * peaks["bf16_tflops"],
            # this timing is a loop of back-to-back launches: the SM clock sits at 1.25-1.4 GHz under the power cap
            # (corr_probe_stats), the regime of the driver's SUSTAINED bf16 figure (1357 MHz), not of its burst one
            "frac_2xbf16_sustained": ops / (sus * 1e12) / sec, "int8_2xbf16_sustained_tops": sus}


def corner_turn_entry(pkg, torch, w, h, x, steps=10):
    """The standalone corner-turn kernel (second realisation) on this config: the kernel alone
    (reads and writes the input once: 2 x in_bytes of HBM traffic) and corr_xengine routed through it."""
    stream = torch.cuda.current_stream()

    def timed(fn):
        for _ in range(3):
            fn()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        ev[0].record(stream)
        for k in range(steps):
            fn()
            ev[k + 1].record(stream)
        torch.cuda.synchronize()
        per = sorted(ev[k].elapsed_time(ev[k + 1]) * 1e-3 for k in range(steps))
        return per[len(per) // 2]

    scratch = torch.empty_like(x)
    vis = h.empty_vis()
    sec_turn = timed(lambda: h.corner_turn(x, scratch, stream))
    del scratch
    h.set_turn(pkg.CORR_TURN_STANDALONE)
    sec_path = timed(lambda: h.xengine(x, vis, stream))
    h.set_turn(pkg.CORR_TURN_FUSED)
    return {"turn_kernel_ms": sec_turn * 1e3, "turn_kernel_gbs": 2.0 * w.in_bytes / sec_turn / 1e9,
            "xengine_ms_through_standalone_turn": sec_path * 1e3}


def cpu_baseline_sweep_parity(torch, w, h, d_in, target_s=10.0):
    """GPU output of one corr_xengine call on d_in against the oracle, channels 0..k-1 (k = all when the budget allows)."""
    import numpy as np
    import oracle
    vis = h.empty_vis()
    vis.fill_(-0x55555555)
    h.xengine(d_in, vis)
    torch.cuda.synchronize()
    x = d_in.cpu().numpy()
    cores = oracle.host_threads()
    t0 = time.perf_counter()
    first = oracle.xengine_ci8(x, 0, 1, threads=1)
    one = max(time.perf_counter() - t0, 1e-4)
    k = int(min(w.n_chan, max(1, target_s * cores / one)))
    t0 = time.perf_counter()
    ref = oracle.xengine_ci8(x, 0, k, threads=cores)
    sec = time.perf_counter() - t0
    ok = bool(np.array_equal(vis[:k].cpu().numpy(), ref)) and bool(np.array_equal(ref[:1], first))
    del vis
    return {"result": "bit-exact" if ok else "MISMATCH", "channels": k, "of": w.n_chan, "oracle_s": round(sec, 2), "cores": cores}


def sweep_entry(pkg, torch, key, peaks, steps=20, warmup=3):
    """Kernel-only numbers of another config (context for 'vs N_I'; not a bench line of its own)."""
    import corrgen
    w = corrgen.CONFIGS[key]
    r = time_config(pkg, torch, w, steps, warmup)
    t_a, t_b = roofline_times(w, peaks)
    sec = r.get("graph_s", r["median_s"])
    out = {"n_inputs": w.n_inputs, "value": w.cmacs / sec, "unit": UNIT, "ms": sec * 1e3,
           "bound": "hbm" if t_a >= t_b else ("tensor" if w.dtype == "ci8" else "alu"),
           "roofline_ms": max(t_a, t_b) * 1e3, "frac": max(t_a, t_b) / sec, "n_buffers": r["n_buffers"]}
    if w.dtype == "ci8" and t_b > 0.5 * t_a:   # tensor-bound or at the ridge: both int8 denominators
        out.update(tensor_fracs(w, sec, peaks))
        out["frac_2xbf16_roofline"] = max(t_a, 8.0 * w.cmacs / (2.0 * peaks["bf16_tflops"] * 1e12)) / sec
    if w.dtype == "cf32":
        out["fp32_peak_tflops"] = fp32_peak_flops(peaks) / 1e12
        out["fp32_peak_source"] = peaks["fp32_source"]
    out["kernel"] = r["handle"].plan_info()["kernel"]
    if key in ("c2", "c4"):
        out["corner_turn"] = corner_turn_entry(pkg, torch, w, r["handle"], r["bufs"][0])
    if "isolated_s" in r and "graph_s" not in r:
        out["ms_isolated"] = r["isolated_s"] * 1e3  # one call on an idle device (burst regime)
        out["frac_isolated"] = max(t_a, t_b) / r["isolated_s"]
        if w.dtype == "ci8" and t_b > 0.5 * t_a:
            out["frac_2xbf16_roofline_isolated"] = max(t_a, 8.0 * w.cmacs / (2.0 * peaks["bf16_tflops"] * 1e12)) / r["isolated_s"]
    if "graph_s" in r:
        out["timing"] = f"CUDA graph of {r['n_buffers']} calls on rotating buffers, replayed (steady state)"
        out["ms_eager"] = r["median_s"] * 1e3  # call by call from Python: host launch-bound
        out["ms_isolated"] = r["isolated_s"] * 1e3  # one call on an idle device (launch + kernel latency)
        if w.dtype == "ci8" and t_b > 0.5 * t_a:
            out["frac_2xbf16_roofline_isolated"] = max(t_a, 8.0 * w.cmacs / (2.0 * peaks["bf16_tflops"] * 1e12)) / r["isolated_s"]
    if "graph4_s" in r:
        out["ms_4streams"] = r["graph4_s"] * 1e3  # the same calls spread over 4 streams of one graph (they overlap)
        out["frac_4streams"] = max(t_a, t_b) / r["graph4_s"]
    if "batch32_s" in r:
        # corr_xengine_batch: one launch per 32 (64) integrations, one stream, distinct buffers
        out["ms_batched"] = r["batch32_s"] * 1e3
        out["frac_batched"] = max(t_a, t_b) / r["batch32_s"]
        out["batched"] = (f"per integration; graph of {r['n_buffers'] // 32} corr_xengine_batch launches x 32 integrations on "
                          f"{r['n_buffers']} distinct buffers ({r['n_buffers'] * w.in_bytes / 1e6:.0f} MB), replayed")
        if "batch64_s" in r:
            out["ms_batched64"] = r["batch64_s"] * 1e3
            out["frac_batched64"] = max(t_a, t_b) / r["batch64_s"]
        # the batched outputs equal the single-call outputs of the same inputs (which the GPU tests pin to the oracle)
        single = r["handle"].empty_vis()
        same = True
        for k in (0, 17, 31):
            r["handle"].xengine(r["batch_bufs"][k], single)
            same = same and bool(torch.equal(single, r["batch_vis"][k]))
        out["batched_equals_single_calls"] = same
    if w.dtype == "ci8":
        # parity of THIS launch configuration at full size: one more call on buffer 0, compared element by element with the
        # oracle on as many whole channels as about 10 s of host time allow (all of them on a 16-core box)
        try:
            out["parity"] = cpu_baseline_sweep_parity(torch, w, r["handle"], r["bufs"][0])
        except Exception as e:
            out["parity"] = {"result": "not checked", "error": str(e)[:200]}
    if w.dtype == "cf32" and w.n_integrations > 1:
        # streaming driver: n_integrations back-to-back integrations from pinned host buffers,
        # H2D of k+1 under the kernel of k; a ring of 4 distinct pinned buffers stands in for the 20
        ring = [torch.from_numpy(w.generate(integration=k)).pin_memory() for k in range(4)]
        hs = [ring[k % 4] for k in range(w.n_integrations)]
        r["handle"].stream_run(hs)  # warm-up (allocates the two device buffers)
        d_vis, st = r["handle"].stream_run(hs)
        rate = w.n_integrations * w.n_time * w.n_chan / st["device_s"]       # complex samples/s per input
        out["stream"] = {"integrations": w.n_integrations, "device_s": st["device_s"], "kernel_s": st["kernel_s"],
                         "h2d_s": st["h2d_s"], "h2d_gbs": w.n_integrations * w.in_bytes / st["h2d_s"] / 1e9,
                         "samples_per_s_per_input": rate, "rtf_vs_15.36MSps": rate / 15.36e6,
                         "rtf_vs_paper_1.28MSps": rate / 1.28e6, "e2e_cmacs_per_s": w.n_integrations * w.cmacs / st["device_s"]}
        try:   # BASELINE.json config 5: the streamed run "checks against a float64 oracle"
            out["stream"]["parity"] = cpu_baseline_stream_parity(w, ring, d_vis, w.n_integrations)
        except Exception as e:
            out["stream"]["parity"] = {"result": "not checked", "error": str(e)[:200]}
        del ring, hs, d_vis
    r["handle"].destroy()
    del r
    torch.cuda.empty_cache()
    return out


def sustained_entry(pkg, torch, key, peaks, seconds=2.0, block=25):
    """The SUSTAINED regime of a tensor-bound config: >= `seconds` of back-to-back corr_xengine calls, CUDA events every
    `block` calls, SM clock / power / throttle reasons sampled through NVML meanwhile.  Under the power cap the SM clock
    falls well below its maximum; this is the regime MEASURED_PEAKS.json's bf16_tflops_sustained was measured in, so
    frac_sustained divides by 2 x that figure and is only ever quoted with the clock record beside it.  The first
    quarter of the loop (clock still settling) is left out of ms."""
    import corrgen
    w = corrgen.CONFIGS[key]
    h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, w.dtype)
    n_buf = 1 if w.in_bytes > 2 * L2_BYTES else min(8, -(-3 * L2_BYTES // w.in_bytes))
    bufs = make_inputs(w, n_buf, torch)
    vis = h.empty_vis()
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for k in range(3):
        h.xengine(bufs[k % n_buf], vis, stream)
    e0.record(stream)
    for k in range(10):
        h.xengine(bufs[k % n_buf], vis, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    est = e0.elapsed_time(e1) * 1e-3 / 10
    n_blocks = max(8, int(seconds / (est * block)) + 1)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(n_blocks + 1)]
    sampler = ClockSampler(index=torch.cuda.current_device(), period=0.02)
    time.sleep(0.2)
    sampler.start()
    ev[0].record(stream)
    for b in range(n_blocks):
        for k in range(block):
            h.xengine(bufs[k % n_buf], vis, stream)
        ev[b + 1].record(stream)
    torch.cuda.synchronize()
    sampler.stop_flag = True
    sampler.join(timeout=1.0)
    total = ev[0].elapsed_time(ev[n_blocks]) * 1e-3
    q = n_blocks // 4
    settled = ev[q].elapsed_time(ev[n_blocks]) * 1e-3 / ((n_blocks - q) * block)
    first = ev[0].elapsed_time(ev[1]) * 1e-3 / block
    t_a, t_b = roofline_times(w, peaks)
    ops = 8.0 * w.cmacs
    burst, sus = 2.0 * peaks["bf16_tflops"] * 1e12, 2.0 * peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]) * 1e12
    out = {"loop_s": total, "calls": n_blocks * block, "ms": settled * 1e3, "ms_first_block": first * 1e3,
           "frac_sustained": max(w.in_bytes / (peaks["hbm_gbs"] * 1e9), ops / sus) / settled,
           "frac_burst": max(w.in_bytes / (peaks["hbm_gbs"] * 1e9), ops / burst) / settled,
           "denominators": "2 x bf16_tflops_sustained / 2 x bf16_tflops (burst) of MEASURED_PEAKS.json, or input bytes / hbm_gbs if larger",
           "clocks": sampler.summary()}
    h.destroy()
    del bufs, vis
    torch.cuda.empty_cache()
    return out


def _r(x, n=4):
    return None if x is None else float(f"{x:.{n}g}")


def _parity_word(p):
    if not isinstance(p, dict):
        return p
    return p.get("result") if p.get("channels") == p.get("of") else f"{p.get('result')} ({p.get('channels')}/{p.get('of')} ch)"


def summary_of(line):
    """Every config's headline figures in < 1.5 KB, written LAST in the JSON line so that a record which keeps only the tail
    of stdout still holds them.  frac_* are fractions of the relevant roofline = max(input bytes / measured HBM bandwidth,
    8 ops x CMACs / peak): burst = loop of ms-scale calls against 2 x bf16 burst, iso = one call on an idle device against
    the same, sus = the >= 2 s loop against 2 x bf16 sustained (its SM clock and power are in by_config.*.sustained)."""
    by = line.get("by_config", {})
    roof = line["roofline"]
    cpu = line.get("cpu_baseline", {})
    s = {"c2": {"ms": _r(line["ms_per_step"]), "frac_burst": _r(roof["frac"]), "parity": cpu.get("parity")}}
    c1 = by.get("c1", {})
    if "ms" in c1:
        s["c1"] = {"ms_graph": _r(c1["ms"]), "frac_graph": _r(c1["frac"]), "ms_b32": _r(c1.get("ms_batched")),
                   "frac_b32": _r(c1.get("frac_batched")), "ms_b64": _r(c1.get("ms_batched64")), "frac_b64": _r(c1.get("frac_batched64")),
                   "b_eq_single": c1.get("batched_equals_single_calls"), "parity": _parity_word(c1.get("parity"))}
    for key in ("c3", "c4"):
        e = by.get(key, {})
        if "ms" not in e:
            continue
        s[key] = {"ms": _r(e["ms"]), "frac_burst": _r(e.get("frac_2xbf16_roofline")), "ms_iso": _r(e.get("ms_isolated")),
                  "frac_iso": _r(e.get("frac_2xbf16_roofline_isolated")), "kernel": e.get("kernel"),
                  "parity": _parity_word(e.get("parity"))}
        su = e.get("sustained", {})
        if "ms" in su:
            s[key].update({"ms_sus": _r(su["ms"]), "frac_sus": _r(su["frac_sustained"]), "sus_mhz": su["clocks"].get("sm_mhz"),
                           "sus_w": su["clocks"].get("power_w_max"), "sus_reasons": su["clocks"].get("reasons")})
    c5 = by.get("c5", {})
    if "ms" in c5:
        st = c5.get("stream", {})
        par = st.get("parity", {})
        s["c5"] = {"ms": _r(c5["ms"]), "frac_fp32": _r(c5["frac"]), "rtf": _r(st.get("rtf_vs_15.36MSps")),
                   "h2d_gbs": _r(st.get("h2d_gbs")), "stream_parity": par.get("result") if isinstance(par, dict) else par}
    for key in ("c2_4bit", "c3_shape_4bit", "c5_fstage"):
        e = by.get(key, {})
        if "ms" in e:
            s[key] = {"ms": _r(e["ms"]), "frac": _r(e["frac"])}
    curve = by.get("vs_n_inputs")
    if isinstance(curve, dict):
        curve = curve.get("points")
    if isinstance(curve, list):
        s["vs_n_inputs_frac_burst"] = {str(p["n_inputs"]): _r(p["frac_burst"], 3) for p in curve if "frac_burst" in p}
    return s


def curve_entry(pkg, torch, peaks, steps=10, warmup=3):
    """The metric's own axis: useful CMAC/s versus N_I at a fixed input volume (~0.5 GB of int8 samples, T = 2000, c4's
    sample recipe), with each point's roofline fraction (HBM or 2 x measured bf16, burst and sustained)."""
    import corrgen
    out = []
    T = 2000
    for n in (32, 64, 128, 256, 512, 1024, 2048, 4096):
        c = max(1, (512 << 20) // (T * 2 * n))
        w = corrgen.scaled(corrgen.CONFIGS["c4"], n_inputs=n, n_chan=c, n_time=T)
        x = torch.from_numpy(w.generate()).cuda()
        h = pkg.corr_create(n, c, T, "ci8")
        vis = h.empty_vis()
        stream = torch.cuda.current_stream()
        for _ in range(warmup):
            h.xengine(x, vis, stream)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        ev[0].record(stream)
        for k in range(steps):
            h.xengine(x, vis, stream)
            ev[k + 1].record(stream)
        torch.cuda.synchronize()
        per = sorted(ev[k].elapsed_time(ev[k + 1]) * 1e-3 for k in range(steps))
        sec = per[len(per) // 2]
        t_a = w.in_bytes / (peaks["hbm_gbs"] * 1e9)
        t_burst = 8.0 * w.cmacs / (2.0 * peaks["bf16_tflops"] * 1e12)
        t_sus = 8.0 * w.cmacs / (2.0 * peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]) * 1e12)
        out.append({"n_inputs": n, "n_chan": c, "n_time": T, "ms": sec * 1e3, "value": w.cmacs / sec, "unit": UNIT,
                    "bound": "hbm" if t_a >= t_burst else "tensor", "frac_burst": max(t_a, t_burst) / sec,
                    "frac_sustained": max(t_a, t_sus) / sec})
        h.destroy()
        del x, vis
        torch.cuda.empty_cache()
    return out


def packed_entry(pkg, torch, peaks, steps=50, warmup=5, n_inputs=None, n_chan=None, n_time=None):
    """c2 in the paper's 1-byte mode (4+4-bit samples): half the input bytes.
    With n_inputs / n_chan / n_time: the same recipe at another shape (the slab plans of the 4-bit kernel)."""
    import corrgen
    w = corrgen.CONFIGS["c2"]
    if n_inputs:
        w = corrgen.scaled(w, n_inputs=n_inputs, n_chan=n_chan, n_time=n_time)
    x = torch.from_numpy(corrgen.pack_ci4(w.generate())).cuda()
    h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, "ci4")
    vis = h.empty_vis()
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        h.xengine(x, vis, stream)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    ev[0].record(stream)
    for k in range(steps):
        h.xengine(x, vis, stream)
        ev[k + 1].record(stream)
    torch.cuda.synchronize()
    per = sorted(ev[k].elapsed_time(ev[k + 1]) * 1e-3 for k in range(steps))
    sec = per[len(per) // 2]
    t_a = h.in_bytes / (peaks["hbm_gbs"] * 1e9)
    t_b = 8.0 * w.cmacs / (2.0 * peaks["bf16_tflops"] * 1e12)
    out = {"n_inputs": w.n_inputs, "n_chan": w.n_chan, "n_time": w.n_time, "dtype": "4+4-bit packed -> s32", "value": w.cmacs / sec,
           "unit": UNIT, "ms": sec * 1e3, "bound": "hbm" if t_a >= t_b else "tensor (2 x bf16 burst)",
           "roofline_ms": max(t_a, t_b) * 1e3, "frac": max(t_a, t_b) / sec, "in_bytes": h.in_bytes}
    h.destroy()
    return out


def fstage_entry(pkg, torch, peaks, steps=50, warmup=5):
    """the F-stage on the raw voltages of one c5 integration (500 spectra x 12 bands of 128
    channels x 64 inputs, complex int8 -> float32 spectra), then F + X back to back (raw voltages -> visibilities).
    HBM-bound: algorithmic bytes = 2 B read + 8 B written per sample."""
    import corrgen
    w = corrgen.CONFIGS["c5"]
    bands = w.n_chan // 128
    B = w.n_time * bands
    raw = torch.from_numpy(corrgen.gauss_i8(B, 128, w.n_inputs, 4, 4.0, 15.0)).cuda()   # 5-bit Gaussian voltages
    f = pkg.corr_fstage_create(w.n_inputs, 128, B)
    h = pkg.corr_create(w.n_inputs, w.n_chan, w.n_time, "cf32")
    spec = torch.empty((w.n_time, w.n_chan, w.n_inputs, 2), dtype=torch.float32, device="cuda")
    vis = h.empty_vis()
    stream = torch.cuda.current_stream()

    def timed(fn):
        for _ in range(warmup):
            fn()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        ev[0].record(stream)
        for k in range(steps):
            fn()
            ev[k + 1].record(stream)
        torch.cuda.synchronize()
        per = sorted(ev[k].elapsed_time(ev[k + 1]) * 1e-3 for k in range(steps))
        return per[len(per) // 2]

    sec_f = timed(lambda: f.run(raw, spec, stream))
    sec_fx = timed(lambda: (f.run(raw, spec, stream), h.xengine(spec, vis, stream)))
    nbytes = f.in_bytes + f.out_bytes
    t_a = nbytes / (peaks["hbm_gbs"] * 1e9)
    out = {"n_inputs": w.n_inputs, "dtype": "s8 -> f32 (128-point forward transform)", "batch": B,
           "ms": sec_f * 1e3, "bytes": nbytes, "achieved_gbs": nbytes / sec_f / 1e9, "bound": "hbm",
           "roofline_ms": t_a * 1e3, "frac": t_a / sec_f, "samples_per_s": B * 128 * w.n_inputs / sec_f,
           "fx_ms": sec_fx * 1e3, "fx_value": w.cmacs / sec_fx, "unit": UNIT}
    # the streaming driver fed with raw voltages (corr_stream_run_fx): a quarter of the PCIe bytes per integration
    ring = [torch.from_numpy(corrgen.gauss_i8(B, 128, w.n_inputs, 40 + k, 4.0, 15.0)).pin_memory() for k in range(4)]
    hs = [ring[k % 4] for k in range(w.n_integrations)]
    h.stream_run(hs, fstage=f)  # warm-up (allocates the device buffers)
    _, st = h.stream_run(hs, fstage=f)
    rate = w.n_integrations * w.n_time * w.n_chan / st["device_s"]
    out["stream_fx"] = {"integrations": w.n_integrations, "device_s": st["device_s"], "kernel_s": st["kernel_s"],
                        "h2d_s": st["h2d_s"], "h2d_bytes_per_integration": f.in_bytes,
                        "h2d_gbs": w.n_integrations * f.in_bytes / st["h2d_s"] / 1e9,
                        "samples_per_s_per_input": rate, "rtf_vs_15.36MSps": rate / 15.36e6,
                        "rtf_vs_paper_1.28MSps": rate / 1.28e6,
                        "e2e_cmacs_per_s": w.n_integrations * w.cmacs / st["device_s"]}
    # the same in the paper's 1-byte mode (4+4-bit raw samples): half the PCIe bytes again
    raw4 = [torch.from_numpy(corrgen.pack_ci4(corrgen.gauss_i8(B, 128, w.n_inputs, 60 + k, 2.5, 7.0))).pin_memory() for k in range(4)]
    f.set_input("ci4")
    hs4 = [raw4[k % 4] for k in range(w.n_integrations)]
    h.stream_run(hs4, fstage=f)
    _, st = h.stream_run(hs4, fstage=f)
    rate = w.n_integrations * w.n_time * w.n_chan / st["device_s"]
    out["stream_fx_4bit"] = {"integrations": w.n_integrations, "device_s": st["device_s"], "kernel_s": st["kernel_s"],
                             "h2d_bytes_per_integration": f.in_bytes, "h2d_gbs": w.n_integrations * f.in_bytes / st["h2d_s"] / 1e9,
                             "samples_per_s_per_input": rate, "rtf_vs_15.36MSps": rate / 15.36e6,
                             "e2e_cmacs_per_s": w.n_integrations * w.cmacs / st["device_s"]}
    f.destroy()
    h.destroy()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="c2")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one replica of the workload per GPU; strong = the workload's channels sharded over the GPUs")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    import corrgen
    w = corrgen.CONFIGS[args.config]
    rank0 = int(os.environ.get("RANK", "0")) == 0
    if args.impl == "reference":
        if rank0:
            run_reference(args, w)
        return

    import torch
    import paper_0906_1887_b200 as pkg
    rank, world, dist = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    pkg.lib()
    peaks = measured_peaks()
    int8_peak_tops(peaks, pkg)
    fp32_peak_flops(peaks, pkg)
    dev = torch.device("cuda", torch.cuda.current_device())

    w_full = w
    window = None
    if args.scaling == "strong" and world > 1:
        c0, c1, _, _ = shard_plan(w, world, rank)
        window = (c0, c1)   # this rank's channel window of the ONE cube (same seed on every rank), read in place
    sampler = ClockSampler(index=torch.cuda.current_device()) if rank == 0 else None
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    r = time_config(pkg, torch, w, args.steps, args.warmup, rank, sampler, window)
    if dist is not None:
        dist.barrier()
    total_s = reduce_max(dist, r["total_s"], dev)
    sec = total_s / args.steps
    h = r["handle"]
    if r["n_buffers"] > 1:
        h.xengine(r["bufs"][0], r["vis"])
        torch.cuda.synchronize()
    gpu_vis = r["vis"].cpu().numpy()

    # the same calls captured into ONE CUDA graph and replayed: no host launch gaps (reported beside the eager figure)
    graph_ms = None
    try:
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            g = torch.cuda.CUDAGraph()
            n_g = 10
            with torch.cuda.graph(g, stream=side):
                for k in range(n_g):
                    h.xengine(r["bufs"][k % r["n_buffers"]], r["vis"], side)
            g.replay()
            torch.cuda.synchronize()
            reps = []
            for _ in range(5):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(side)
                g.replay()
                e1.record(side)
                torch.cuda.synchronize()
                reps.append(e0.elapsed_time(e1) / n_g)
            graph_ms = sorted(reps)[len(reps) // 2]
            del g
    except Exception:
        graph_ms = None
    e2e = time_e2e(pkg, torch, w, h, args.e2e_steps, 0 if window is not None else rank)
    e2e_sec = reduce_max(dist, e2e["ms_per_step"] * 1e-3, dev)
    e2e["value"] = (w_full.cmacs if (args.scaling == "strong" and world > 1) else world * w.cmacs) / e2e_sec
    e2e["ms_per_step"] = e2e_sec * 1e3

    if rank != 0:
        return
    t_a, t_b = roofline_times(w, peaks)
    kern = r["median_s"]
    if t_a >= t_b:
        roof = {"bound": "hbm", "achieved": w.in_bytes / kern / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s"}
    elif w.dtype == "ci8":
        roof = {"bound": "tensor", "achieved": 8.0 * w.cmacs / kern / 1e12, "peak": int8_peak_tops(peaks), "unit": "TOP/s"}
    else:
        roof = {"bound": "alu", "achieved": 8.0 * w.cmacs / kern / 1e12, "peak": fp32_peak_flops(peaks) / 1e12, "unit": "TFLOP/s"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["peak_source"] = peaks["int8_source"] if roof["bound"] == "tensor" else (peaks["fp32_source"] if roof["bound"] == "alu" else peaks["source"])
    roof["int8_peak_tops"] = int8_peak_tops(peaks)
    roof["int8_peak_source"] = peaks["int8_source"]
    roof["fp32_peak_measured"] = fp32_peak_flops(peaks) / 1e12
    roof["fp32_peak_source"] = peaks["fp32_source"]
    roof["fp32_peak_derived"] = FP32_PEAK_DERIVED / 1e12
    if "fp32_probe" in peaks:
        roof["fp32_probe_tflops"] = peaks["fp32_probe"]
    if roof["bound"] == "tensor":
        roof.update(tensor_fracs(w, kern, peaks))
    plan = h.plan_info()      # the kernel and schedule the library planned (corr_plan_info), not a re-derivation
    roof["kernel"] = plan["kernel"]
    roof["plan"] = {k: plan[k] for k in ("gsize", "slices", "grid", "mixed", "stages", "wide", "resident")}
    roof["kernel_ms"] = kern * 1e3
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    traffic = json.load(open(tpath)).get(args.config) if os.path.exists(tpath) else None
    roof["traffic"] = traffic
    roof["traffic_source"] = ("profiles/traffic.json: dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full "
                              "capture of this kernel (not measured in this run)") if traffic is not None else None

    total_cmacs = w_full.cmacs if (args.scaling == "strong" and world > 1) else world * w.cmacs
    line = {"metric": METRIC, "value": total_cmacs / sec, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak",
            "vs_baseline": None, "dtype": "s8 x s8 -> s32" if w.dtype == "ci8" else "f32", "data": "synthetic",
            "config": product_config(w, world, args.scaling, r["n_buffers"]),
            "clocks": sampler.summary() if sampler else None,
            "e2e": e2e, "gpu_launches": r["launches"], "roofline": roof,
            "graph_ms_per_step": graph_ms}
    if not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(w, gpu_vis=gpu_vis)
    if args.config in ("c2", "c4") and world == 1 and not args.no_sweep:
        try:   # the standalone corner turn (a1, second realisation) measured on the headline workload
            line["corner_turn"] = corner_turn_entry(pkg, torch, w, h, r["bufs"][0])
        except Exception as e:
            line["corner_turn"] = {"error": str(e)[:200]}
    del r
    h.destroy()
    torch.cuda.empty_cache()
    if not args.no_sweep and world == 1:
        sweep = {}
        for key in ("c1", "c2", "c3", "c4", "c5"):
            if key == args.config:
                continue
            try:
                sweep[key] = sweep_entry(pkg, torch, key, peaks)
            except Exception as e:  # the headline line must survive a failing side measurement
                sweep[key] = {"error": str(e)[:200]}
        try:
            sweep["c2_4bit"] = packed_entry(pkg, torch, peaks)
        except Exception as e:
            sweep["c2_4bit"] = {"error": str(e)[:200]}
        try:   # the 4-bit kernel on slab plans (N_I = 256: 5-deep ring of 24 KB stages), c3's shape with c2's sample recipe
            sweep["c3_shape_4bit"] = packed_entry(pkg, torch, peaks, steps=20, warmup=3, n_inputs=256, n_chan=512, n_time=4000)
        except Exception as e:
            sweep["c3_shape_4bit"] = {"error": str(e)[:200]}
        try:
            sweep["c5_fstage"] = fstage_entry(pkg, torch, peaks)
        except Exception as e:
            sweep["c5_fstage"] = {"error": str(e)[:200]}
        try:
            sweep["vs_n_inputs"] = curve_entry(pkg, torch, peaks)
        except Exception as e:
            sweep["vs_n_inputs"] = {"error": str(e)[:200]}
        for key in ("c3", "c4"):   # the seconds-long regime, with its clock record (runs last: it heats the chip)
            if isinstance(sweep.get(key), dict) and "ms" in sweep[key]:
                try:
                    sweep[key]["sustained"] = sustained_entry(pkg, torch, key, peaks)
                except Exception as e:
                    sweep[key]["sustained"] = {"error": str(e)[:200]}
        line["by_config"] = sweep
        line["summary"] = summary_of(line)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
