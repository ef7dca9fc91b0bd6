#!/usr/bin/env python
"""bench.py -- whitened injected samples/s of the AMPLFI data-generation hot path on B200.

One "step" = one pass of the whole hot path over one batch of BASELINE.json configs[2]
(training-throughput shape): Welch PSD of a 64 s window of the GPU-resident strip + fused
gather / waveform / projection / injection / whitening of batch 2048 x 3 detectors x 16384 samples.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "whitened injected samples/sec (3-det, 2048 Hz)"
UNIT = "samples/s"
WORKLOAD = ("c2 training-throughput: batch 2048 x H1+L1+V1, fs 2048 Hz, 8 s segments (16384), noise gathered "
            "from a resident quarter-day strip [3, 44236800] at random per-(sample,detector) offsets, Welch PSD "
            "(64 s, 2 s Hann, 50% overlap, mean) re-estimated every step, IMRPhenomD + aligned spins, Table-1 priors")


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--batch", type=int, default=2048)
    ap.add_argument("--strip-len", type=int, default=44236800)
    ap.add_argument("--cpu-sample", type=int, default=1024, help="samples of the batch the CPU oracle is timed on")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="skip the other BASELINE configs (c0, c1, c3 over 1000 seeded runs, c4) measured after the timed region")
    ap.add_argument("--config", default="c2", choices=["c0", "c1", "c2", "c3", "c4", "sweep", "next"],
                    help="c2 (default): the contract line.  c3: online latency p50/p99 over --runs seeded runs.  "
                         "c4: bandwidth stress (batch 8192 x 3 x 65536).  sweep: segment length 1-16 s at 4096 Hz.")
    ap.add_argument("--runs", type=int, default=1000)
    return ap.parse_args()


KERNEL_SOURCES = ("inject_whiten_v3.cu", "fft_tan.cuh", "fft_packed.cuh", "fft_core.cuh", "spec_layout.cuh")


def kernel_source_hash():
    """sha256 over the sources of the dominant kernel: profiles/kernel_counters.txt records the hash of the build its ncu
    numbers were captured from, and they are reported only while the sources still match."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2407_19048_b200", "csrc", name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def kernel_counters():
    """(dram bytes per launch, fp32 lane-operations per sample, note) from one ncu capture, or (None, None, why)."""
    path = os.path.join(ROOT, "profiles", "kernel_counters.txt")
    try:
        with open(path) as fh:
            rec = json.load(fh)
    except Exception:
        return None, None, "profiles/kernel_counters.txt missing"
    if rec.get("source_hash") != kernel_source_hash():
        return None, None, "kernel sources changed since the capture (%s)" % rec.get("capture", "?")
    return rec.get("dram_bytes_per_launch"), rec.get("fp32_lane_ops_per_sample"), rec.get("capture")


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference)
# ------------------------------------------------------------------------------------------------

def oracle_step(wl, rows):
    """The whole hot path for `rows` samples of the workload, in the oracle (fp64, host)."""
    from oracle import project as OP, waveform as OW, welch as OWE, whiten as OWH
    o, nb = wl.extra["bg_offset"], wl.extra["n_bg"]
    psd = OWE.welch(wl.strip[:, o:o + nb].astype(np.float64), wl.fs, wl.nperseg)
    params = wl.params[rows]
    noise = OWH.gather(wl.strip, wl.offsets[rows], wl.n)
    hp, hc, _ = OW.waveform_fd(wl.approximant, params, wl.n, wl.fs, wl.f_lo, wl.f_hi)
    h_det, _ = OP.project(hp, hc, params, wl.gmst, wl.det_ids, wl.n, wl.fs)
    return OWH.inject_whiten(noise, h_det, psd, wl.fs, wl.f_lo, wl.f_hi)


def time_oracle(wl, n_rows, steps=1, warmup=0):
    """-> (samples/s, seconds per step, cores actually used = process CPU time / wall time)."""
    rows = np.arange(n_rows) % wl.batch
    for _ in range(warmup):
        oracle_step(wl, rows)
    t0, c0 = time.perf_counter(), time.process_time()
    for _ in range(steps):
        oracle_step(wl, rows)
    wall, cpu = time.perf_counter() - t0, time.process_time() - c0
    dt = wall / steps
    return n_rows * wl.n_det * wl.n / dt, dt, round(cpu / wall, 2)


def run_reference(args):
    import workloads as WL
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = WL.make_c2(batch=max(args.cpu_sample, 4), strip_len=min(args.strip_len, 1 << 24))
    n_rows = args.cpu_sample
    steps = max(1, min(args.steps, 3))
    warm = min(args.warmup, 1)
    value, dt, cores = time_oracle(wl, n_rows, steps=steps, warmup=warm)
    sample = "%d of 2048 samples (x3 detectors x 16384) + the full 64 s Welch per step; strip shortened to %d" % (
        n_rows, wl.strip.shape[1])
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warm, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "cores_note": "process CPU time / wall time of the numpy oracle", "host_cores": os.cpu_count()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "world_size": int(os.environ.get("WORLD_SIZE", "1"))}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# B200 arm
# ------------------------------------------------------------------------------------------------

class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 20 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def run_b200(args):
    import torch
    import paper_2407_19048_b200 as A      # raises if libamplfi.so is missing: no fallback
    import workloads as WL

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the B200 arm has no CPU fallback")
    if local >= torch.cuda.device_count():
        raise SystemExit("bench.py: rank %d wants cuda:%d but this node has %d GPU(s); one rank per GPU, ranks are never stacked on a device"
                         % (rank, local, torch.cuda.device_count()))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    # ---- synthetic workload (host, seeded), uploaded once: "before commencing training" ----
    from workloads import sharding as SH
    wl = WL.make_c2(batch=args.batch, seed=SH.rank_seed(0xA3D30002, rank), strip_len=args.strip_len)
    B, D, N = wl.batch, wl.n_det, wl.n
    plan = A.Plan(N, wl.fs, wl.det_ids, B, nperseg=wl.nperseg)
    strip = torch.from_numpy(wl.strip).to(dev)
    params_h = torch.from_numpy(wl.params).pin_memory()
    offsets_h = torch.from_numpy(wl.offsets).pin_memory()
    params = params_h.to(dev)
    offsets = offsets_h.to(dev)
    o, nb = wl.extra["bg_offset"], wl.extra["n_bg"]
    bg = strip[:, o:o + nb]                                     # strided view: rows are L apart
    psd = torch.empty((D, wl.nperseg // 2 + 1), dtype=torch.float32, device=dev)
    out = torch.empty((B, D, N), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()

    def step(p=params, off=offsets):
        # one data-generation step = Welch PSD + waveform/projection/injection/whitening (one C-ABI call; the
        # two-call form amplfi_psd_welch + amplfi_inject_whiten gives identical results, tests/test_gpu_parity.py)
        A.amplfi_assemble_batch(plan, B, bg, strip, p, wl.f_lo, wl.f_hi, offsets=off, approximant=wl.approximant,
                                gmst=wl.gmst, psd=psd, out=out, stream=stream)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()

    # ---- device-resident timing: exactly K steps, CUDA events on the launching stream ----
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    plan.set_timing(True)
    launches0 = A.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    total_ms = e0.elapsed_time(e1)
    launches = A.launch_count() - launches0
    kernel_ms = plan.kernel_times_ms()
    plan.set_timing(False)
    clocks = sampler.stop() if rank == 0 else None
    total_ms = SH.max_over_ranks(total_ms, dist, dev)
    ms_per_step = total_ms / args.steps
    value = SH.aggregate_throughput(B * D * N, world, ms_per_step)

    # ---- end to end: per-step inputs from pinned host memory, result read back to the host ----
    e2e = None
    if not args.no_e2e:
        # Two output buffers on the device and in pinned host memory: the read-back of step i runs on a copy stream while
        # step i + 1 computes (every step's inputs still come from the host and every step's result still reaches the host
        # inside the timed region; PCIe carries 403 MB per step, so the copy, not the kernels, sets this number).
        out_h = [torch.empty((B, D, N), dtype=torch.float32).pin_memory() for _ in range(2)]
        out_d = [out, torch.empty_like(out)]
        k2 = max(4, min(args.steps, 10))
        p_d, off_d = torch.empty_like(params), torch.empty_like(offsets)
        copy_stream = torch.cuda.Stream(device=dev)
        done_compute = [torch.cuda.Event() for _ in range(2)]
        done_copy = [torch.cuda.Event() for _ in range(2)]

        def step_e2e(i):
            j = i & 1
            p_d.copy_(params_h, non_blocking=True)
            off_d.copy_(offsets_h, non_blocking=True)
            stream.wait_event(done_copy[j])                      # buffer j was read back two steps ago
            A.amplfi_assemble_batch(plan, B, bg, strip, p_d, wl.f_lo, wl.f_hi, offsets=off_d, approximant=wl.approximant,
                                    gmst=wl.gmst, psd=psd, out=out_d[j], stream=stream)
            done_compute[j].record(stream)
            copy_stream.wait_event(done_compute[j])
            with torch.cuda.stream(copy_stream):
                out_h[j].copy_(out_d[j], non_blocking=True)
                done_copy[j].record(copy_stream)

        for j in range(2):
            done_copy[j].record(copy_stream)
        for i in range(2):
            step_e2e(i)
        barrier()
        e0.record(stream)
        for i in range(k2):
            step_e2e(i)
        stream.wait_stream(copy_stream)                          # the last read-backs are inside the timed region
        e1.record(stream)
        barrier()
        ms2 = e0.elapsed_time(e1)
        ms2 = SH.max_over_ranks(ms2, dist, dev)
        e2e = {"value": SH.aggregate_throughput(B * D * N, world, ms2 / k2), "unit": UNIT,
               "h2d_bytes_per_step": int(params_h.numel() * 8 + offsets_h.numel() * 8),
               "d2h_bytes_per_step": int(out_h[0].numel() * 4), "steps": k2, "ms_per_step": ms2 / k2}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (fused inject+whiten): 8 algorithmic bytes per output sample ----
    peak, peak_src = peaks()
    k_ms = float(np.mean(kernel_ms)) if kernel_ms else None
    alg_bytes = 8.0 * B * D * N
    traffic, lane_ops, counters_note = kernel_counters()
    roofline = None
    if k_ms:
        ach = alg_bytes / (k_ms * 1e-3) / 1e9
        # secondary ceiling: fp32 lane-operations on the FMA pipe (128 lanes/clk/SM), executed fp32
        # instructions per output sample from the ncu source page of the captured build (profiles/kernel_counters.txt)
        sm_clk = (clocks or {}).get("sm_mhz") or 1965.0
        try:
            alu_peak, alu_src = A.probe_fp32_pipe() / 1e12, "measured in this run (amplfi_probe_fp32_pipe: packed FMA loop)"
        except Exception:
            alu_peak, alu_src = 148 * 128 * sm_clk * 1e6 / 1e12, "nominal 148 SMs x 128 lanes x SM clock"
        alu = None
        if lane_ops:
            alu_ach = lane_ops * B * D * N / (k_ms * 1e-3) / 1e12
            alu = {"bound": "alu", "achieved": alu_ach, "peak": alu_peak, "unit": "T fp32 lane-op/s",
                   "frac": alu_ach / alu_peak, "lane_ops_per_sample": lane_ops, "sm_mhz": sm_clk, "peak_source": alu_src}
        roofline = {"bound": "hbm", "kernel": "v3::inject_whiten3_kernel<fused>", "achieved": ach, "peak": peak,
                    "unit": "GB/s", "frac": ach / peak, "frac_of_nominal_8TBps": ach / 8000.0, "peak_source": peak_src,
                    "traffic": traffic, "counters": counters_note, "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": k_ms,
                    "kernel_share_of_step": k_ms / ms_per_step, "launches_timed": len(kernel_ms), "alu": alu}

    # ---- the other BASELINE.json configs (configs[0], [1], [3], [4]) in the same run, after the timed region ----
    other = None
    if world == 1 and not args.no_other_configs:
        del out
        torch.cuda.empty_cache()
        other = {"c0": measure_small(A, WL, torch, dev, stream, "c0", 200),
                 "c1": measure_small(A, WL, torch, dev, stream, "c1", 200),
                 "c3": measure_c3(A, WL, torch, dev, stream, 1000),
                 "c4": measure_c4(A, WL, torch, dev, stream, 5)}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, dt, cores = time_oracle(wl, args.cpu_sample)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "cores_note": "process CPU time / wall time of the numpy oracle",
               "host_cores": os.cpu_count(), "kind": "oracle",
               "seconds": dt, "sample": "%d of %d samples (x%d detectors x %d) + the full 64 s Welch, one pass"
               % (args.cpu_sample, B, D, N)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "batch_per_gpu": B, "n_det": D, "n": N, "strip_len": int(wl.strip.shape[1]),
                       "l2_policy": "inputs larger than L2 (random 64 KB gathers from a %.0f MB strip + %.0f MB output per step)"
                       % (wl.strip.nbytes / 1e6, B * D * N * 4 / 1e6),
                       "parallelism": "batch sharded, no collective" if world > 1 else "single GPU"},
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
            "hbm_gbs_step": 8.0 * B * D * N / (ms_per_step * 1e-3) / 1e9, "other_configs": other}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()



# ------------------------------------------------------------------------------------------------
# The other BASELINE.json configs as functions (used by --config c0 | c1 | c3 | c4 and by the "other_configs" key of the
# contract line)
# ------------------------------------------------------------------------------------------------

C3_WORKLOAD = ("c3 online-latency: batch 1 x H1+L1+V1, 8 s at 2048 Hz, Welch from the 128 s preceding background (4 s Hann, "
               "50% overlap), IMRPhenomD injection; run r uses seed 0xA3D30003 + r; CUDA events around one "
               "amplfi_assemble_batch call, inputs resident")


def measure_c3(A, WL, torch, dev, stream, runs):
    """One amplfi_assemble_batch call per candidate, inputs resident; measured both as plain stream launches and as a
    replayed CUDA graph of the same call (the online service keeps its buffers in place)."""
    plan = A.Plan(16384, 2048.0, (0, 1, 2), 1, nperseg=8192)
    bg = torch.empty((3, 262144), dtype=torch.float32, device=dev)
    noise = torch.empty((1, 3, 16384), dtype=torch.float32, device=dev)
    params = torch.empty((1, 11), dtype=torch.float64, device=dev)
    psd = torch.empty((3, 4097), dtype=torch.float32, device=dev)
    out = torch.empty((1, 3, 16384), dtype=torch.float32, device=dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def call(st):
        A.amplfi_assemble_batch(plan, 1, bg, noise, params, 20.0, 1000.0, approximant=A.IMRPHENOMD, gmst=0.0,
                                psd=psd, out=out, stream=st)

    # the seeded inputs are synthesised on host threads in blocks of 125 runs BEFORE the block is timed (no host thread runs
    # beside the timed launches)
    from concurrent.futures import ThreadPoolExecutor
    pool = ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1))
    ready = {}

    def load(r):
        if r not in ready:
            ready.clear()
            block = range(r, min(r + 125, runs))
            for q, wl in zip(block, pool.map(lambda q: WL.make_c3(run=q), block)):
                ready[q] = wl
        wl = ready[r]
        bg.copy_(torch.from_numpy(wl.bg)); noise.copy_(torch.from_numpy(wl.noise)); params.copy_(torch.from_numpy(wl.params))

    load(0)
    for _ in range(3):
        call(stream)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    cs = torch.cuda.Stream()
    cs.wait_stream(stream)
    with torch.cuda.graph(graph, stream=cs):
        call(torch.cuda.current_stream())
    torch.cuda.synchronize()
    lat, lat_g = [], []
    for r in range(runs):
        load(r)
        torch.cuda.synchronize()
        e0.record(stream); call(stream); e1.record(stream)
        torch.cuda.synchronize()
        lat.append(e0.elapsed_time(e1) * 1e3)
        ref = out.clone()
        e0.record(stream); graph.replay(); e1.record(stream)
        torch.cuda.synchronize()
        lat_g.append(e0.elapsed_time(e1) * 1e3)
        assert torch.equal(ref, out)
    pool.shutdown(wait=True)
    res = []
    for name, v in (("stream launches", np.array(lat)), ("CUDA graph replay", np.array(lat_g))):
        res.append({"metric": "online PSD+whiten device latency", "unit": "us", "higher_is_better": False,
                    "launch": name, "p50": float(np.percentile(v, 50)), "p99": float(np.percentile(v, 99)),
                    "mean": float(v.mean()), "min": float(v.min()), "max": float(v.max()), "runs": len(v),
                    "dtype": "f32", "data": "synthetic", "config": {"workload": C3_WORKLOAD}})
    return res


def measure_small(A, WL, torch, dev, stream, config, runs):
    """The two small BASELINE configs: device time of one step (c0: fused inject+whiten with the analytic PSD, dense noise;
    c1: amplfi_assemble_batch with its own 64 s background), stream launches and a replayed CUDA graph."""
    wl = WL.make_c0() if config == "c0" else WL.make_c1()
    B, D, N = wl.batch, wl.n_det, wl.n
    plan = A.Plan(N, wl.fs, wl.det_ids, B, nperseg=wl.nperseg)
    noise = torch.from_numpy(wl.noise).to(dev)
    params = torch.from_numpy(wl.params).to(dev)
    out = torch.empty((B, D, N), dtype=torch.float32, device=dev)
    if config == "c0":
        psd = torch.from_numpy(wl.psd_scaled).to(dev)

        def call(st):
            A.amplfi_inject_whiten(plan, B, noise, psd, wl.f_lo, wl.f_hi, approximant=wl.approximant, params=params,
                                   gmst=wl.gmst, out=out, stream=st)
    else:
        bg = torch.from_numpy(wl.bg).to(dev)
        psd = torch.empty((D, wl.nperseg // 2 + 1), dtype=torch.float32, device=dev)

        def call(st):
            A.amplfi_assemble_batch(plan, B, bg, noise, params, wl.f_lo, wl.f_hi, approximant=wl.approximant, gmst=wl.gmst,
                                    psd=psd, out=out, stream=st)
    for _ in range(3):
        call(stream)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    cs = torch.cuda.Stream()
    cs.wait_stream(stream)
    with torch.cuda.graph(graph, stream=cs):
        call(torch.cuda.current_stream())
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    res = []
    for name, fn in (("stream launches", lambda: call(stream)), ("CUDA graph replay", graph.replay)):
        lat = []
        for _ in range(runs):
            e0.record(stream); fn(); e1.record(stream)
            torch.cuda.synchronize()
            lat.append(e0.elapsed_time(e1) * 1e3)
        v = np.array(lat)
        res.append({"metric": "device time of one step", "unit": "us", "higher_is_better": False, "launch": name,
                    "p50": float(np.percentile(v, 50)), "p99": float(np.percentile(v, 99)), "runs": len(v),
                    "samples_per_s_at_p50": B * D * N / (float(np.percentile(v, 50)) * 1e-6), "dtype": "f32",
                    "data": "synthetic", "config": {"workload": config, "batch": B, "n_det": D, "n": N}})
    return res


def measure_throughput(A, torch, dev, stream, wl, steps, warmup, kernel_time=False):
    """ms per step, samples/s and launches per step of amplfi_psd_welch + fused amplfi_inject_whiten on a strip workload
    (kernel_time: also the mean device time of the inject+whiten launches, bracketed by events inside the library)."""
    B, D, N = wl.batch, wl.n_det, wl.n
    plan = A.Plan(N, wl.fs, wl.det_ids, B, nperseg=wl.nperseg)
    strip = torch.from_numpy(wl.strip).to(dev)
    params = torch.from_numpy(wl.params).to(dev)
    offsets = torch.from_numpy(wl.offsets).to(dev)
    o, nb = wl.extra["bg_offset"], wl.extra["n_bg"]
    bg = strip[:, o:o + nb]
    psd = torch.empty((D, wl.nperseg // 2 + 1), dtype=torch.float32, device=dev)
    out = torch.empty((B, D, N), dtype=torch.float32, device=dev)

    def step():
        A.amplfi_psd_welch(plan, bg, psd=psd, stream=stream)
        A.amplfi_inject_whiten(plan, B, strip, psd, wl.f_lo, wl.f_hi, offsets=offsets, approximant=wl.approximant,
                               params=params, gmst=wl.gmst, out=out, stream=stream)
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    if kernel_time:
        plan.set_timing(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = A.launch_count()
    e0.record(stream)
    for _ in range(steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    k_ms = None
    if kernel_time:
        kt = plan.kernel_times_ms()
        plan.set_timing(False)
        k_ms = sum(kt) / len(kt) if kt else None
    assert bool(torch.isfinite(out[:: max(1, B // 16)]).all())
    sps = B * D * N / (ms * 1e-3)
    n_l = (A.launch_count() - l0) // steps
    del plan, strip, out
    torch.cuda.empty_cache()
    if kernel_time:
        return ms, sps, n_l, k_ms
    return ms, sps, n_l


C4_WORKLOAD = ("c4 bandwidth stress: batch 8192 x H1+L1+V1, fs 4096 Hz, 16 s segments (65536), gathered from a [3, 2^26] strip, "
               "Welch from 128 s (4 s Hann), IMRPhenomD")


def measure_c4(A, WL, torch, dev, stream, steps, batch=8192):
    peak, peak_src = peaks()
    wl = WL.make_c4(batch=batch)
    ms, sps, n_l, k_ms = measure_throughput(A, torch, dev, stream, wl, steps, 3, kernel_time=True)
    kernel = None
    if k_ms:
        gbs = 8.0 * wl.batch * wl.n_det * wl.n / (k_ms * 1e-3) / 1e9
        kernel = {"kernel": "v3::inject_whiten3_kernel<15, fused> (clusters of two CTAs)", "kernel_ms": k_ms, "achieved": gbs,
                  "unit": "GB/s", "frac": gbs / peak, "kernel_share_of_step": k_ms / ms}
    return {"metric": METRIC.replace("2048 Hz", "4096 Hz"), "value": sps, "unit": UNIT, "ms_per_step": ms,
            "higher_is_better": True, "dtype": "f32", "data": "synthetic", "gpu_launches_per_step": int(n_l),
            "hbm_gbs_step": 8.0 * sps / 1e9, "frac_of_measured_hbm": 8.0 * sps / 1e9 / peak, "peak_source": peak_src,
            "roofline_kernel": kernel,
            "config": {"workload": C4_WORKLOAD, "batch": batch}}

# ------------------------------------------------------------------------------------------------
# Other BASELINE.json configs: not the contract line; one JSON line per measurement
# ------------------------------------------------------------------------------------------------

def run_extra(args):
    import torch
    import paper_2407_19048_b200 as A
    import workloads as WL
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the B200 arm has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream()
    peak, peak_src = peaks()

    def throughput(wl, steps, warmup):
        return measure_throughput(A, torch, dev, stream, wl, steps, warmup)

    if args.config == "c3":
        for d in measure_c3(A, WL, torch, dev, stream, args.runs):
            print(json.dumps(d))
        return

    if args.config in ("c0", "c1"):
        for d in measure_small(A, WL, torch, dev, stream, args.config, args.runs):
            print(json.dumps(d))
        return

    if args.config == "next":
        # SURVEY.md 8(f) rows on the c2 workload: two data views, time-domain waveforms, median Welch, truncated filter
        wl = WL.make_c2(batch=args.batch, strip_len=args.strip_len)
        B, D, N = wl.batch, wl.n_det, wl.n
        plan = A.Plan(N, wl.fs, wl.det_ids, B, nperseg=wl.nperseg)
        strip = torch.from_numpy(wl.strip).to(dev)
        params = torch.from_numpy(wl.params).to(dev)
        offsets = torch.from_numpy(wl.offsets).to(dev)
        t_shift = torch.from_numpy(np.random.Generator(np.random.Philox(5)).uniform(0.0, 1.0, B)).to(dev)
        o, nb = wl.extra["bg_offset"], wl.extra["n_bg"]
        bg = strip[:, o:o + nb]
        psd = torch.empty((D, wl.nperseg // 2 + 1), dtype=torch.float32, device=dev)
        out = torch.empty((B, D, N), dtype=torch.float32, device=dev)
        out2 = torch.empty((B, D, N), dtype=torch.float32, device=dev)
        h_t = torch.empty((B, 2, N), dtype=torch.float32, device=dev)
        fdur = 1.0
        out_c = torch.empty((B, D, N - int(fdur * wl.fs)), dtype=torch.float32, device=dev)
        A.amplfi_psd_welch(plan, bg, psd=psd, stream=stream)

        def timed(fn, steps=max(5, min(args.steps, 50)), warmup=3):
            for _ in range(warmup):
                fn()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l0 = A.launch_count()
            e0.record(stream)
            for _ in range(steps):
                fn()
            e1.record(stream)
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / steps, (A.launch_count() - l0) // steps

        rows = []
        ms, nl = timed(lambda: A.amplfi_inject_whiten(plan, B, strip, psd, wl.f_lo, wl.f_hi, offsets=offsets, params=params,
                                                      gmst=wl.gmst, out=out, stream=stream))
        rows.append(("amplfi_inject_whiten (fused, one view; reference point)", ms, nl, B * D * N, 8.0 * B * D * N))
        ms, nl = timed(lambda: A.amplfi_inject_whiten_views(plan, B, strip, psd, wl.f_lo, wl.f_hi, params, t_shift, offsets=offsets,
                                                            gmst=wl.gmst, out=out, out2=out2, stream=stream))
        rows.append(("amplfi_inject_whiten_views (two views d, d')", ms, nl, 2 * B * D * N, 12.0 * B * D * N))
        ms, nl = timed(lambda: A.amplfi_waveform_td(plan, A.IMRPHENOMD, params, wl.f_lo, wl.f_hi, h_t=h_t, stream=stream))
        rows.append(("amplfi_waveform_td (h+, hx time series)", ms, nl, 2 * B * N, 4.0 * 2 * B * N))
        ms, nl = timed(lambda: A.amplfi_inject_whiten_fir(plan, B, strip, psd, wl.f_lo, wl.f_hi, fdur, crop=True, offsets=offsets,
                                                          params=params, gmst=wl.gmst, out=out_c, stream=stream))
        rows.append(("amplfi_inject_whiten_fir (1 s filter, cropped)", ms, nl, B * D * N, 4.0 * B * D * (2 * N - int(fdur * wl.fs))))
        ms, nl = timed(lambda: A.amplfi_psd_welch(plan, bg, psd=psd, stream=stream))
        rows.append(("amplfi_psd_welch average=mean (64 s, 63 segments x 3)", ms, nl, 3 * nb, 4.0 * 3 * nb))
        ms, nl = timed(lambda: A.amplfi_psd_welch(plan, bg, average=1, psd=psd, stream=stream))
        rows.append(("amplfi_psd_welch average=median", ms, nl, 3 * nb, 4.0 * 3 * nb))
        hp = torch.empty((B, N // 2 + 1, 2), dtype=torch.float32, device=dev)
        hc = torch.empty_like(hp)
        fl = torch.empty((B,), dtype=torch.int32, device=dev)
        ms, nl = timed(lambda: A.amplfi_waveform_fd(plan, A.IMRPHENOMD, params, wl.f_lo, wl.f_hi, hp=hp, hc=hc, flags=fl, stream=stream))
        rows.append(("amplfi_waveform_fd (IMRPhenomD h+, hx materialised; %.3g waveforms/s; the paper: 1000 in ~0.15 s on an A40, "
                     "PAPER.md:104)" % (B / (ms * 1e-3)), ms, nl, 2 * B * (N // 2 + 1), 16.0 * B * (N // 2 + 1)))
        for name, ms, nl, samples, alg_bytes in rows:
            print(json.dumps({"metric": "8(f) rows on the c2 workload", "call": name, "ms_per_call": ms, "gpu_launches_per_call": int(nl),
                              "samples_per_s": samples / (ms * 1e-3), "algorithmic_gbs": alg_bytes / (ms * 1e-3) / 1e9,
                              "frac_of_measured_hbm": alg_bytes / (ms * 1e-3) / 1e9 / peak, "dtype": "f32", "data": "synthetic",
                              "config": {"batch": B, "n_det": D, "n": N}}))
        return

    if args.config == "c4":
        print(json.dumps(measure_c4(A, WL, torch, dev, stream, max(3, min(args.steps, 10)))))
        return

    # sweep: fixed total samples (2^27 per detector), segment length 1..256 s at 4096 Hz (n = 2^12 .. 2^20)
    for t_seg in (1.0, 2.0, 4.0, 8.0, 16.0, 32.0, 64.0, 128.0, 256.0):
        n = int(t_seg * 4096)
        batch = (1 << 27) // n
        wl = WL.make_c4(batch=batch, t_seg=t_seg)
        wl.nperseg = min(wl.nperseg, n)                              # Welch window no longer than the segment
        ms, sps, n_l = throughput(wl, max(3, min(args.steps, 10)), 3)
        flops = 2 * 2.5 * n * np.log2(n) * batch * 3                  # forward + inverse real transforms
        print(json.dumps({"metric": "segment-length sweep", "t_seg": t_seg, "n": n, "batch": batch, "value": sps, "unit": UNIT,
                          "ms_per_step": ms, "hbm_gbs_step": 8.0 * sps / 1e9, "frac_of_measured_hbm": 8.0 * sps / 1e9 / peak,
                          "fft_gflops": flops / (ms * 1e-3) / 1e9, "gpu_launches_per_step": int(n_l), "dtype": "f32",
                          "data": "synthetic"}))


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` with N > 1 and no launcher: start N ranks (one per GPU) under torch.distributed.run on
    this node and let them run this same command line.  Returns the launcher's exit code."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                  # the communicator line shows the ranks and the transport
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


if __name__ == "__main__":
    a = parse()
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ and a.config == "c2":
        sys.exit(respawn_under_torchrun(a))
    if a.impl == "reference":
        run_reference(a)
    elif a.config != "c2":
        run_extra(a)
    else:
        run_b200(a)
