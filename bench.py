#!/usr/bin/env python
"""bench.py -- X-engine throughput on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg3] [--impl reference]

A "step" is one pass of the whole hot path (S1 unpack/stage, S2 tile schedule, S3 tensor-core
cross-multiply, S4 span-accumulate) over one batch of synthetic input: all spans of the config,
the first with accumulate=0 and the rest accumulating into the persistent visibility buffer.
Default workload: BASELINE.json configs[2] ("cfg3": 512 inputs, 3072 channels, 1024 samples, ci8,
2 spans) -- the 512-input ci8 station config the north_star's target is quoted on.

value       useful int8 TOPS = 8 * ntime * nchan * nbaselines * nspans / time, inputs resident in HBM
e2e         same metric through bfXcorrExecuteHost: pinned HOST spans copied in and the visibility
            buffer copied back inside the timed region
roofline    dominant kernel (the only kernel): algorithmic ops (and bytes) per launch / mean launch
            duration from CUDA events on the launching stream, against MEASURED_PEAKS.json
            roofline.same_mix_peak: what a no-math streaming kernel with the step's read : write mix
            (bfXcorrMemoryProbe) reaches in the same run -- the HBM ceiling of this access mix on this box
cpu_baseline the CPU oracle (oracle/, as it stands) timed on this box's host cores on a bounded
            sample of the same workload -- a baseline, not the target; one_thread: its per-core rate
parity      the buffer the TIMED launches left behind, compared bit for bit with the oracle on the
            channels the cpu_baseline leg computed
ms_per_step mean over the timed region; ms_per_step_median / _min: per-step sums of the launch durations
sustained   the same step back to back for >= 1 s with its own clock record (the default timed region
            ends before the board reaches its power cap)
N > 1       channels are independent: every rank runs the same per-GPU workload on
            its own GPU with no collective on the data path ("weak" scaling); time = max over ranks.
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

METRIC = "X-engine int8 TOPS (useful ops: 8 per complex MAC, lower triangle incl. autos)"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": float(p["hbm_gbs"]), "bf16_burst": float(p["bf16_tflops"]),
                "bf16_sustained": float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), "source": "measured"}
    # fallback stated in the B200 profiling recipe
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """SM clock, power and clock-event (throttle) reasons sampled DURING the timed region.

    NVML is polled in-process every ~2 ms by a thread that is initialised in the constructor, so the first sample
    falls inside the timed region even when that lasts only tens of milliseconds; `nvidia-smi -lms 50` (which
    needs ~100 ms to come up) is the fallback when pynvml cannot be used."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, gpu_index: int):
        self.rows = []        # nvidia-smi fallback: csv lines
        self.samples = []     # NVML: (sm_mhz, power_w, reason_mask)
        self.proc = None
        self.gpu = gpu_index
        self.nvml = None
        self.handle = None
        self.sm_max = None
        self.stop_flag = threading.Event()
        self.thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            try:
                import torch
                uuid = str(torch.cuda.get_device_properties(gpu_index).uuid)
                if not uuid.startswith("GPU-"):
                    uuid = "GPU-" + uuid
                self.handle = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                self.handle = pynvml.nvmlDeviceGetHandleByIndex(gpu_index)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self._poll_once(pynvml)   # fails here, not in the thread, if a query is unsupported
            self.samples.clear()
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def _poll_once(self, nv):
        sm = float(nv.nvmlDeviceGetClockInfo(self.handle, nv.NVML_CLOCK_SM))
        pw = nv.nvmlDeviceGetPowerUsage(self.handle) / 1000.0
        try:
            mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
        except Exception:
            mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
        self.samples.append((sm, pw, mask))

    def _poll(self):
        nv = self.nvml
        while not self.stop_flag.is_set():
            try:
                self._poll_once(nv)
            except Exception:
                break
            time.sleep(0.002)

    def start(self):
        if self.nvml is not None:
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def _stop_nvml(self):
        self.stop_flag.set()
        self.thread.join(timeout=2)
        nv = self.nvml
        bits = [(nv.nvmlClocksThrottleReasonHwSlowdown, "hw_slowdown"),
                (nv.nvmlClocksThrottleReasonHwThermalSlowdown, "hw_thermal_slowdown"),
                (nv.nvmlClocksThrottleReasonSwThermalSlowdown, "sw_thermal_slowdown"),
                (nv.nvmlClocksThrottleReasonSwPowerCap, "sw_power_cap")]
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["no samples"]}
        sm_sorted = sorted(s[0] for s in self.samples)
        reasons = sorted({name for _, _, m in self.samples for bit, name in bits if m & int(bit)})
        return {"sm_mhz": sm_sorted[len(sm_sorted) // 2], "sm_min_mhz": sm_sorted[0], "sm_max_mhz": self.sm_max,
                "power_w_max": max(s[1] for s in self.samples), "samples": len(self.samples), "reasons": reasons,
                "source": "nvml, polled every ~2 ms inside the timed region"}

    def stop(self):
        if self.nvml is not None and self.thread is not None:
            return self._stop_nvml()
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(self.NAMES, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm_sorted = sorted(sm)
        return {"sm_mhz": sm_sorted[len(sm_sorted) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons), "source": "nvidia-smi -lms 50"}


def workload_numbers(cfg):
    nb = cfg.nbaselines
    ops_span = 8.0 * cfg.ntime * cfg.nchan * nb
    samples_span = float(cfg.ntime) * cfg.nchan * cfg.ninputs
    in_bytes = float(cfg.span_bytes)
    out_bytes = float(cfg.out_bytes)
    # algorithmic bytes: span read once, visibilities written once (+ read once when accumulating)
    bytes_all = cfg.nspans * in_bytes + out_bytes + (cfg.nspans - 1) * 2 * out_bytes
    return dict(ops_span=ops_span, samples_span=samples_span, in_bytes=in_bytes, out_bytes=out_bytes,
                ops_step=ops_span * cfg.nspans, samples_step=samples_span * cfg.nspans, bytes_step=bytes_all)


def config_dict(cfg, extra=None):
    d = {"workload": "%s: %d inputs x %d channels x %d samples, ci%d, %d span(s) per step (BASELINE.json configs[%d])" % (
        cfg.name, cfg.ninputs, cfg.nchan, cfg.ntime, cfg.dtype, cfg.nspans, int(cfg.name[3:]) - 1),
        "ninputs": cfg.ninputs, "nchan": cfg.nchan, "ntime": cfg.ntime, "dtype": "ci%d" % cfg.dtype,
        "nspans": cfg.nspans, "seed": cfg.seed}
    if extra:
        d.update(extra)
    return d


def spaced_channels(nchan: int, n: int):
    return sorted(set(int(round(k * (nchan - 1) / max(1, n - 1))) for k in range(n))) if n > 1 else [0]


# the oracle legs' input: at most this many bytes of span per sampled slab (the seeded generator works in int64 temporaries,
# a dozen bytes per sample while it runs; cfg5 has 16384 cheap channels and the sample would otherwise grow to the whole span)
ORACLE_SAMPLE_MAX_BYTES = 1 << 30


def channel_slab_numpy(cfg, span: int, chans):
    """generate_channel_slab in channel chunks of <= 32 Mi samples (on the GPU when there is one), as one numpy array."""
    import numpy as np
    import torch
    from xcorr_inputs import generate_channel_slab
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    per = max(1, (32 << 20) // (cfg.ntime * cfg.ninputs))
    parts = [generate_channel_slab(cfg, span, chans[a:a + per], device=dev).cpu().numpy() for a in range(0, len(chans), per)]
    return parts[0] if len(parts) == 1 else np.concatenate(parts, axis=1)


def oracle_sample(cfg, target_s: float):
    """Time the oracle (as it stands) on a bounded channel subset of the workload, all spans accumulated.
    Returns (seconds, channels, threads, oracle result [len(channels)][B][2], one-thread info)."""
    import oracle
    from xcorr_inputs import generate_channel_slab
    nthreads = oracle.threads()
    # calibration: one channel per thread, one span
    chans = spaced_channels(cfg.nchan, min(cfg.nchan, nthreads))
    x = channel_slab_numpy(cfg, 0, chans)
    t0 = time.perf_counter()
    oracle.xcorr(x, cfg.ninputs, len(chans), cfg.ntime, cfg.dtype)
    tcal = time.perf_counter() - t0
    per_wave = tcal / len(chans) * min(len(chans), nthreads)  # seconds of one "wave" of nthreads channels, one span
    waves = max(1, int(target_s / max(per_wave * cfg.nspans, 1e-9)))
    cap = max(nthreads, ORACLE_SAMPLE_MAX_BYTES // (cfg.ntime * cfg.ninputs * cfg.bytes_per_sample))
    chans = spaced_channels(cfg.nchan, min(cfg.nchan, waves * nthreads, cap))
    slabs = [channel_slab_numpy(cfg, s, chans) for s in range(cfg.nspans)]
    t0 = time.perf_counter()
    out = oracle.xcorr(slabs[0], cfg.ninputs, len(chans), cfg.ntime, cfg.dtype)
    for s in range(1, cfg.nspans):
        oracle.xcorr(slabs[s], cfg.ninputs, len(chans), cfg.ntime, cfg.dtype, out=out, accumulate=True)
    dt = time.perf_counter() - t0
    # per-core rate: the same oracle on one thread, one channel, one span
    one = None
    try:
        oracle.set_threads(1)
        x1 = slabs[0][:, :1].copy()
        t0 = time.perf_counter()
        oracle.xcorr(x1, cfg.ninputs, 1, cfg.ntime, cfg.dtype)
        d1 = time.perf_counter() - t0
        one = {"value": 8.0 * cfg.ntime * cfg.nbaselines / d1 / 1e12, "unit": "TOPS", "cores": 1,
               "sample": "1 channel, 1 span; %.3f s" % d1}
    finally:
        oracle.set_threads(nthreads)
    return dt, chans, nthreads, out, one


def run_reference(args, cfg):
    """--impl reference: the CPU oracle as the reference arm (there is no reference implementation
    of this path: /root/reference holds only the paper).  Each step = a bounded channel subset."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from xcorr_inputs import generate_channel_slab
    nthreads = oracle.threads()
    wl = workload_numbers(cfg)
    nch = min(cfg.nchan, max(1, nthreads))
    chans = sorted(set(int(round(k * (cfg.nchan - 1) / max(1, nch - 1))) for k in range(nch))) if nch > 1 else [0]
    slabs = [generate_channel_slab(cfg, s, chans).numpy() for s in range(cfg.nspans)]

    def step():
        out = oracle.xcorr(slabs[0], cfg.ninputs, len(chans), cfg.ntime, cfg.dtype)
        for s in range(1, cfg.nspans):
            oracle.xcorr(slabs[s], cfg.ninputs, len(chans), cfg.ntime, cfg.dtype, out=out, accumulate=True)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    frac = len(chans) / cfg.nchan
    tops = wl["ops_step"] * frac / dt / 1e12
    sample = "%d of %d channels (evenly spaced), all %d span(s), full ntime and ninputs, per step" % (
        len(chans), cfg.nchan, cfg.nspans)
    line = {"impl": "reference", "metric": METRIC, "value": tops, "unit": "TOPS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int8 x int8 -> int32", "data": "synthetic",
            "config": config_dict(cfg, {"sample": sample}),
            "samples_per_s": wl["samples_step"] * frac / dt,
            "cpu_baseline": {"value": tops, "unit": "TOPS", "cores": nthreads, "kind": "oracle", "sample": sample},
            "e2e": {"value": tops, "unit": "TOPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_beamform(args, cfg):
    """Second workload on the same spans (include/bfbeamform.h): one step = every span of the config beamformed once."""
    import numpy as np
    import torch
    import oracle
    import paper_1708_00720_b200 as bfx
    from xcorr_inputs import generate_channel_slab, generate_span, generate_weights
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the beamformer has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    K, N, C, T = args.nbeam, cfg.ninputs, cfg.nchan, cfg.ntime
    peaks = load_peaks()
    spans = [generate_span(cfg, s, device=dev) for s in range(cfg.nspans)]
    w = generate_weights(cfg.seed, C, K, N, device=dev)
    out = torch.empty((T, C, K, 2), dtype=torch.int32, device=dev)
    plan = bfx.bfBeamformCreate(N, C, T, K, cfg.dtype)
    stream = torch.cuda.current_stream()
    bfx.bfBeamformSetWeights(plan, w.data_ptr(), stream.cuda_stream)
    flush = None if cfg.span_bytes * cfg.nspans > 126e6 else torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step(rec=None):
        for s in range(cfg.nspans):
            if flush is not None:
                flush.zero_()
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            bfx.bfBeamformExecute(plan, spans[s].data_ptr(), out.data_ptr(), stream.cuda_stream)
            e1.record(stream)
            if rec is not None:
                rec.append((e0, e1))

    sampler = ClockSampler(0)
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler.start()
    rec = []
    for _ in range(args.steps):
        step(rec)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    launch_ms = [a.elapsed_time(b) for a, b in rec]
    t_launch = sum(launch_ms) / len(launch_ms) * 1e-3
    ms_per_step = t_launch * 1e3 * cfg.nspans       # kernel time only: an L2 flush (if any) sits between launches
    bfx.bfBeamformDestroy(plan)
    bytes_launch = float(cfg.span_bytes) + float(out.numel() * 4) + 4.0 * C * K * N   # span + beams + int8 weight rows, once each
    samples = float(T) * C * N
    roofline = {"bound": "hbm", "achieved": bytes_launch / t_launch / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "traffic": None, "kernel": "beamform_kernel", "algorithmic_bytes_per_launch": bytes_launch,
                "peak_source": peaks["source"]}
    roofline["frac"] = roofline["achieved"] / roofline["peak"]
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            tr = json.load(f).get("beamform_%s_k%d" % (cfg.name, K))
        if tr:
            roofline["traffic"] = tr["dram_bytes_per_launch"]
            roofline["traffic_source"] = tr["source"]
    except (OSError, ValueError, KeyError):
        pass
    cpu = None
    if not args.no_cpu_baseline:
        nthreads = oracle.threads()
        per_chan_macs = float(T) * K * N
        nch = int(max(1, min(C, args.cpu_seconds * 2.0e8 * nthreads / per_chan_macs,   # ~2e8 complex MAC/s/thread
                             max(nthreads, ORACLE_SAMPLE_MAX_BYTES // (T * N * cfg.bytes_per_sample)))))
        chans = sorted(set(int(round(k * (C - 1) / max(1, nch - 1))) for k in range(nch))) if nch > 1 else [0]
        xs = channel_slab_numpy(cfg, 0, chans)
        ws = generate_weights(cfg.seed, C, K, N, channels=chans).numpy()
        t0 = time.perf_counter()
        oracle.beamform(xs, ws, N, len(chans), T, K, cfg.dtype)
        dt = time.perf_counter() - t0
        cpu = {"value": samples * len(chans) / C / dt, "unit": "complex samples/s", "cores": nthreads, "kind": "oracle",
               "sample": "%d of %d channels (evenly spaced), one span, all samples and beams; %.1f s" % (len(chans), C, dt)}
    line = {"metric": "beamformer input rate (complex samples/s, %d beams)" % K, "value": samples / t_launch,
            "unit": "complex samples/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int8 x int8 -> int32", "data": "synthetic",
            "config": config_dict(cfg, {"op": "beamform", "nbeam": K,
                                        "l2": "inputs_exceed_l2" if flush is None else "l2_flushed_between_launches"}),
            "tops": 8.0 * samples * K / t_launch / 1e12, "clocks": clocks, "e2e": None,
            "gpu_launches": len(rec), "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg3", help="cfg1..cfg5 (BASELINE.json configs[0..4])")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--algo", default="tcgen05", choices=["tcgen05", "simt", "gauss3"],
                    help="tcgen05: the product path; simt: the CUDA-core cross-check kernel; gauss3: the three-multiplication ci4 variant")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--e2e-steps", type=int, default=8, help="steps of the end-to-end leg (enough that pipeline fill and drain do not dominate)")
    ap.add_argument("--sustain-seconds", type=float, default=1.0, help="length of the sustained run reported as `sustained` (0 = skip)")
    ap.add_argument("--no-probe", action="store_true", help="skip the same-mix memory probe")
    ap.add_argument("--op", default="xcorr", choices=["xcorr", "beamform"],
                    help="xcorr: the hot path (the driver's line); beamform: the second workload on the same spans "
                         "(SURVEY.md 8f N1), 1 GPU, its own JSON line")
    ap.add_argument("--nbeam", type=int, default=32)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    from xcorr_inputs import CONFIGS, generate_span
    cfg = CONFIGS[args.config]
    if args.op == "beamform":
        run_beamform(args, cfg)
        return
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    # --gpus N without a launcher: start the N ranks here (one process per GPU, torch.distributed.run does the
    # rendezvous on 127.0.0.1); under torchrun the environment already carries RANK / WORLD_SIZE
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))

    import torch
    import paper_1708_00720_b200 as bfx

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the X-engine has no CPU fallback")
    if world != args.gpus:
        raise SystemExit("bench.py --gpus %d was started with WORLD_SIZE=%d" % (args.gpus, world))
    if local_rank >= torch.cuda.device_count():
        raise SystemExit("bench.py: rank %d has no GPU (%d visible)" % (local_rank, torch.cuda.device_count()))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    wl = workload_numbers(cfg)
    peaks = load_peaks()
    algo = {"tcgen05": bfx.BF_XCORR_ALGO_TCGEN05, "simt": bfx.BF_XCORR_ALGO_SIMT, "gauss3": bfx.BF_XCORR_ALGO_TCGEN05_GAUSS3}[args.algo]

    # ---- synthetic spans, resident in HBM (every rank holds one full per-GPU workload: a channel shard)
    spans = [generate_span(cfg, s, device=dev) for s in range(cfg.nspans)]
    out = torch.empty((cfg.nchan, cfg.nbaselines, 2), dtype=torch.int32, device=dev)
    plan = bfx.bfXcorrCreate(cfg.ninputs, cfg.nchan, cfg.ntime, cfg.dtype)
    bfx.bfXcorrSetAlgo(plan, algo)
    stream = torch.cuda.current_stream()
    sptr = stream.cuda_stream
    launches = 0

    def step(record=None):
        nonlocal launches
        for s in range(cfg.nspans):
            if record is not None:
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
            bfx.bfXcorrExecute(plan, spans[s].data_ptr(), out.data_ptr(), s > 0, sptr)
            launches += bfx.bfXcorrGetLaunchCount(plan)
            if record is not None:
                e1.record(stream)
                record.append((s, e0, e1))

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    def max_over_ranks(v):
        if dist is None:
            return v
        t = torch.tensor([v], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    sampler = ClockSampler(local_rank) if rank == 0 else None   # NVML comes up here, outside the timed region
    for _ in range(args.warmup):
        step()
    barrier()
    if rank == 0:
        sampler.start()
    launches = 0
    rec = []
    t_begin = torch.cuda.Event(enable_timing=True); t_end = torch.cuda.Event(enable_timing=True)
    t_begin.record(stream)
    for _ in range(args.steps):
        step(rec)
    t_end.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over_ranks(t_begin.elapsed_time(t_end))
    ms_per_step = total_ms / args.steps
    per_span_ms = {}
    for s, e0, e1 in rec:
        per_span_ms.setdefault(s, []).append(e0.elapsed_time(e1))
    launch_ms = [sum(v) / len(v) for _, v in sorted(per_span_ms.items())]
    mean_launch_ms = sum(sum(v) for v in per_span_ms.values()) / max(1, sum(len(v) for v in per_span_ms.values()))
    # per-step kernel time (sum over the step's launches), for the median / min (>= 20 repetitions)
    step_ms = sorted(sum(per_span_ms[s][k] for s in per_span_ms) for k in range(args.steps))
    timed_launches = launches
    kernel_names = sorted({bfx.bfXcorrGetKernelName(plan, s > 0) for s in range(cfg.nspans)})

    # ---- parity on the TIMED kernel's output: `out` now holds the last timed step (all spans accumulated)
    parity, cpu = None, None
    if rank == 0 and not args.no_cpu_baseline:
        dt, chans, nthreads, exp, one = oracle_sample(cfg, args.cpu_seconds)
        frac = len(chans) / cfg.nchan
        got = out[torch.tensor(chans, device=dev)].cpu()
        equal = bool(torch.equal(got, torch.from_numpy(exp)))
        parity = {"channels": len(chans), "of": cfg.nchan, "equal": equal,
                  "what": "every visibility of the sampled channels after the last timed step, bit for bit against the oracle"}
        cpu = {"value": wl["ops_step"] * frac / dt / 1e12, "unit": "TOPS", "cores": nthreads, "kind": "oracle",
               "sample": "%d of %d channels (evenly spaced), all %d span(s), full ntime and ninputs; %.1f s" % (
                   len(chans), cfg.nchan, cfg.nspans, dt),
               "samples_per_s": wl["samples_step"] * frac / dt, "one_thread": one}
        del got, exp

    # ---- sustained: the same step back to back for >= sustain seconds, with its own clock record
    sustained = None
    if args.sustain_seconds > 0:
        n_sus = max(args.steps, int(args.sustain_seconds * 1e3 / ms_per_step) + 1)
        s_sampler = ClockSampler(local_rank) if rank == 0 else None
        barrier()
        if rank == 0:
            s_sampler.start()
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(n_sus):
            step()
        b.record(stream)
        barrier()
        s_clocks = s_sampler.stop() if rank == 0 else None
        s_ms = max_over_ranks(a.elapsed_time(b)) / n_sus
        sustained = {"value": wl["ops_step"] * world / (s_ms * 1e-3) / 1e12, "unit": "TOPS", "ms_per_step": s_ms,
                     "steps": n_sus, "clocks": s_clocks}

    # ---- the same-mix HBM ceiling: a no-math streaming kernel moving the step's algorithmic bytes
    same_mix = None
    if rank == 0 and not args.no_probe:
        probe_ms = []
        for s in range(cfg.nspans):
            ts = []
            for k in range(5):
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                bfx.bfXcorrMemoryProbe(plan, spans[s].data_ptr(), out.data_ptr(), s > 0, sptr)
                e1.record(stream)
                torch.cuda.synchronize()
                if k >= 2:
                    ts.append(e0.elapsed_time(e1))
            probe_ms.append(sum(ts) / len(ts))
        same_mix = {"gbs": wl["bytes_step"] / (sum(probe_ms) * 1e-3) / 1e9, "launch_ms": probe_ms,
                    "kernel": "mem_probe_kernel (reads the span, writes / read-modify-writes the visibilities, no math)"}
    barrier()

    # ---- end to end through the host-buffer entry point
    e2e = None
    if not args.no_e2e:
        try:
            host_spans = [torch.empty(cfg.span_bytes, dtype=torch.uint8, pin_memory=True) for _ in range(cfg.nspans)]
            for h, d in zip(host_spans, spans):
                h.copy_(d.reshape(-1))
            host_out = torch.empty((cfg.nchan, cfg.nbaselines, 2), dtype=torch.int32, pin_memory=True)
            torch.cuda.synchronize()

            def e2e_step():
                for s in range(cfg.nspans):
                    last = s == cfg.nspans - 1
                    bfx.bfXcorrExecuteHost(plan, host_spans[s].data_ptr(), out.data_ptr(),
                                           host_out.data_ptr() if last else 0, s > 0, sptr)

            e2e_step()
            barrier()
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for _ in range(args.e2e_steps):
                e2e_step()
            b.record(stream)
            barrier()
            e_ms = max_over_ranks(a.elapsed_time(b)) / args.e2e_steps
            e2e = {"value": wl["ops_step"] * world / (e_ms * 1e-3) / 1e12, "unit": "TOPS",
                   "h2d_bytes_per_step": int(cfg.span_bytes * cfg.nspans), "d2h_bytes_per_step": int(cfg.out_bytes),
                   "ms_per_step": e_ms, "steps": args.e2e_steps,
                   "samples_per_s": wl["samples_step"] * world / (e_ms * 1e-3),
                   "api": "bfXcorrExecuteHost (pinned host spans in, visibility buffer out after the last span)"}
            del host_spans, host_out
        except RuntimeError as ex:  # pinned allocation refused, etc.
            e2e = {"value": None, "unit": "TOPS", "error": str(ex)[:200]}

    bfx.bfXcorrDestroy(plan)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    value = wl["ops_step"] * world / (ms_per_step * 1e-3) / 1e12
    # ---- roofline of the (only) kernel, per launch, averaged over the spans of a step
    ops_launch = wl["ops_span"]
    bytes_launch = wl["bytes_step"] / cfg.nspans
    t_launch = mean_launch_ms * 1e-3
    long_region = total_ms > 1000.0
    bf16_peak = peaks["bf16_sustained"] if long_region else peaks["bf16_burst"]
    int8_peak = 2.0 * bf16_peak  # guide's nominal int8:bf16 dense ratio (4.5 : 2.25 PFLOP/s)
    tensor = {"bound": "tensor", "achieved": ops_launch / t_launch / 1e12, "peak": int8_peak, "unit": "TOPS"}
    tensor["frac"] = tensor["achieved"] / tensor["peak"]
    hbm = {"bound": "hbm", "achieved": bytes_launch / t_launch / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s"}
    hbm["frac"] = hbm["achieved"] / hbm["peak"]
    main_r, alt_r = (tensor, hbm) if tensor["frac"] >= hbm["frac"] else (hbm, tensor)
    roofline = dict(main_r)
    # DRAM traffic of the same kernel on the same workload from the committed ncu capture (profiles/), per launch
    roofline["traffic"] = None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            tr = json.load(f).get(cfg.name)
        if tr and args.algo == "tcgen05":
            roofline["traffic"] = tr["dram_bytes_per_launch"]
            roofline["traffic_source"] = tr["source"]
    except (OSError, ValueError, KeyError):
        pass
    roofline["peak_source"] = "%s (%s; int8 = 2 x bf16 %s)" % (
        peaks["source"], "MEASURED_PEAKS.json" if peaks["source"] == "measured" else "B200_PROFILING.md fallback",
        "sustained" if long_region else "burst")
    roofline["kernel"] = "; ".join(kernel_names)   # bfXcorrGetKernelName: the dispatch rule lives in the library
    # context: tcgen05.mma kind::i8 issue-rate probe on this pool (profiles/round1.md): 8192 MAC/clk/SM -> 4.6 POPS at 1.9 GHz
    roofline["int8_mma_probe_peak_tops"] = 4610.0
    roofline["launch_ms"] = launch_ms
    roofline["algorithmic_ops_per_launch"] = ops_launch
    roofline["algorithmic_bytes_per_launch"] = bytes_launch
    roofline["other_bound"] = alt_r
    roofline["frac_of_nominal_int8_4500"] = tensor["achieved"] / 4500.0
    if same_mix is not None:
        # what a no-math kernel with the same read : write mix reaches on this box in this run, beside the copy peak
        roofline["same_mix_peak"] = same_mix["gbs"]
        roofline["same_mix_frac"] = hbm["achieved"] / same_mix["gbs"]
        roofline["same_mix_probe"] = same_mix

    line = {"metric": METRIC, "value": value, "unit": "TOPS", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int8 x int8 -> int32", "data": "synthetic",
            "config": config_dict(cfg, {"l2": "inputs_exceed_l2" if cfg.span_bytes * cfg.nspans > 126e6 else
                                        "inputs_fit_l2 (latency-bound tiny case)",
                                        "parallelism": "channels sharded, no collective" if world > 1 else "1 gpu",
                                        "algo": args.algo}),
            "samples_per_s": wl["samples_step"] * world / (ms_per_step * 1e-3),
            "ms_per_step_median": step_ms[len(step_ms) // 2], "ms_per_step_min": step_ms[0],
            "clocks": clocks, "e2e": e2e, "gpu_launches": timed_launches, "roofline": roofline,
            "cpu_baseline": cpu, "parity": parity, "sustained": sustained}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
