"""bench.py -- one JSON line per run (contract in DESIGN.md "Measurement").

A "step" is one pass of the whole hot path (a1-a10, one chime_bf_execute) over one batch of
synthetic CHIME-shaped baseband.  Default: one channel group of BASELINE.json configs[3] per GPU (128 coarse
channels x 49152 samples x 2048 inputs = 12.9 GB in, 268 MB out, device-resident); --workload cfg1 = configs[1]
(4 channels, 403 MB).  metric = input baseband GB/s (and, beside it, the number of coarse channels that rate
sustains in real time, 1 channel = 0.8 GB/s).

  python bench.py [--gpus N] [--steps K] [--warmup W]          CUDA arm (configs[3] channel group)
  python bench.py --workload cfg1                              CUDA arm on configs[1]
  python bench.py --impl reference ...                         oracle arm (CPU, bounded sample)
  python bench.py --workload cfg3 [--chunks 80]                full-band streaming (configs[3]), 1 GPU
  python bench.py --workload dedisp                            dedispersion kernel (HBM-bound), 1 GPU
"""
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

METRIC = "input baseband GB/s and coarse channels sustained in real time per B200"
UNIT = "GB/s"
BYTES_PER_CHAN_SAMPLE = 2048.0
REALTIME_SAMPLES_PER_S = 390625.0                 # 1 / 2.56 us  (Table 1)
GBS_PER_CHANNEL = BYTES_PER_CHAN_SAMPLE * REALTIME_SAMPLES_PER_S / 1e9   # 0.8 GB/s
# Nominal flops per (channel, sample): FFTs only / everything.
FFT_FLOPS = 256000.0
ALL_FLOPS = 342016.0
# FP32 peak: 148 SMs x 128 lanes x 2 flop x sm clock (DESIGN.md derives it; clock from MEASURED_PEAKS).
N_SM, LANES = 148, 128


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            p = [x.strip() for x in r.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for n, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(n_cells, seed_cfg=1):
    """Times the oracle, as it stands, on n_cells output cells (1 cell = 1 channel x 384 samples) of the
    configs[1] workload.  Returns (seconds, chan_samples, cores)."""
    import numpy as np
    import oracle
    import synth
    oracle.build()
    cfg = synth.CONFIGS[seed_cfg]
    C, T = cfg["n_coarse"], cfg["n_time"]
    seed = synth.config_seed(seed_cfg)
    freqs = synth.config_freqs(seed_cfg)
    gains = synth.gains(seed, C, flagged_frac=cfg["flagged"])
    rng = np.random.default_rng(seed)
    cells = [(int(rng.integers(C)), int(rng.integers(T // 384))) for _ in range(n_cells)]
    blocks = [synth.noise_bytes(seed, 1, 384, chan0=c, time0=384 * R, n_time_total=T).numpy()[0]
              for (c, R) in cells]
    t0 = time.perf_counter()
    for (c, R), blk in zip(cells, blocks):
        I, _ = oracle.cell(blk, float(freqs[c]), gains=gains[c])
        oracle.quantize(I)
    dt = time.perf_counter() - t0
    return dt, n_cells * 384, oracle.max_threads()


def run_reference(args):
    """--impl reference: the oracle on the host cores, each step a bounded sample (4 cells)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cells_per_step = 4
    for _ in range(args.warmup):
        oracle_sample(1)
    t_tot, cs_tot, cores = 0.0, 0, 1
    for _ in range(args.steps):
        dt, cs, cores = oracle_sample(cells_per_step)
        t_tot += dt
        cs_tot += cs
    gbs = cs_tot * BYTES_PER_CHAN_SAMPLE / t_tot / 1e9
    sample = f"{cells_per_step} cells (channel x 384-sample frame) of configs[1] per step, oracle as it stands"
    line = {
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "channels_realtime": gbs / GBS_PER_CHANNEL,
        "config": {"workload": "configs[1] single node load: 4 coarse channels x 49152 samples x 2048 inputs "
                               "(bounded sample of its output cells)"},
        "cpu_baseline": {"value": gbs, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": gbs, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_cuda(args):
    import numpy as np
    import torch

    import paper_1702_04728_b200 as bf
    import synth

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    bf.load_library()

    # ---- workload: channels sharded over ranks (weak scaling: every GPU its own C channels) ----
    cfg = synth.CONFIGS[1]
    T = cfg["n_time"]
    C = synth.CONFIGS[3]["group"] if args.workload == "group" else cfg["n_coarse"]
    seed = synth.config_seed(3 if args.workload == "group" else 1)
    from paper_1702_04728_b200.sharding import weak_scaling_shard
    chan0, _ = weak_scaling_shard(C, rank)
    chan0 %= 1024 - C + 1
    freqs = synth.chime_freqs_mhz(C, 1, k0=chan0)
    gains = synth.gains(seed + 1000 * rank, C, flagged_frac=cfg["flagged"])
    plan = bf.plan_create_ex(C, freq_mhz=freqs, gains=gains, zero_pad=args.zero_pad, upchan_len=args.upchan, n_time=T)
    d_in = synth.noise_bytes(seed, C, T, device="cuda", chan0=chan0)
    d_out = torch.empty(plan.out_shape, dtype=torch.uint8, device="cuda")
    in_bytes, out_bytes = plan.in_bytes, plan.out_elems
    # end to end (host buffers through the C-ABI) on the first 4 channels: PCIe moves 403 MB per step in ~8 ms;
    # the whole 12.9 GB group would only repeat the same PCIe-bound rate 32 times
    Ce = min(C, cfg["n_coarse"])
    plan_e = plan if Ce == C else bf.plan_create_ex(Ce, freq_mhz=freqs[:Ce], gains=gains[:Ce], zero_pad=args.zero_pad,
                                                    upchan_len=args.upchan, n_time=T)
    h_in = d_in[:Ce].cpu().pin_memory()
    h_out = torch.empty(plan_e.out_shape, dtype=torch.uint8).pin_memory()
    e2e_in_bytes, e2e_out_bytes = plan_e.in_bytes, plan_e.out_elems
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()

    # ---- device-resident: K steps, per-step CUDA events on the launching stream ----
    for _ in range(max(args.warmup, 3)):
        plan.execute(d_in, d_out, stream=stream)
    barrier()
    if rank == 0:
        # keep the GPU under the same load (untimed) until nvidia-smi delivers its first sample, so that the
        # clock record covers the timed region that follows
        t_wait = time.perf_counter()
        while not sampler.rows and time.perf_counter() - t_wait < 3.0:
            for _ in range(10):
                plan.execute(d_in, d_out, stream=stream)
            torch.cuda.synchronize()
    barrier()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for a, b in evs:
        a.record(stream)
        plan.execute(d_in, d_out, stream=stream)
        b.record(stream)
    e1.record(stream)
    barrier()
    total_ms = e0.elapsed_time(e1)
    kern_ms = float(np.mean([a.elapsed_time(b) for a, b in evs]))

    # ---- end to end through the C-ABI with HOST buffers (H2D + kernel + D2H inside the call) ----
    n_e2e = max(2, min(args.steps, 5))
    plan_e.execute_host(h_in, h_out, stream=stream)
    barrier()
    t0 = time.perf_counter()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record(stream)
    for _ in range(n_e2e):
        plan_e.execute_host(h_in, h_out, stream=stream)
    g1.record(stream)
    barrier()
    e2e_ms = g0.elapsed_time(g1)
    clocks = sampler.stop() if rank == 0 else None
    assert torch.equal(h_out, d_out[:Ce].cpu()), "host path and device path disagree"
    status = plan.kernel_status() | plan_e.kernel_status()
    assert status == 0, f"a pipeline hand-over timed out inside the kernel (status {status})"
    # the roofline denominator, measured on this device under this run's clocks
    peak_ffma, peak_ffma2 = bf.measure_fp32_peak(3000, stream=stream) if rank == 0 else (0.0, 0.0)

    if dist is not None:
        t = torch.tensor([total_ms, kern_ms, e2e_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, kern_ms, e2e_ms = [float(x) for x in t.tolist()]
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    gbs = world * args.steps * in_bytes / (total_ms * 1e-3) / 1e9
    e2e_gbs = world * n_e2e * e2e_in_bytes / (e2e_ms * 1e-3) / 1e9
    peaks, peak_kind = measured_peaks()
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    fp32_peak = N_SM * LANES * 2 * sm_mhz * 1e6 / 1e12
    chan_samples = C * T
    import math
    # nominal FFT flops per (channel, sample): 8 rows x 5 NP log2 NP (N-S) + 2048 series x 5 log2 U (time)
    fft_flops = 8 * 5.0 * args.zero_pad * math.log2(args.zero_pad) + 2048 * 5.0 * math.log2(args.upchan)
    assert (args.zero_pad, args.upchan) != (512, 128) or fft_flops == FFT_FLOPS
    ach = fft_flops * chan_samples / (kern_ms * 1e-3) / 1e12
    hbm_peak = float(peaks["hbm_gbs"])
    hbm_ach = (in_bytes + out_bytes) / (kern_ms * 1e-3) / 1e9
    traffic, traffic_src = None, None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            tj = json.load(f)
        if args.zero_pad == 512 and args.upchan == 128:     # the profile is of the default setting (cfg1 launch):
            # scaled to this launch by the algorithmic bytes (traffic is 1.00x algorithmic in the profile)
            traffic = float(tj["dram_bytes_per_launch"]) * (in_bytes + out_bytes) / float(tj["algorithmic_bytes"])
            traffic_src = tj["source"]
    except Exception:
        pass
    line = {
        "metric": METRIC, "value": gbs, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "channels_realtime": gbs / GBS_PER_CHANNEL,
        "realtime_fraction_full_band": gbs / (1024 * GBS_PER_CHANNEL),
        "config": {"workload": (f"one channel group of configs[3] (full-band streaming) per GPU: {C} coarse channels x "
                                if args.workload == "group" else
                                f"configs[1] single node load per GPU: {C} coarse channels x ") +
                               f"{T} samples x 2048 inputs, zero_pad {args.zero_pad}, upchan {args.upchan}, "
                               "random gains, 2% flagged, device-resident",
                   "in_bytes_per_step": in_bytes, "out_bytes_per_step": out_bytes,
                   "l2": f"input ({in_bytes / 1e6:.0f} MB) larger than L2 (126 MB); no flush needed",
                   "parallelism": f"channel-sharded x{world}, no collective"},
        "roofline": {"bound": "alu", "achieved": ach, "peak": fp32_peak, "unit": "TFLOP/s",
                     "frac": ach / fp32_peak, "traffic": traffic,
                     "traffic_unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum)",
                     "traffic_source": traffic_src, "algorithmic_bytes": in_bytes + out_bytes,
                     "peak_measured": peak_ffma2, "frac_of_measured": ach / peak_ffma2 if peak_ffma2 else None,
                     "peak_measured_note": f"chime_bf_measure_fp32_peak in this run: FFMA {peak_ffma:.1f}, FFMA2 "
                                           f"{peak_ffma2:.1f} TFLOP/s",
                     "kernel": f"chime4::umma_beamform_kernel<{args.upchan}>", "kernel_ms": kern_ms,
                     "flops_per_chan_sample": fft_flops,
                     "note": f"FP32 peak = 148 SM x 128 lanes x 2 x {sm_mhz:.0f} MHz ({peak_kind} sm_max_mhz); "
                             "nominal FFT flops (5 n log2 n) per BASELINE north_star",
                     "hbm": {"achieved": hbm_ach, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_ach / hbm_peak,
                             "peak_kind": peak_kind}},
        "e2e": {"value": e2e_gbs, "unit": UNIT, "h2d_bytes_per_step": e2e_in_bytes,
                "d2h_bytes_per_step": e2e_out_bytes, "steps": n_e2e,
                "workload": f"chime_bf_execute_host on the first {Ce} channels of the step (pinned host buffers; "
                            "PCIe-bound, so more channels would repeat the same rate)"},
        "gpu_launches": args.steps * plan.launches_per_execute,
        "clocks": clocks,
    }
    if world == 1 and args.workload == "group":     # outside the timed region of the step: the (f1) kernel's own roofline
        line["dedisp"] = dedisp_subrecords()
    if not args.no_cpu_baseline and world == 1:     # the oracle is timed on rank 0 at N = 1 only
        dt, cs, cores = oracle_sample(256)
        v = cs * BYTES_PER_CHAN_SAMPLE / dt / 1e9
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "256 output cells (channel x 384 samples) of configs[1], "
                                          f"{dt:.1f} s of oracle time", "channels_realtime": v / GBS_PER_CHANNEL}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_cfg3(args):
    """--workload cfg3: BASELINE.json configs[3], full-band streaming.  1024 channels x 49152-sample chunks as
    8 channel groups of 128 (12.9 GB each) through two device-resident buffers on two CUDA streams, looped
    for --chunks full-band chunks (80 = 10.07 s of telescope time, 8.25 TB).  Host/PCIe ingest is not part
    of it (819 GB/s cannot come from a host); the buffers hold seeded noise and are re-used."""
    import torch

    import paper_1702_04728_b200 as bf
    import synth
    from paper_1702_04728_b200.streaming import FullBandStreamer

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(0)
    bf.load_library()
    cfg = synth.CONFIGS[3]
    C, T, G = cfg["n_coarse"], cfg["n_time"], cfg["group"]
    seed = synth.config_seed(3)
    st = FullBandStreamer(C, G, T, freq_mhz=synth.config_freqs(3))
    for i, buf in enumerate(st.in_bufs):
        buf.copy_(synth.noise_bytes(seed, G, T, device="cuda", chan0=i * G))
    outs = [torch.empty(st.group_out_shape, dtype=torch.uint8, device="cuda") for _ in range(st.n_groups)]
    sampler = ClockSampler(0)
    sampler.start()
    st.run_chunk(None, out_u8=outs)                       # warm-up: one full-band chunk (8 launches)
    st.synchronize()
    torch.cuda.synchronize()
    e0 = torch.cuda.Event(enable_timing=True)
    ends = [torch.cuda.Event(enable_timing=True) for _ in st.streams]
    e0.record(st.streams[0])
    st.streams[1].wait_event(e0)
    st.launches = 0
    for _ in range(args.chunks):
        st.run_chunk(None, out_u8=outs)
    for e, s in zip(ends, st.streams):
        e.record(s)
    st.synchronize()
    torch.cuda.synchronize()
    ms = max(e0.elapsed_time(e) for e in ends)
    clocks = sampler.stop()
    total_bytes = float(args.chunks) * C * T * BYTES_PER_CHAN_SAMPLE
    gbs = total_bytes / (ms * 1e-3) / 1e9
    tel_s = args.chunks * T / REALTIME_SAMPLES_PER_S
    line = {
        "metric": METRIC, "value": gbs, "unit": UNIT, "n_gpus": 1, "steps": args.chunks, "warmup": 1,
        "ms_per_step": ms / args.chunks, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "channels_realtime": gbs / GBS_PER_CHANNEL,
        "realtime_fraction_full_band": gbs / (1024 * GBS_PER_CHANNEL),
        "config": {"workload": "configs[3] full band streaming: 1024 coarse channels x 49152-sample chunks, "
                               "8 channel groups of 128 on two streams / two device buffers (ping-pong), "
                               f"{args.chunks} chunks = {tel_s:.2f} s of telescope time, {total_bytes / 1e12:.2f} TB",
                   "telescope_seconds": tel_s, "wall_seconds": ms * 1e-3,
                   "paper_rate": "6.4 Tbps = 800 GB/s as printed (PAPER.md:43); exact product 819.2 GB/s",
                   "l2": "each group (12.9 GB) is far larger than L2"},
        "gpu_launches": st.launches, "clocks": clocks,
    }
    print(json.dumps(line))
    st.destroy()
    return 0


def dedisp_subrecords(steps=20):
    """Sub-records of the default line: the dedispersion kernel on a configs[2]-shaped beam
    array, uint8 [64 channels][1017 frames][1024 beams][16 fine] = 1.07 GB (>> L2), at DM 10 and DM 40, through
    chime_bf_dedisperse_beams_noalloc (no allocation inside the timed region).  HBM-bound: achieved = algorithmic bytes
    (input bytes on some track + uint32 output) / CUDA-event time per launch, against the measured HBM peak."""
    import torch

    import paper_1702_04728_b200 as bf
    import synth

    cfg = synth.CONFIGS[2]
    C, R = cfg["n_coarse"], cfg["n_time"] // 384
    freqs = synth.config_freqs(2)
    g = torch.Generator(device="cuda").manual_seed(synth.config_seed(2))
    beams = torch.randint(0, 256, (C, R, 1024, 16), dtype=torch.uint8, device="cuda", generator=g)
    peaks, peak_kind = measured_peaks()
    stream = torch.cuda.current_stream()
    recs = []
    for dm in (10.0, 40.0):
        _, mx = bf.dedisp_delays_ex(freqs, dm)
        n_out = R - mx
        out = torch.empty((1024, n_out), dtype=torch.int32, device="cuda")
        for _ in range(3):
            bf.dedisperse_beams_noalloc(beams, freqs, dm, out, stream=stream)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            bf.dedisperse_beams_noalloc(beams, freqs, dm, out, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        nbytes = C * n_out * 1024 * 16 + out.numel() * 4
        ach = nbytes / (ms * 1e-3) / 1e9
        recs.append({"dm": dm, "n_out": n_out, "kernel": "chime_dd::dedisperse_kernel", "kernel_ms": ms, "steps": steps,
                     "bound": "hbm", "achieved": ach, "peak": float(peaks["hbm_gbs"]), "unit": "GB/s",
                     "frac": ach / float(peaks["hbm_gbs"]), "algorithmic_bytes": nbytes, "peak_kind": peak_kind})
        del out
    del beams
    torch.cuda.empty_cache()
    return recs


def run_dedisp(args):
    """--workload dedisp: the dedispersion kernel on a configs[2]-shaped beam array:
    uint8 [64 channels][1017 frames][1024 beams][16 fine] = 1.07 GB (>> L2), DM --dm (10: 0.19 s sweep)."""
    import torch

    import paper_1702_04728_b200 as bf
    import synth

    torch.cuda.set_device(0)
    cfg = synth.CONFIGS[2]
    C, T = cfg["n_coarse"], cfg["n_time"]
    plan = bf.plan_create_ex(C, freq_mhz=synth.config_freqs(2), n_time=T)
    g = torch.Generator(device="cuda").manual_seed(synth.config_seed(2))
    beams = torch.randint(0, 256, plan.out_shape, dtype=torch.uint8, device="cuda", generator=g)
    dm = args.dm
    _, n_out = plan.dedisp_delays(dm)
    out = torch.empty((1024, n_out), dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()
    sampler = ClockSampler(0)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        plan.dedisperse(beams, dm, out_u32=out, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        plan.dedisperse(beams, dm, out_u32=out, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    clocks = sampler.stop()
    peaks, peak_kind = measured_peaks()
    # algorithmic bytes: each (channel, fine) contributes n_out frames of 1024 beams -> C * n_out * 16384 input bytes
    # (frames outside every track are never needed), plus the uint32 output
    in_bytes = C * n_out * 1024 * 16
    nbytes = in_bytes + out.numel() * 4
    ach = nbytes / (ms * 1e-3) / 1e9
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            tj = json.load(f)["dedisp"]
        if dm == 10.0:
            traffic = float(tj["dram_bytes_per_launch"])
    except Exception:
        pass
    line = {
        "metric": "dedispersion input GB/s (uint8 beams)", "value": in_bytes / (ms * 1e-3) / 1e9, "unit": UNIT,
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8->u32", "data": "synthetic",
        "config": {"workload": "dedisperse configs[2]-shaped beams: 64 channels x 1017 frames x 1024 beams x 16 fine "
                               f"(1.07 GB), DM {dm}, {n_out} output samples per beam", "l2": "input >> L2"},
        "roofline": {"bound": "hbm", "achieved": ach, "peak": float(peaks["hbm_gbs"]), "unit": "GB/s",
                     "frac": ach / float(peaks["hbm_gbs"]), "traffic": traffic, "algorithmic_bytes": nbytes,
                     "kernel": "chime_dd::dedisperse_kernel", "kernel_ms": ms, "peak_kind": peak_kind},
        "gpu_launches": args.steps, "clocks": clocks,
    }
    print(json.dumps(line))
    plan.destroy()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default="group", choices=["group", "cfg1", "cfg3", "dedisp"],
                    help="cfg1 (default, the contract's step) or cfg3 (full-band streaming, 1 GPU)")
    ap.add_argument("--chunks", type=int, default=80, help="cfg3: full-band chunks to stream")
    ap.add_argument("--zero-pad", type=int, default=512, choices=[256, 512, 1024],
                    help="cfg1: padded N-S length (512 = the paper's and the contract's setting)")
    ap.add_argument("--upchan", type=int, default=128, choices=[128, 256], help="cfg1: up-channelisation length")
    ap.add_argument("--dm", type=float, default=10.0, help="dedisp: nominal DM (pc/cm^3)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "dedisp":
        return run_dedisp(args)
    return run_cfg3(args) if args.workload == "cfg3" else run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
