#!/usr/bin/env python
"""bench.py -- the driver's measurement contract for the DMAS-k hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

One step = one pass of the whole hot path (ingest, delay, interpolated gather,
signed root, power sums, Newton combination, axial band-pass, Hilbert-FIR envelope, log compression, frame
batching) over one batch of 64 synthetic frames of the headline workload C2b (BASELINE.json north_star:
128 elements x 2048 samples x 1024x256 pixels, order 3, batched frames), through the C ABI (pab_beamform).
`value` = frames/s with the RF already resident in HBM; `e2e` = the same through pab_beamform_host with host
buffers (pinned), H2D and D2H inside the timed region.  Rank 0 prints ONE JSON line.

Multi-GPU: frames are independent, the path has no exchange step: replicas only, one context per GPU, each
rank runs its own 64-frame batch ("scaling": "weak"), no data-path collective; max-over-ranks timing.

--impl reference times the fp64 CPU oracle (oracle/) as it stands on the host cores, on a bounded sample of
the same workload (this tier's reference arm); rank 0 only.
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

ORDER = 3
FRAMES = 64
WORKLOAD = "C2b"
POST = dict(mode="log", f_center=10e6, f_halfwidth=2.5e6, n_taps_bp=64, n_taps_hilbert=63, dyn_range_db=60.0)
N_SETS = 4          # rotating input/output buffer sets: 4 x (64 MiB RF + 64 MiB image) = 512 MiB > 126 MB L2
METRIC = "beamformed frames/s, order-3 DMAS, 128ch (C2b: 128 el x 2048 samp x 1024x256 px, 64-frame batches, " \
         "band-pass + envelope + log)"

# Work per item (pixel x element x frame) of the fused beamforming kernel at order 3 as this build runs it (cached
# interpolation taps: no delay square root in the kernel): XU (MUFU) lane-ops = 2 (lg2 + ex2
# of the cube root); FP32-pipe slots = 6 (interpolation 2, x 1/3, three accumulations); HBM bytes = RF in + image
# out + the 4-byte tap table of the geometry, once per launch.  (With in-kernel delays the algorithmic figures are
# 2 + 1/64 and 6 + 3/64: one square root and three FP32 slots per (pixel, element), shared by the 64 frames.)
XU_PER_ITEM = 2.0
FP32_PER_ITEM = 6.0
# What the build issues per item (its SASS mix, profiles/r2_headline_sass.txt): two of a thread's 16 frames take their cube
# root on the FMA pipe (pab_math.cuh cbrt_fma2), so 14/16 x 2 = 1.75 MUFU per item; the interpolation and the power sums
# are packed f32x2 (one slot per two frames).  The roofline fraction keeps the algorithmic 2.0 in its numerator.
XU_PER_ITEM_ISSUED = 1.75
DELAY_CACHE = "all"
SM_COUNT = 148
NCU_TRAFFIC_BYTES = 181_827_584 + 49_893_376   # per 64-frame launch; profiles/r2_headline_ncu.md
NCU_TRAFFIC_COMMIT = "666c3df (round 2)"   # the build that capture was taken on: the constant goes stale silently otherwise
XU_LANES_PER_CLK_SM = 16
FP32_LANES_PER_CLK_SM = 128


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.t.join(timeout=2)
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": float(max(power))}


def make_inputs(n_frames: int, seed_offset: int = 0):
    """Seeded synthetic C2b frames (paper_2203_14906_b200/synth.py)."""
    from paper_2203_14906_b200 import synth
    w = synth.make_config(WORKLOAD, seed=1012 + seed_offset, n_frames=n_frames)
    return w.geom, w.rf


def oracle_step(orc, rf, g, nthreads=0):
    """The oracle's whole path on rf [F][N][S]: fp64 beamform (route B) + band-pass + envelope + log."""
    img, used = orc.beamform(rf, g, ORDER, nthreads=nthreads, return_threads=True)
    orc.post(img, g, POST["f_center"], POST["f_halfwidth"], POST["n_taps_bp"], POST["n_taps_hilbert"],
             POST["dyn_range_db"], mode="log")
    return used


def time_oracle(n_frames: int, steps: int, warmup: int):
    """frames/s of the oracle as it stands on the host cores; each step = n_frames frames of the C2b workload."""
    import oracle as orc
    orc.build()
    g, rf = make_inputs(n_frames)
    used = 1
    for _ in range(warmup):
        used = oracle_step(orc, rf, g)
    t0 = time.perf_counter()
    for _ in range(steps):
        used = oracle_step(orc, rf, g)
    dt = time.perf_counter() - t0
    return n_frames * steps / dt, dt / steps * 1e3, used


def run_reference(args, rank: int):
    if rank != 0:
        return
    sample_frames = 2
    fps, ms, cores = time_oracle(sample_frames, args.steps, args.warmup)
    sample = f"{sample_frames} frames of C2b per step (of the 64-frame batch), fp64 route B + post chain, OpenMP"
    line = {"impl": "reference", "metric": METRIC, "value": fps, "unit": "frames/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD + "+post", "order": ORDER, "frames_per_step": sample_frames,
                       "n_elem": 128, "n_samp": 2048, "nz": 1024, "nx": 256},
            "cpu_baseline": {"value": fps, "unit": "frames/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": fps, "unit": "frames/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def max_over_ranks(values, world: int, device):
    """Replicas-only timing rule: every rank measures its own replica, the job's time is the max over ranks."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def run_ours(args, rank: int, local_rank: int, world: int):
    import torch
    import torch.distributed as dist
    from paper_2203_14906_b200 import binding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    binding.load(build_if_missing=True)             # nvcc-builds libpab.so if absent; raises when it cannot (no fallback)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    g, rf_np = make_inputs(FRAMES, seed_offset=rank)
    rf_host = torch.from_numpy(rf_np).pin_memory()
    rf_sets = [torch.roll(rf_host, r, 0).to(dev) for r in range(N_SETS)]
    out_sets = [torch.empty((FRAMES, g.nz, g.nx), dtype=torch.float32, device=dev) for _ in range(N_SETS)]
    out_host = torch.empty((FRAMES, g.nz, g.nx), dtype=torch.float32).pin_memory()
    bf = binding.Beamformer(g, post=POST, delay_cache=DELAY_CACHE)
    stream = torch.cuda.current_stream(dev)
    items_per_frame = g.nz * g.nx * g.n_elem
    K, W = args.steps, max(args.warmup, 3)

    def step(i):
        bf.beamform(rf_sets[i % N_SETS], ORDER, out=out_sets[i % N_SETS], stream=stream)

    # ---- device-resident throughput: K steps in one timed region, barrier + synchronize on both sides ----
    for i in range(W):
        step(i)
    barrier()
    bf.set_profile(8 * K + 8)
    clocks = ClockSampler(local_rank)
    if rank == 0:
        clocks.start()
        time.sleep(0.3)
    barrier()
    n0 = bf.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(K):
        step(W + i)
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = bf.launch_count() - n0
    prof = bf.get_profile(reset=True)
    bf.set_profile(0)
    clk = clocks.stop() if rank == 0 else None

    # ---- end to end: pab_beamform_host, pinned host buffers, H2D + D2H inside the timed region ----
    Ke = max(3, min(K, 10))
    for _ in range(2):
        bf.beamform_host(rf_host, ORDER, out=out_host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        bf.beamform_host(rf_host, ORDER, out=out_host)      # returns after the last D2H has finished
    torch.cuda.synchronize()
    e2e_sync_ms = (time.perf_counter() - t0) * 1e3
    checksum = float(out_host[0, 512, 128])

    # the streaming form: pab_beamform_host_async per step, one pab_host_sync at the end; successive steps overlap
    # (H2D of step i + 1, kernels of step i, D2H of step i - 1).  Two pinned buffer pairs in rotation, every copy of every
    # step inside the timed region.
    rf_host2 = torch.from_numpy(rf_np).pin_memory()
    out_host2 = torch.empty((FRAMES, g.nz, g.nx), dtype=torch.float32).pin_memory()
    pairs = [(rf_host, out_host), (rf_host2, out_host2)]
    Ka = max(6 * Ke, 48)          # enough steps for the one ramp-up and drain of the stream (2.4 ms) to weigh < 4 %
    for i in range(3):
        bf.beamform_host_async(pairs[i & 1][0], ORDER, pairs[i & 1][1])
    bf.host_sync()
    barrier()
    t0 = time.perf_counter()
    for i in range(Ka):
        bf.beamform_host_async(pairs[i & 1][0], ORDER, pairs[i & 1][1])
    bf.host_sync()
    e2e_ms = (time.perf_counter() - t0) * 1e3 * Ke / Ka          # scaled to Ke steps, like the other e2e figures
    checksum_async = float(out_host2[0, 512, 128])

    # the same with int16 transport (BASELINE.json config C5: the ADC data is int16): the C2b frames quantised to
    # 15 bits of their peak, scale restored by pab_set_input; half the host-to-device bytes
    peak_rf = float(np.max(np.abs(rf_np)))
    q_scale = peak_rf / 32000.0
    rf16_host = torch.from_numpy(np.rint(rf_np / q_scale).astype(np.int16)).pin_memory()
    bf16 = binding.Beamformer(g, dtype="int16", scale=q_scale, post=POST, delay_cache=DELAY_CACHE)
    for _ in range(2):
        bf16.beamform_host(rf16_host, ORDER, out=out_host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        bf16.beamform_host(rf16_host, ORDER, out=out_host)
    torch.cuda.synchronize()
    e2e16_sync_ms = (time.perf_counter() - t0) * 1e3
    for i in range(3):
        bf16.beamform_host_async(rf16_host, ORDER, pairs[i & 1][1])
    bf16.host_sync()
    barrier()
    t0 = time.perf_counter()
    for i in range(Ka):
        bf16.beamform_host_async(rf16_host, ORDER, pairs[i & 1][1])
    bf16.host_sync()
    e2e16_ms = (time.perf_counter() - t0) * 1e3 * Ke / Ka
    bf16.close()
    box = binding.measure_peaks() if rank == 0 else None      # bare pinned cudaMemcpyAsync rates of this box, same run
    # what a stream of steps can reach at best: a step's H2D and D2H bytes as bare pinned copies on two streams at once
    # (both directions of the link busy, as in the streaming form), same run
    d_probe_in = torch.empty_like(rf_host, device=dev)
    d_probe_out = torch.empty_like(out_host, device=dev)
    s_a, s_b = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
    bidir_ms = 0.0
    for rep in range(2):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(8):
            with torch.cuda.stream(s_a):
                d_probe_in.copy_(rf_host, non_blocking=True)
            with torch.cuda.stream(s_b):
                out_host2.copy_(d_probe_out, non_blocking=True)
        torch.cuda.synchronize()
        bidir_ms = (time.perf_counter() - t0) * 1e3 / 8
    del d_probe_in, d_probe_out

    # ---- beamform-only (raw output) throughput, for the stage breakdown ----
    bf_raw = binding.Beamformer(g, delay_cache=DELAY_CACHE)
    for i in range(3):
        bf_raw.beamform(rf_sets[i % N_SETS], ORDER, out=out_sets[i % N_SETS], stream=stream)
    torch.cuda.synchronize()
    r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    r0.record(stream)
    for i in range(K):
        bf_raw.beamform(rf_sets[i % N_SETS], ORDER, out=out_sets[i % N_SETS], stream=stream)
    r1.record(stream)
    torch.cuda.synchronize()
    raw_ms = r0.elapsed_time(r1) / K
    bf_raw.close()

    # the in-kernel-delay (table-free) headline beside the cached one
    bf_nc = binding.Beamformer(g, delay_cache="off")
    for i in range(3):
        bf_nc.beamform(rf_sets[i % N_SETS], ORDER, out=out_sets[i % N_SETS], stream=stream)
    torch.cuda.synchronize()
    bf_nc.set_profile(4 * K + 8)
    for i in range(K):
        bf_nc.beamform(rf_sets[i % N_SETS], ORDER, out=out_sets[i % N_SETS], stream=stream)
    torch.cuda.synchronize()
    nc_ms, nc_n = bf_nc.get_profile()["beamform"]
    nc_launch_ms = nc_ms / max(nc_n, 1)
    bf_nc.close()

    ms_total, e2e_ms, e2e16_ms, e2e_sync_ms, e2e16_sync_ms = max_over_ranks([ms_total, e2e_ms, e2e16_ms, e2e_sync_ms, e2e16_sync_ms], world, dev)
    if rank == 0:
        peaks = read_peaks()
        ms_step = ms_total / K
        fps = world * FRAMES * K / (ms_total * 1e-3)
        bf_ms, bf_n = prof["beamform"]
        bf_launch_ms = bf_ms / max(bf_n, 1)
        frames_per_launch = FRAMES * K / max(bf_n, 1)
        items_per_launch = items_per_frame * frames_per_launch
        f_hz = peaks["sm_max_mhz"] * 1e6
        xu_peak = SM_COUNT * XU_LANES_PER_CLK_SM * f_hz
        fp32_peak = SM_COUNT * FP32_LANES_PER_CLK_SM * f_hz
        hbm_bytes = frames_per_launch * (g.n_elem * g.n_samp * 4 + g.nz * g.nx * 4) + g.nz * g.nx * g.n_elem * 4
        t_xu = items_per_launch * XU_PER_ITEM / xu_peak
        t_fp32 = items_per_launch * FP32_PER_ITEM / fp32_peak
        t_hbm = hbm_bytes / (peaks["hbm_gbs"] * 1e9)
        achieved = items_per_launch * XU_PER_ITEM / (bf_launch_ms * 1e-3)
        roofline = {"bound": "alu", "kernel": "bf_cached_kernel<3,4,false,0,1> (fused tap fetch + interpolation + root + power sums + Newton, 16 "
                              "frames per thread, cached interpolation taps, packed f32x2 arithmetic, 2 of 16 roots on the FMA pipe)",
                    "achieved": achieved / 1e9, "peak": xu_peak / 1e9, "unit": "Gop/s (XU/MUFU lane-ops)",
                    "frac": achieved / xu_peak, "frac_definition": "XU (MUFU) pipe term of T_roof (DESIGN.md reading B3)",
                    "frac_xu": t_xu / (bf_launch_ms * 1e-3),
                    "frac_fp32_hbm": max(t_fp32, t_hbm) / (bf_launch_ms * 1e-3),      # north_star's literal FMA-rate reading
                    "in_kernel_delays": {"launch_ms": nc_launch_ms,
                                         "frac_xu": items_per_launch * (XU_PER_ITEM + 1.0 / FRAMES) / xu_peak / (nc_launch_ms * 1e-3)},
                    "traffic": NCU_TRAFFIC_BYTES, "traffic_commit": NCU_TRAFFIC_COMMIT,
                    "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture of this "
                                      "kernel at this workload: profiles/r2_headline_ncu.md",
                    "peak_source": f"148 SM x 16 XU lanes/clk x {peaks['sm_max_mhz']:.0f} MHz (sm_max_mhz, "
                                   f"{peaks['source']}); DESIGN.md Roofline",
                    "launch_ms": bf_launch_ms, "launches_timed": bf_n,
                    "t_roof_ms": {"xu": t_xu * 1e3, "fp32": t_fp32 * 1e3, "hbm": t_hbm * 1e3},
                    "algorithmic_per_item": {"xu_ops": XU_PER_ITEM, "fp32_slots": FP32_PER_ITEM,
                                             "hbm_bytes": hbm_bytes / items_per_launch},
                    "issued_per_item": {"xu_ops": XU_PER_ITEM_ISSUED,
                                        "xu_pipe_busy": items_per_launch * XU_PER_ITEM_ISSUED / xu_peak / (bf_launch_ms * 1e-3),
                                        "note": "2 of 16 cube roots per thread run on the FMA pipe; frac keeps the algorithmic 2.0"},
                    "items_per_s": items_per_launch / (bf_launch_ms * 1e-3),
                    "hbm_achieved_gbs": hbm_bytes / (bf_launch_ms * 1e-3) / 1e9, "hbm_peak_gbs": peaks["hbm_gbs"]}
        stages = {k: {"ms_per_step": v[0] / K, "launches_per_step": v[1] / K} for k, v in prof.items()}
        line = {"metric": METRIC, "value": fps, "unit": "frames/s", "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": WORKLOAD + "+post", "order": ORDER, "frames_per_step": FRAMES,
                           "n_elem": g.n_elem, "n_samp": g.n_samp, "nz": g.nz, "nx": g.nx, "post": "log",
                           "delay_cache": DELAY_CACHE,
                           "parallelism": f"replicas x{world}, no collective",
                           "l2": f"inputs/outputs rotate over {N_SETS} buffer sets (512 MiB) > 126 MB L2"},
                "items_per_s": fps * items_per_frame,
                "e2e": {"value": world * FRAMES * Ke / (e2e_ms * 1e-3), "unit": "frames/s",
                        "h2d_bytes_per_step": int(rf_host.numel() * 4), "d2h_bytes_per_step": int(out_host.numel() * 4),
                        "ms_per_step": e2e_ms / Ke, "steps": Ka,
                        "api": "pab_beamform_host_async per step + one pab_host_sync (pinned host buffers; successive steps overlap)",
                        "checksum": checksum_async,
                        "blocking_call": {"value": world * FRAMES * Ke / (e2e_sync_ms * 1e-3), "ms_per_step": e2e_sync_ms / Ke, "steps": Ke,
                                          "api": "pab_beamform_host (returns after its last D2H)", "checksum": checksum,
                                          "int16_value": world * FRAMES * Ke / (e2e16_sync_ms * 1e-3)},
                        "h2d_ceiling_gbs": box["h2d_pinned_gbs"], "d2h_ceiling_gbs": box["d2h_pinned_gbs"],
                        "copy_bound_ms": max(rf_host.numel() * 4 / box["h2d_pinned_gbs"], out_host.numel() * 4 / box["d2h_pinned_gbs"]) * 1e-6,
                        "copy_bound_bidir_ms": bidir_ms,
                        "frac_of_copy_bound_bidir": bidir_ms / (e2e_ms / Ke),
                        "int16_input": {"value": world * FRAMES * Ke / (e2e16_ms * 1e-3), "ms_per_step": e2e16_ms / Ke,
                                        "h2d_bytes_per_step": int(rf16_host.numel() * 2),
                                        "note": "same frames quantised to int16 (scale restored by pab_set_input)"}},
                "timing_note": "per-launch profiling events (pab_set_profile) are recorded inside the timed region: "
                               "two event records per kernel, a slight downward bias of value",
                "box_peaks": box,
                "gpu_launches": int(launches), "clocks": clk, "roofline": roofline, "stages": stages,
                "raw_only": {"ms_per_step": raw_ms, "frames_per_s": FRAMES / (raw_ms * 1e-3),
                             "items_per_s": FRAMES * items_per_frame / (raw_ms * 1e-3)}}
        if not args.no_cpu_baseline:
            n_cpu = 16
            cfps, cms, cores = time_oracle(n_cpu, 2, 0)
            import oracle as _orc
            _g1, _rf1 = make_inputs(1)
            _t0 = time.perf_counter()
            oracle_step(_orc, _rf1, _g1, nthreads=1)
            single = 1.0 / (time.perf_counter() - _t0)
            line["cpu_baseline"] = {"value": cfps, "unit": "frames/s", "cores": cores, "kind": "oracle",
                                    "single_thread_value": single,
                                    "sample": f"2 passes over the first {n_cpu} frames of the step's 64-frame C2b batch, "
                                              "fp64 route B + post chain"}
        print(json.dumps(line), flush=True)
    bf.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# XU (MUFU) lane-ops and FP32-pipe slots per item, by order: (per item, per (pixel, element)) -- DESIGN.md Roofline
_XU = {1: (0.0, 1.0), 2: (1.0, 1.0), 3: (2.0, 1.0), 4: (2.0, 1.0), 5: (2.0, 1.0), 6: (2.0, 1.0), 7: (2.0, 1.0), 8: (2.0, 1.0)}
_FP32 = {1: (3.0, 3.0), 2: (4.0, 3.0), 3: (6.0, 3.0), 4: (7.0, 3.0), 5: (9.0, 3.0), 6: (14.0, 3.0), 7: (16.0, 3.0),
         8: (18.0, 3.0)}


def run_sweep(args):
    """--sweep: every config and order of SURVEY.md section 8 (C1..C5, C2b) on one GPU, one JSON line each:
    ms per call, frames/s, items/s, per-stage CUDA-event times and the roofline terms.  Not the driver's line."""
    import torch
    from paper_2203_14906_b200 import binding, synth
    torch.cuda.set_device(0)
    binding.load(build_if_missing=True)
    peaks = read_peaks()
    f_hz = peaks["sm_max_mhz"] * 1e6
    cases = [("C1", 1, (1, 2, 3, 4, 5), False, "none"), ("C2", 1, (1, 2, 3), False, "none"),
             ("C2b", 64, (1, 2, 3), False, "none"), ("C2b", 64, (3,), False, "cf"), ("C3", 256, (3,), True, "none"),
             ("C4", 1, (4, 5), False, "none"), ("C4", 16, (4, 5), False, "none"), ("C4", 16, (5,), False, "cf"),
             ("C5", 1024, (3,), True, "none"), ("C2b", 64, (6, 8), False, "none"), ("C2b", 64, (1, 2, 3), False, "nearest"), ("C4", 16, (4, 5), False, "nearest")]
    cases += [("C2", 1, (1, 2, 3), False, "cache-single"), ("C4", 1, (4, 5), False, "cache-single"),
              ("C2b", 64, (1, 2, 3), False, "cache-all"), ("C4", 16, (4, 5), False, "cache-all"),
              ("C2b", 64, (3,), False, "cf-cache-all"), ("C4", 16, (5,), False, "cf-cache-all"),
              ("C2b", 64, (6, 8), False, "cache-all"),
              ("C3", 256, (3,), True, "cache-all"), ("C5", 1024, (3,), True, "cache-all"),
              ("C2", 1, (1, 2, 3), False, "nearest"), ("C4", 1, (4, 5), False, "nearest"),
              ("C2", 1, (3,), False, "cf"), ("C4", 1, (5,), False, "cf")]
    if args.case:                         # --case C2:1:cache-single[:3]  ->  one config / frame count / mode [/ order]
        want = args.case.split(":")
        cases = [c for c in cases if c[0] == want[0] and str(c[1]) == want[1] and c[4] == want[2]]
        if len(want) > 3:
            cases = [(c[0], c[1], (int(want[3]),), c[3], c[4]) for c in cases]
    for cfg, F, orders, post, weight in cases:
        interp = "nearest" if weight == "nearest" else "linear"
        cache = weight.split("cache-")[1] if "cache-" in weight else "off"
        weight = "cf" if weight.startswith("cf") else "none"
        gen = min(F, 64)
        w = synth.make_config(cfg, n_frames=gen)
        g = w.geom
        call_frames = min(F, 64) if cfg == "C5" else F          # C5 streams in batches of 64 (BASELINE.json)
        n_calls = F // call_frames
        rf = torch.from_numpy(np.concatenate([w.rf] * (call_frames // gen), axis=0)).cuda()
        dtype = "int16" if w.rf.dtype == np.int16 else "float32"
        out = torch.empty((call_frames, g.nz, g.nx), dtype=torch.float32, device="cuda")
        bf = binding.Beamformer(g, dtype=dtype, post=dict(w.post) if post else None, weight=weight, interp=interp,
                                delay_cache=cache)
        items = g.nz * g.nx * g.n_elem
        for order in orders:
            reps = max(3, min(50, int(0.2 / max(1e-5, items * F * 1e-12))))
            for _ in range(3):
                bf.beamform(rf, order, out=out)
            torch.cuda.synchronize()
            bf.set_profile(16 * reps * n_calls + 16)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps * n_calls):
                bf.beamform(rf, order, out=out)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps                      # whole stream of F frames
            prof = bf.get_profile()
            bf.set_profile(0)
            fpt = bf.plan()["frames_per_thread"] if F >= 4 else 1
            if order >= 4:
                fpt = min(fpt, 8)
            if order >= 6:
                fpt = min(fpt, 4)
            if weight == "cf":
                fpt = min(fpt, 4 if order >= 4 else 8)
            share = min(fpt, F)                                  # frames sharing one delay computation (algorithmic: the batch)
            batch = min(F, 64)
            xu = _XU[order][0] + _XU[order][1] / batch
            if interp == "nearest":          # no MUFU and no delay arithmetic in the hot loop; u, u^2.. accumulation only
                xu = 0.0
            if cache != "off" and (F < 4 or cache == "all"):
                xu = _XU[order][0]            # taps come from the table: no delay square root in the kernel
            diag_share = 0
            if cache == "off" and F < 4 and interp == "linear" and bf.plan()["diagonal"] == 2:
                # table-free diagonal kernel: one delay (one MUFU, 3 FP32-equivalent slots) per diagonal, shared by the
                # 16 (orders 1..3) or 8 (orders 4, 5, and every order under CF weighting) pairs of the diagonal a thread owns
                diag_share = 16 if (order <= 3 and weight == "none") else 8
                xu = _XU[order][0] + _XU[order][1] / diag_share
            taps_from_table = cache != "off" and (F < 4 or cache == "all")       # no delay arithmetic in the kernel at all
            fp = _FP32[order][0] + (0.0 if taps_from_table else _FP32[order][1] / batch) + ((1.0 if order % 2 else 2.0) if weight == "cf" else 0.0)
            if interp == "nearest":
                fp = {1: 1.0, 2: 3.0, 3: 4.0, 4: 5.0, 5: 7.0}[order]
                if F < 4 and bf.plan()["diagonal"] == 1:      # single frames on the diagonal kernel: roots per item, not per RF sample
                    xu = _XU[order][0]
            if diag_share:
                fp = _FP32[order][0] + _FP32[order][1] / diag_share + ((1.0 if order % 2 else 2.0) if weight == "cf" else 0.0)
            t_xu = items * F * xu / (SM_COUNT * XU_LANES_PER_CLK_SM * f_hz) * 1e3
            t_fp = items * F * fp / (SM_COUNT * FP32_LANES_PER_CLK_SM * f_hz) * 1e3
            in_b = g.n_elem * g.n_samp * (2 if dtype == "int16" else 4)
            t_hbm = F * (in_b + g.nz * g.nx * 4) / (peaks["hbm_gbs"] * 1e9) * 1e3
            # secondary ceiling (not in the roofline denominator): shared-memory bandwidth, 128 B/clk/SM; the
            # interpolated path gathers 2 x 4 bytes per item, the nearest-sample path 4
            t_sm = items * F * (4.0 if interp == "nearest" else 8.0) / (SM_COUNT * 128.0 * f_hz) * 1e3
            bf_ms = prof["beamform"][0] / reps
            print(json.dumps({"sweep": cfg, "order": order, "frames": F, "post": "log" if post else "raw", "weight": weight, "interp": interp, "delay_cache": cache,
                              "dtype_in": dtype, "n_elem": g.n_elem, "n_samp": g.n_samp, "nz": g.nz, "nx": g.nx,
                              "ms_per_stream": round(ms, 5), "frames_per_s": round(F / (ms * 1e-3), 1),
                              "items_per_s": round(items * F / (ms * 1e-3), 0),
                              "stage_ms": {k: round(v[0] / reps, 5) for k, v in prof.items()},
                              "beamform_launches": prof["beamform"][1] / reps, "frames_per_thread": share,
                              "pairs_per_delay": diag_share if diag_share else share,
                              "t_roof_ms": {"xu": round(t_xu, 5), "fp32": round(t_fp, 5), "hbm": round(t_hbm, 5)},
                              "t_smem_ceiling_ms": round(t_sm, 5),
                              "beamform_roofline_frac": round(max(t_xu, t_fp, t_hbm) / bf_ms, 4),
                              "in_range": bf.plan()["in_range"]}), flush=True)
        bf.close()
        del rf, out


# Paper Table II: ms per frame on a GeForce GT 730, DAS / DMAS / DMAS-3 / DMAS-4 / DMAS-5.  Context
# only: the paper states neither N, S nor the precision (reading A19).
_TABLE2_MS = {512: (2.912, 3.028, 3.309, 4.4, 5.133), 1024: (11.051, 11.6, 12.718, 17.121, 20.03),
              2048: (43.438, 45.784, 50.205, 68.006, 79.653)}


def run_table2(args):
    """--table2: square pixel grids shaped like the paper's Table II (512^2, 1024^2, 2048^2), orders 1..5, 128
    elements x 4096 samples, single frames and 16-frame batches, in both delay modes (nearest = the paper's own
    integer-delay formulation with a delay table, linear = the interpolated path with cached interpolation taps).
    One JSON line per case."""
    import torch
    from paper_2203_14906_b200 import binding, synth
    torch.cuda.set_device(0)
    binding.load(build_if_missing=True)
    rng = np.random.default_rng(1020)
    N, S, fs, c, pitch = 128, 4096, 40e6, 1540.0, 0.3e-3
    rf16 = torch.from_numpy((rng.standard_normal((16, N, S)) * 0.3).astype(np.float32)).cuda()
    for side in (512, 1024, 2048):
        dx = pitch / (side // 128)            # columns on a sub-multiple of the pitch (38.4 mm wide): the taps are then
        g = synth.Geometry(N, S, fs, c, pitch, side, side, -(side - 1) / 2 * dx, dx, 5e-3, 60e-3 / (side - 1)).f32()   # translation invariant
        out = torch.empty((16, side, side), dtype=torch.float32, device="cuda")
        for interp in ("nearest", "linear"):
            bf = binding.Beamformer(g, interp=interp, delay_cache="all" if interp == "linear" else "off")
            for F in (1, 16):
                for order in (1, 2, 3, 4, 5):
                    rf = rf16[:F]
                    for _ in range(2):
                        bf.beamform(rf, order, out=out[:F])
                    torch.cuda.synchronize()
                    reps = 5
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    for _ in range(reps):
                        bf.beamform(rf, order, out=out[:F])
                    e1.record()
                    torch.cuda.synchronize()
                    ms = e0.elapsed_time(e1) / reps / F
                    print(json.dumps({"table2": f"{side}x{side}", "interp": interp, "order": order, "frames_per_call": F,
                                      "n_elem": N, "n_samp": S, "ms_per_frame": round(ms, 5),
                                      "frames_per_s": round(1e3 / ms, 1),
                                      "items_per_s": round(side * side * N / (ms * 1e-3), 0),
                                      "paper_gt730_ms_per_frame": _TABLE2_MS[side][order - 1]}), flush=True)
            bf.close()
        del out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--table2", action="store_true", help="square grids shaped like the paper's Table II; 1 GPU")
    ap.add_argument("--sweep", action="store_true", help="per-config table (C1..C5), one JSON line each; 1 GPU")
    ap.add_argument("--case", default="", help="with --sweep: only config:frames:mode[:order], e.g. C2:1:cache-single:3")
    ap.add_argument("--peaks", action="store_true", help="pab_measure_peaks: MUFU / FFMA / LDS.128 unit rates and pinned "
                                                         "copy rates of this box, one JSON line; 1 GPU")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.peaks:
        if rank == 0:
            from paper_2203_14906_b200 import binding
            binding.load(build_if_missing=True)
            print(json.dumps({"peaks": binding.measure_peaks()}), flush=True)
        return
    if args.sweep or args.table2:
        if rank == 0:
            run_sweep(args) if args.sweep else run_table2(args)
        return
    if world != args.gpus and world == 1 and args.gpus > 1:
        raise SystemExit("bench.py --gpus N > 1 must be launched with torch.distributed.run (one rank per GPU)")
    run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
