#!/usr/bin/env python
"""bench.py — throughput of the fused SK hot path (arXiv 1808.10365) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload cfg1|cfg4|...]

A step is one pass of the whole hot path (unpack -> S1/S2 -> Eq. 14 -> flag) over one synthetic
frame of the workload.  Metric: SK input samples/s (1 sample = 1 byte of 4+4-bit data), whole job.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement".
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "sk_input_samples_per_s"
UNIT = "samples/s"
FALLBACK_HBM_GBS = 6650.0


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20, help="K: sk_frame calls captured in the CUDA graph")
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="cfg1")
    ap.add_argument("--zero", action="store_true", help="excise flagged cells in place (a8)")
    ap.add_argument("--seconds", type=float, default=1.0,
                    help="length of the timed steady-state region: the K-step graph is replayed back to back for "
                         "about this long inside one CUDA-event pair (after half as long untimed)")
    ap.add_argument("--burst-seconds", type=float, default=0.02,
                    help="extra 'burst' object: the same replays for this long after --cooldown seconds of idle "
                         "(0 = skip); not the headline")
    ap.add_argument("--cooldown", type=float, default=0.5, help="idle seconds before the burst window")
    ap.add_argument("--sweep", action="store_true", help="--workload cfg3: time every (M, N) point of config 3")
    ap.add_argument("--sweep-seconds", type=float, default=0.25, help="timed seconds per sweep point")
    ap.add_argument("--serialize", action="store_true",
                    help="do not pass SK_FRAME_INPUTS_READY: each frame waits for the previous one to finish")
    ap.add_argument("--e2e-steps", type=int, default=0, help="0 = min(steps, 20)")
    ap.add_argument("--op", default="frame", choices=["frame", "multi", "rebin", "single", "sim", "cm", "ceiling", "memonly", "eager", "fig5", "fig6", "firstpass"],
                    help="frame = the fused hot path (the contract's line); rebin / single = the SURVEY 8(f) "
                         "outputs next to it (sk_rebin_sums factor 2, sk_single), timed on config-4-sized sums")
    ap.add_argument("--path", default="auto", choices=["auto", "ldg"],
                    help="A/B timing: ldg = the direct-load kernel instead of the TMA stream kernel (the SK_FRAME_PLAN_LDG bit of the call's flags)")
    ap.add_argument("--lanes", type=int, default=0, choices=[0, 1, 2, 4, 8, 16],
                    help="A/B timing: force a slab width of 16*lanes inputs (SK_FRAME_PLAN_LANES in the call's flags); 0 = automatic")
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def workload(name):
    import sk_synth
    idx = {"cfg0": 0, "cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4}[name]
    return sk_synth.config(idx)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def stored_profile(name):
    """The row of profiles/roofline_traffic.csv (from the committed ncu --set full captures) for this
    workload / op, or {}: dram bytes, warp instructions and issue utilisation per launch."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "roofline_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == name:
                    return row
    except Exception:
        pass
    return {}


def stored_traffic(name):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed capture, or None."""
    row = stored_profile(name)
    return int(row["dram_bytes_per_launch"]) if row else None


# Philox4x32-10 as the oracle fixes it (one 32-bit word per component, ten rounds): 20 IMAD.WIDE per call
# of 4 words = 2 complex samples, each holding the half-rate fmaheavy pipe of a sub-partition for 4 cycles
# (bench.py --op ceiling: IDP / FFMA2 / IMAD class instructions issue every 2 cycles per warp, a wide multiply
# is two of them): 40 pipe cycles per complex sample and lane, before any digitising or Box-Muller.
PHILOX_PIPE_CYCLES_PER_SAMPLE = 40.0


def method_roofline(name, samples_per_launch, achieved_samples_per_s, bytes_written_per_sample):
    """Roofline object of the two simulators against what the METHOD needs, not against the kernel's own
    instruction count: the lower of the HBM rate for the bytes a sample writes and the generator's floor on
    the fmaheavy pipe (PHILOX_PIPE_CYCLES_PER_SAMPLE).  The kernel's issue utilisation from
    the committed ncu capture is reported beside it as what it is: IPC, not a fraction of a roofline."""
    hbm, hbm_src = peaks()
    philox = 592 * 1.965e9 * 32.0 / PHILOX_PIPE_CYCLES_PER_SAMPLE / 1e9            # Gsamples/s
    hbm_bound = hbm / bytes_written_per_sample if bytes_written_per_sample else float("inf")
    peak = min(philox, hbm_bound)
    row = stored_profile(name)
    out = {"bound": "alu" if philox <= hbm_bound else "hbm", "achieved": achieved_samples_per_s / 1e9, "unit": "Gsamples/s",
           "peak": peak, "frac": achieved_samples_per_s / 1e9 / peak,
           "traffic": int(row["dram_bytes_per_launch"]) if row else None,
           "peak_source": "min(Philox4x32-10 floor: 592 sub-partitions x 1.965 GHz x 32 lanes / %g fmaheavy cycles per "
                          "sample = %.0f Gsamples/s; HBM write at %g B per sample: %s)"
                          % (PHILOX_PIPE_CYCLES_PER_SAMPLE, philox, bytes_written_per_sample,
                             "%.0f Gsamples/s" % hbm_bound if bytes_written_per_sample else "none, nothing is stored"),
           "frac_of_hbm_write_roofline": (achieved_samples_per_s / 1e9 / hbm_bound) if bytes_written_per_sample else None}
    if row:
        per32 = float(row["warp_instructions_per_launch"]) * 32.0 / samples_per_launch
        out["issue"] = {"warp_instructions_per_32_samples": per32, "ncu_issue_active_pct": float(row["issue_active_pct"]),
                        "note": "IPC of the kernel's own instruction stream (profiles/%s), not a roofline" % row["source"]}
    return out


def sm_ceiling(sk, torch, dev, sm_mhz, sm_max_mhz, achieved_samples_per_s, warps=12):
    """The SM-side ceiling of the hot loop, MEASURED in this run (skb_loop_ceiling of the bench library: the kernel's
    a1-a3 loop on a fixed shared-memory tile, no memory traffic, `warps` warps per SM as in the kernel):
    sub-partition cycles per 32 samples -> samples/s at the SM clock the timed region ran at."""
    from paper_1808_10365_b200 import benchlib
    cyc = benchlib.loop_ceiling(warps, 100, dev)
    subp = 4 * torch.cuda.get_device_properties(dev).multi_processor_count
    out = {"subpartition_cycles_per_32_samples": cyc, "warps_per_sm": warps, "subpartitions": subp,
           "samples_per_s_at_sm_max": subp * 32 * (sm_max_mhz or 1965) * 1e6 / cyc,
           "what": "skb_loop_ceiling (libsk_b200_bench.so): the stream kernel's tile loop alone (no HBM, TMA, barrier or epilogue)"}
    if sm_mhz:
        out["samples_per_s_at_observed_clock"] = subp * 32 * sm_mhz * 1e6 / cyc
        out["frac_at_observed_clock"] = achieved_samples_per_s / out["samples_per_s_at_observed_clock"]
    return out


def run_ceiling(args):
    """--op ceiling: the SM-side ceiling of the hot loop for 4..16 warps per SM, the same loop with one
    kind of instruction left out (attribution by removal), and the issue rates of its instructions."""
    import torch
    from paper_1808_10365_b200 import benchlib
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    n0 = benchlib.launch_count()
    benchlib.loop_ceiling(12, 20, dev)
    pts = [{"warps_per_sm": w, "subpartition_cycles_per_32_samples": benchlib.loop_ceiling(w, 200, dev)}
           for w in (4, 8, 12, 16)]
    removal = {name: benchlib.loop_ceiling(12, 200, dev, variant=v) for name, v in benchlib.VARIANTS.items()
               if name != "memonly"}
    pipes = {name: benchlib.pipe_rate(m, 16, dev) for m, name in enumerate(benchlib.PIPE_MODES)}
    # the loop alone for ~1.5 s with the NVML record: what the arithmetic draws without any memory traffic
    sampler = ClockSampler(0)
    sampler.start()
    t_lo = time.perf_counter()
    sampler.window = (t_lo, None)
    cyc_long, calls = [], 0
    while time.perf_counter() - t_lo < 1.5:
        cyc_long.append(benchlib.loop_ceiling(12, 4000, dev))
        calls += 1
    t_hi = time.perf_counter()
    sampler.window = (t_lo, t_hi)
    loop_clocks = sampler.summary()
    sampler.stop_flag = True
    subp = 4 * torch.cuda.get_device_properties(dev).multi_processor_count
    loop_rate = subp * 32 * (loop_clocks["sm_mhz"] or 1965) * 1e6 / (sum(cyc_long) / len(cyc_long))
    best = min(p["subpartition_cycles_per_32_samples"] for p in pts if p["warps_per_sm"] <= 12)
    print(json.dumps({
        "op": "ceiling", "metric": "sm_side_ceiling_samples_per_s", "value": subp * 32 * 1.965e9 / best, "unit": "samples/s",
        "n_gpus": 1, "steps": 1, "warmup": 1, "higher_is_better": True, "data": "synthetic", "dtype": "u8->u32",
        "config": {"workload": "the stream kernel's tile loop on a fixed shared-memory tile (no HBM traffic)",
                   "value_is": "sub-partitions x 32 lanes x 1.965 GHz / cycles per 32 samples at 12 warps per SM",
                   "points": pts,
                   "removal_at_12_warps": removal,
                   "removal_note": "sub-partition cycles per 32 samples of the same loop with one kind of instruction left "
                                   "out (sums are then wrong): no_fadd2 = without sub.rn.f32x2, no_prmt = without the four "
                                   "PRMT per word, no_unpack = without LOP3/SHF/LOP3",
                   "subpartition_cycles_per_warp_instruction": pipes,
                   "pipes_note": "16 warps per SM, 8 independent chains per lane; pairs count two instructions",
                   "loop_for_1.5_s": {"clocks": loop_clocks, "samples_per_s": loop_rate,
                                      "pj_per_sample": (loop_clocks["power_w"] or 0) / loop_rate * 1e12,
                                      "note": "12 warps per SM, back-to-back launches: board power of the arithmetic "
                                              "alone (no HBM traffic), idle power included"}},
        "gpu_launches": int(benchlib.launch_count() - n0)}))


def run_memonly(args):
    """--op memonly: is memory the limit?  The product's TMA stream kernel (skb_stream of the bench library:
    same loads, ring, epilogue, finalizer and programmatic dependent launch) on config-1 frames, once with the
    product's loop body and once with the arithmetic replaced by an XOR of the loaded words, in the headline's
    steady-state protocol (a CUDA graph of 200 launches replayed for --seconds inside one event pair, after half
    as long untimed) and in a burst after --cooldown seconds of idle."""
    import torch
    import sk_synth
    from paper_1808_10365_b200 import benchlib
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cfg = workload(args.workload)
    l2 = 126 * 1024 * 1024
    nbuf = max(4, -(-5 * l2 // cfg.nbytes))
    bufs = [sk_synth.make_frame(cfg, device=dev, frame=fid) for fid in frame_ids(0, nbuf)]
    B = cfg.T // cfg.M
    stream = torch.cuda.Stream(device=dev)
    SK = torch.empty((B, cfg.F), dtype=torch.float32, device=dev)
    mask = torch.empty((B, cfg.F), dtype=torch.uint8, device=dev)
    ws = benchlib.stream_workspace(cfg.T, cfg.F, cfg.E, cfg.M, dev)
    torch.cuda.synchronize()
    peak, peak_src = peaks()
    n0 = benchlib.launch_count()
    rows = []
    G = 200

    def barrier():
        torch.cuda.synchronize()

    for name in ("product", "memonly"):
        var = benchlib.VARIANTS[name]
        with torch.cuda.stream(stream):
            for i in range(5):
                benchlib.stream(var, bufs[i % nbuf], cfg.M, SK, mask, ws, inputs_ready=True, stream=stream)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            for i in range(G):
                benchlib.stream(var, bufs[i % nbuf], cfg.M, SK, mask, ws, inputs_ready=True, stream=stream)
        with torch.cuda.stream(stream):
            graph.replay()
        torch.cuda.synchronize()
        sampler = ClockSampler(0)
        sampler.start()
        time.sleep(args.cooldown)
        ms_b, reps_b, clocks_b = timed_replays(torch, graph, stream, args.burst_seconds or 0.02, 2e-5, G, barrier, sampler)
        timed_replays(torch, graph, stream, args.seconds / 2, ms_b * 1e-3 / (reps_b * G), G, barrier)
        ms, reps, clocks = timed_replays(torch, graph, stream, args.seconds, ms_b * 1e-3 / (reps_b * G), G, barrier, sampler)
        sampler.stop_flag = True
        per = ms / (reps * G)
        per_b = ms_b / (reps_b * G)
        rows.append({"variant": name, "us_per_frame": per * 1e3, "read_gbs": cfg.nbytes / per / 1e6,
                     "frac_of_peak": cfg.nbytes / per / 1e6 / peak, "clocks": clocks,
                     "pj_per_byte": (clocks["power_w"] or 0) / (cfg.nbytes / (per * 1e-3)) * 1e12,
                     "burst": {"us_per_frame": per_b * 1e3, "read_gbs": cfg.nbytes / per_b / 1e6,
                               "frac_of_peak": cfg.nbytes / per_b / 1e6 / peak, "clocks": clocks_b}})
    print(json.dumps({
        "op": "memonly", "metric": "hbm_read_gbs", "value": rows[1]["read_gbs"], "unit": "GB/s", "n_gpus": 1,
        "steps": G, "warmup": 5, "ms_per_step": rows[1]["us_per_frame"] * 1e-3, "higher_is_better": True,
        "data": "synthetic", "dtype": "u8",
        "config": {"workload": cfg.name, "frame_bytes": cfg.nbytes, "frames": nbuf,
                   "launch": "one CUDA graph of %d skb_stream launches (programmatic dependent launch, inputs ready), "
                             "replayed for %.2f s inside one CUDA-event pair after %.2f s untimed; burst: %.2f s after "
                             "%.1f s idle" % (G, args.seconds, args.seconds / 2, args.burst_seconds or 0.02, args.cooldown),
                   "peak_gbs": peak, "peak_source": peak_src},
        "variants": rows, "gpu_launches": int(benchlib.launch_count() - n0)}))


def run_eager(args):
    """--op eager: what a caller WITHOUT a CUDA graph gets.  Plain back-to-back sk_frame calls issued from a C
    loop (skb_frame_loop of the bench library calls the product's own entry point), with and without
    SK_FRAME_INPUTS_READY, for about --seconds each after half as long untimed; device time from a CUDA-event
    pair around the loop, host time per call from the loop's own clock."""
    import torch
    import paper_1808_10365_b200 as sk
    import sk_synth
    from paper_1808_10365_b200 import benchlib
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cfg = workload(args.workload)
    l2 = 126 * 1024 * 1024
    nbuf = 10 if cfg.nbytes > l2 else max(4, -(-5 * l2 // cfg.nbytes))
    nbuf = max(2, min(nbuf, int(torch.cuda.mem_get_info()[0] * 0.8) // cfg.nbytes))
    bufs = [sk_synth.make_frame(cfg, device=dev, frame=fid) for fid in frame_ids(0, nbuf)]
    sk_mean = null_mean(sk, sk_synth, cfg, dev)
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        ws = sk.workspace_for(cfg.T, cfg.F, cfg.E, cfg.M, dev, stream.cuda_stream)
        out = sk.sk_frame(bufs[0], cfg.M, n_sigma=5.0, sk_mean=sk_mean, workspace=ws, stream=stream)
    torch.cuda.synchronize()
    peak, peak_src = peaks()
    n0 = sk.sk_launch_count()
    rows = []
    for name, flags in (("SK_FRAME_INPUTS_READY", sk.binding.SK_FRAME_INPUTS_READY), ("no flag (each frame waits for the previous one)", 0)):
        benchlib.frame_loop(bufs, cfg.M, out.SK, out.mask, ws, 50, flags, sk_mean=sk_mean, stream=stream)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        benchlib.frame_loop(bufs, cfg.M, out.SK, out.mask, ws, 200, flags, sk_mean=sk_mean, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        est = e0.elapsed_time(e1) * 1e-3 / 200
        calls = max(200, int(args.seconds / est))
        benchlib.frame_loop(bufs, cfg.M, out.SK, out.mask, ws, calls // 2, flags, sk_mean=sk_mean, stream=stream)
        sampler = ClockSampler(0)
        sampler.start()
        torch.cuda.synchronize()
        t_lo = time.perf_counter()
        sampler.window = (t_lo, None)
        e0.record(stream)
        host_s = benchlib.frame_loop(bufs, cfg.M, out.SK, out.mask, ws, calls, flags, sk_mean=sk_mean, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        sampler.window = (t_lo, time.perf_counter())
        clocks = sampler.summary()
        sampler.stop_flag = True
        per = e0.elapsed_time(e1) * 1e-3 / calls
        # the host cost of a call by itself: 16 calls into an idle stream (the loop above runs at the device's
        # pace once the launch queue is full, so its host time per call is just the device time again)
        idle = []
        for _ in range(20):
            torch.cuda.synchronize()
            idle.append(benchlib.frame_loop(bufs, cfg.M, out.SK, out.mask, ws, 16, flags, sk_mean=sk_mean, stream=stream) / 16)
        torch.cuda.synchronize()
        rows.append({"flags": name, "calls": calls, "us_per_frame": per * 1e6, "host_us_per_call": host_s / calls * 1e6,
                     "host_us_per_call_idle_stream": sorted(idle)[len(idle) // 2] * 1e6,
                     "samples_per_s": cfg.nbytes / per, "read_gbs": cfg.nbytes / per / 1e9,
                     "frac_of_peak": cfg.nbytes / per / 1e9 / peak, "clocks": clocks})
    print(json.dumps({
        "op": "eager", "metric": METRIC, "value": rows[0]["samples_per_s"], "unit": UNIT, "n_gpus": 1,
        "steps": rows[0]["calls"], "warmup": rows[0]["calls"] // 2, "ms_per_step": rows[0]["us_per_frame"] * 1e-3,
        "higher_is_better": True, "data": "synthetic", "dtype": "u8->u32/f64",
        "config": {"workload": cfg.name, "frame_bytes": cfg.nbytes, "frames": nbuf,
                   "launch": "NO CUDA graph: plain back-to-back sk_frame calls from a C loop (skb_frame_loop), one stream",
                   "peak_gbs": peak, "peak_source": peak_src},
        "cases": rows, "gpu_launches": int(sk.sk_launch_count() - n0)}))


def frame_ids(rank, nbuf):
    """Frame numbers rank `rank` draws: disjoint between ranks (weak scaling, independent frames)."""
    return [rank * 1000 + i for i in range(nbuf)]


def max_over_ranks(x, world, device):
    """A duration as the job sees it: the slowest rank's (no-op for one process)."""
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(samples_per_rank_step, world, steps, ms):
    """Whole-job throughput: the samples all ranks processed / the slowest rank's time."""
    return samples_per_rank_step * world * steps / (ms * 1e-3)


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.samples, self.names, self.stop_flag, self.ok = [], {}, False, False
        self.max_mhz = None
        self.power_limit = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            try:
                self.power_limit = pynvml.nvmlDeviceGetEnforcedPowerLimit(self.h) / 1000.0
            except Exception:
                self.power_limit = None
            self.ok = True
        except Exception:
            self.ok = False
        self.window = None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        self.names = names = {
            nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap",
        } if hasattr(nv, "nvmlClocksEventReasonHwSlowdown") else {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
        }
        while not self.stop_flag:
            try:
                t = time.perf_counter()
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                try:
                    pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                except Exception:
                    pw = None
                self.samples.append((t, mhz, r, pw))
            except Exception:
                pass
            time.sleep(0.0002)

    def summary(self):
        """Median SM clock and throttle reasons of the samples INSIDE the window (never of others)."""
        if not self.ok or not self.window:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0, "power_w": None,
                    "power_limit_w": self.power_limit}
        lo, hi = self.window
        inside = [(m, r, pw) for (t, m, r, pw) in list(self.samples) if lo <= t <= (hi or 1e30)]
        mhz = sorted(m for m, _, _ in inside)
        watts = sorted(pw for _, _, pw in inside if pw is not None)
        reasons = sorted({nm for _, r, _ in inside for bit, nm in self.names.items() if r & bit})
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(inside), "power_w": watts[len(watts) // 2] if watts else None,
                "power_limit_w": self.power_limit}


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores, on the same workload/metric.
    Each step is one full frame of the workload when that fits a few seconds, else a slab of blocks."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import sk_synth
    from oracle import sk_oracle
    cfg = workload(args.workload)
    # bounded sample: at ~0.2 Gsamples/s keep one step near half a second
    max_bytes = 100 * 1024 * 1024
    blocks = max(1, min(cfg.B, max_bytes // (cfg.M * cfg.F * cfg.E)))
    sub = cfg.with_(T=blocks * cfg.M)
    host = sk_synth.make_frame(sub).numpy()
    steps = max(1, min(args.steps, 20))
    warm = max(0, min(args.warmup, 5))
    n_sigma = 5.0                                          # as the GPU arm
    sk_mean = round(float(sk_oracle.frame(null_frame(sk_synth, cfg, cfg.M).numpy(), cfg.M)["SK"].astype("float64").mean()), 4)
    for _ in range(warm):
        sk_oracle.frame(host, cfg.M, n_sigma=n_sigma, sk_mean=sk_mean)
    t0 = time.perf_counter()
    for _ in range(steps):
        sk_oracle.frame(host, cfg.M, n_sigma=n_sigma, sk_mean=sk_mean)
    dt = time.perf_counter() - t0
    v = host.size * steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": dt / steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "E": cfg.E, "F": cfg.F, "T": cfg.T, "M": cfg.M, "N": cfg.E,
                   "n_sigma": n_sigma, "sk_mean": sk_mean, "zero_flagged": False,
                   "sample": f"{blocks} of {cfg.B} blocks per step ({host.size} samples)"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"{steps} steps x {host.size} samples of {cfg.name}"},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_sim(args):
    """--op sim: the App. B simulator (sk_sim_digitised) writing config-1-shaped frames, then the
    null mean through sk_frame + sk_moments."""
    import torch
    import paper_1808_10365_b200 as sk
    import sk_synth
    torch.cuda.set_device(0)
    cfg = sk_synth.config(1)
    thr = sk_synth.digitiser_thresholds(sk_synth.sigma_per_input(cfg)).cuda()
    bufs = [torch.empty(cfg.T, cfg.F, cfg.E, dtype=torch.uint8, device="cuda") for _ in range(4)]
    K, W = args.steps, max(args.warmup, 3)
    for i in range(W):
        sk.sk_sim_digitised(cfg.T, cfg.F, cfg.E, thr, 1, i, out=bufs[i % 4])
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = sk.sk_launch_count()
    e0.record()
    for i in range(K):
        sk.sk_sim_digitised(cfg.T, cfg.F, cfg.E, thr, 1, 100 + i, out=bufs[i % 4])
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / K
    mean, var = sk.sk_moments(sk.sk_frame(bufs[0], cfg.M).SK)
    print(json.dumps({
        "op": "sim", "metric": "simulated_samples_per_s", "value": cfg.nbytes / (ms * 1e-3), "unit": "samples/s",
        "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": True, "data": "synthetic",
        "dtype": "u32->u8", "config": {"workload": cfg.name + " shape, per-input sigma ~ U[1.5,3.5]",
                                       "null_mean": float(mean[0].item()), "null_var": float(var[0].item())},
        "roofline": method_roofline("sim", cfg.nbytes, cfg.nbytes / (ms * 1e-3), 1.0),
        "gpu_launches": int(sk.sk_launch_count() - n0) }))


def run_cm(args):
    """--op cm: one point of Fig. 5: 1000 datasets, n = 256, N = 4096 receivers."""
    import torch
    import paper_1808_10365_b200 as sk
    torch.cuda.set_device(0)
    D, M, N, amp = 1000, 256, 4096, 0.5
    K, W = min(args.steps, 5), 3
    for i in range(W):
        sk.sk_sim_common_mode(D, M, N, amp, seed=i)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = sk.sk_launch_count()
    e0.record()
    for i in range(K):
        SK = sk.sk_sim_common_mode(D, M, N, amp, seed=100 + i)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / K
    mean, var = sk.sk_moments(SK)
    print(json.dumps({
        "op": "cm", "metric": "simulated_samples_per_s", "value": D * M * N / (ms * 1e-3), "unit": "samples/s",
        "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": True, "data": "synthetic",
        "dtype": "f64", "config": {"workload": f"App. A: {D} datasets x n={M} x N={N}, common-mode amplitude {amp}",
                                   "mean": float(mean[0].item()), "var": float(var[0].item()),
                                   "n_eff": 4.0 / (M * float(var[0].item()))},
        "roofline": method_roofline("cm", D * M * N, D * M * N / (ms * 1e-3), 0.0),
        "gpu_launches": int(sk.sk_launch_count() - n0)}))


def run_fig5(args):
    """--op fig5: App. A / Fig. 5 of the paper on the device: variance of SK~ over 1000
    datasets of n = 256 samples x N receivers against the amplitude of a common-mode signal, and the
    effective number of receivers N_eff = 4 / (n var)."""
    import torch
    import paper_1808_10365_b200 as sk
    torch.cuda.set_device(0)
    D, n = 1000, 256
    amps = (0.0, 0.03, 0.1, 0.3, 1.0, 3.0)
    n0 = sk.sk_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    rows = []
    for N in (128, 256, 512, 1024, 2048, 4096):
        pts = []
        for a in amps:
            mean, var = sk.sk_moments(sk.sk_sim_common_mode(D, n, N, a, seed=1808 + N))
            v = float(var[0].item())
            pts.append({"amp": a, "mean": float(mean[0].item()), "var": v, "n_eff": 4.0 / (n * v)})
        rows.append({"N": N, "var_predicted_independent": 4.0 / (n * N), "points": pts})
    e1.record()
    torch.cuda.synchronize()
    total = sum(D * n * r["N"] * len(amps) for r in rows)
    print(json.dumps({
        "op": "fig5", "metric": "simulated_samples_per_s", "value": total / (e0.elapsed_time(e1) * 1e-3), "unit": "samples/s",
        "n_gpus": 1, "steps": 1, "warmup": 0, "ms_per_step": e0.elapsed_time(e1), "higher_is_better": True,
        "data": "synthetic", "dtype": "f64",
        "config": {"workload": f"App. A / Fig. 5: {D} datasets x n={n}, x = z + amp*c, variance of SK~ and N_eff = 4/(n var)",
                   "var_predicted_single_receiver": 4.0 / n, "table": rows},
        "gpu_launches": int(sk.sk_launch_count() - n0)}))


def run_fig6(args):
    """--op fig6: App. B / Fig. 6 on the device: moments of SK~ on 4+4-bit data with an
    RMS of 1.52 LSB per component against the same moments of float ('non-digitised') Gaussian data, for
    M = 256 and N = 16 ... 2048 combined receivers."""
    import torch
    import paper_1808_10365_b200 as sk
    import sk_synth
    torch.cuda.set_device(0)
    M, E, B = 256, 2048, 1024
    thr = sk_synth.digitiser_thresholds(torch.full((E,), 1.52, dtype=torch.float64)).cuda()
    n0 = sk.sk_launch_count()
    data = sk.sk_sim_digitised(B * M, 1, E, thr, seed=6, frame=0)
    rows = []
    for N in (16, 64, 256, 1024, 2048):
        mean, var = sk.sk_moments(sk.sk_frame(data, M, first_n=N).SK)
        fm, fv = sk.sk_moments(sk.sk_sim_common_mode(B, M, N, 0.0, seed=66 + N))
        rows.append({"N": N, "digitised_mean": float(mean[0].item()), "float_mean": float(fm[0].item()),
                     "mean_difference": float(mean[0].item()) - float(fm[0].item()),
                     "digitised_var_over_4_MN": float(var[0].item()) * M * N / 4.0,
                     "float_var_over_4_MN": float(fv[0].item()) * M * N / 4.0})
    torch.cuda.synchronize()
    print(json.dumps({
        "op": "fig6", "metric": "null_mean_offset", "value": rows[-1]["mean_difference"], "unit": "SK", "n_gpus": 1,
        "steps": 1, "warmup": 0, "higher_is_better": False, "data": "synthetic", "dtype": "u8 / f64",
        "config": {"workload": f"App. B / Fig. 6: {B} blocks of M={M} x E={E}, 4+4-bit round-and-clip Gaussian, RMS 1.52 LSB "
                               "(sk_sim_digitised -> sk_frame -> sk_moments) against float Gaussian data (sk_sim_common_mode, amp 0)",
                   "value_is": "digitised - float mean of SK~ at N = 2048", "table": rows},
        "gpu_launches": int(sk.sk_launch_count() - n0)}))


def run_aux(args):
    """--op rebin|single: one of the small HBM-bound kernels beside the hot path, on S1/S2 arrays of
    config 4's size (16384 cells x 2048 inputs: 256 MiB for the pair, > L2), five rotating copies (1.25 GiB,
    ten times the L2, so that no launch finds a part of its input still resident)."""
    import torch
    import paper_1808_10365_b200 as sk
    import sk_synth
    torch.cuda.set_device(0)
    cfg = sk_synth.config(2)
    frame = sk_synth.make_frame(cfg, device="cuda")
    S1, S2 = sk.sk_power_sums(frame, cfg.M)
    del frame
    reps = 8                                               # config 2's 2048 cells x 8 = config 4's 16384
    ncopies = 5
    sums = [(S1.repeat(reps, 1, 1), S2.repeat(reps, 1, 1)) for _ in range(ncopies)]
    B, F, E = sums[0][0].shape
    n = B * F * E
    fn = (lambda a, b: sk.sk_rebin_sums(a, b, cfg.M, 2)) if args.op == "rebin" else (lambda a, b: sk.sk_single(a, b, cfg.M))
    alg = n * 8 + (n * 8 // 2 if args.op == "rebin" else n * 4)
    K, W = max(args.steps, 50), max(args.warmup, 3)
    for i in range(W):
        fn(*sums[i % ncopies])
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = sk.sk_launch_count()
    e0.record()
    for i in range(K):
        fn(*sums[i % ncopies])
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / K
    peak, peak_src = peaks()
    print(json.dumps({
        "op": args.op, "metric": "sums_elements_per_s", "value": n / (ms * 1e-3), "unit": "elements/s",
        "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": True, "data": "synthetic",
        "dtype": "u32" if args.op == "rebin" else "u32->f64->f32",
        "config": {"workload": f"S1,S2 [{B}][{F}][{E}] uint32 (config 4's size), M={cfg.M}",
                   "l2": "%d rotating copies, 256 MiB each" % ncopies},
        "roofline": {"bound": "hbm", "achieved": alg / (ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": alg / (ms * 1e-3) / 1e9 / peak, "traffic": stored_traffic(args.op), "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": alg},
        "gpu_launches": int(sk.sk_launch_count() - n0)}))


def run_firstpass(args):
    """--op firstpass: what in-place excision costs the FIRST time a frame is excised.  The headline
    --zero lines replay frames that earlier steps already excised (the same bytes are rewritten); here
    every timed frame is fresh: the working copies are restored from masters outside the timed region,
    then one CUDA graph of one sk_frame call per frame runs inside a CUDA-event pair.  Three cases on
    the same frames: no excision, the workload's own flags, and every cell flagged (the flag centre moved
    far away) — the worst case for the fused finalizer, which excises a whole cell with one warp."""
    import statistics
    import torch
    import paper_1808_10365_b200 as sk
    import sk_synth
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cfg = workload(args.workload)
    l2 = 126 * 1024 * 1024
    nbuf = max(4, -(-4 * l2 // cfg.nbytes))
    nbuf = max(2, min(nbuf, int(torch.cuda.mem_get_info()[0] * 0.4) // cfg.nbytes))
    masters = [sk_synth.make_frame(cfg, device=dev, frame=fid) for fid in frame_ids(0, nbuf)]
    work = [m.clone() for m in masters]
    sk_mean = null_mean(sk, sk_synth, cfg, dev)
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        ws = sk.workspace_for(cfg.T, cfg.F, cfg.E, cfg.M, dev, stream.cuda_stream)
        out = sk.sk_frame(work[0], cfg.M, n_sigma=5.0, sk_mean=sk_mean, workspace=ws, stream=stream)
    torch.cuda.synchronize()
    n0 = sk.sk_launch_count()
    rows = []
    reps = max(args.steps, 5)
    for name, zero, centre in (("no excision", False, sk_mean), ("excision, the workload's own flags", True, sk_mean),
                               ("excision, every cell flagged", True, sk_mean + 10.0)):
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=stream):
            for i in range(nbuf):                 # the first call waits for everything before it (the restore)
                sk.sk_frame(work[i], cfg.M, n_sigma=5.0, sk_mean=centre, zero_flagged=zero, out=out, workspace=ws,
                            stream=stream, inputs_ready=i > 0)
        times, flagged = [], 0.0
        for r in range(reps + 2):
            with torch.cuda.stream(stream):
                for w, m in zip(work, masters):
                    w.copy_(m)                    # fresh bytes: outside the timed region
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(stream):
                e0.record(stream)
                graph.replay()
                e1.record(stream)
            torch.cuda.synchronize()
            if r >= 2:
                times.append(e0.elapsed_time(e1) / nbuf)
            flagged = float(out.mask.float().mean().item())
        ms = statistics.median(times)
        excised = sum(int((w != m).any(dim=2).sum().item()) for w, m in zip(work[-1:], masters[-1:])) if zero else 0
        rows.append({"case": name, "ms_per_frame": ms, "read_gbs": cfg.nbytes / ms / 1e6,
                     "flagged_fraction_last_frame": flagged, "rows_changed_last_frame": excised,
                     "bytes_excised_per_frame": int(round(flagged * cfg.nbytes)) if zero else 0})
    base = rows[0]["ms_per_frame"]
    for r in rows[1:]:
        extra = (r["ms_per_frame"] - base) * 1e-3
        r["extra_us_per_frame"] = extra * 1e6
        r["excision_write_gbs"] = r["bytes_excised_per_frame"] / extra / 1e9 if extra > 0 and r["bytes_excised_per_frame"] else None
    print(json.dumps({
        "op": "firstpass", "metric": "ms_per_frame", "unit": "ms", "higher_is_better": False, "n_gpus": 1,
        "steps": reps, "warmup": 2, "data": "synthetic", "dtype": "u8->u32/f64",
        "config": {"workload": cfg.name, "E": cfg.E, "F": cfg.F, "T": cfg.T, "M": cfg.M, "frame_bytes": cfg.nbytes,
                   "frames": nbuf, "launch": "one CUDA graph of one sk_frame call per frame, SK_FRAME_INPUTS_READY after the "
                   "first; working copies restored from masters before every replay; median of %d replays" % reps},
        "cases": rows, "value": rows[1]["ms_per_frame"], "ms_per_step": rows[1]["ms_per_frame"],
        "gpu_launches": int(sk.sk_launch_count() - n0)}))


def null_mean(sk, sk_synth, cfg, dev, M=None):
    """The flag centre the paper's way: mean SK of an RFI-free simulation with the
    workload's per-input sigmas (the 4-bit null mean is not 1: App. B)."""
    M = M or cfg.M
    null = null_frame(sk_synth, cfg, M).to(dev)
    return round(float(sk.sk_frame(null, M).SK.double().mean().item()), 4)


def null_frame(sk_synth, cfg, M):
    """The RFI-free simulation both arms centre their flag on: drawn on the CPU, so that the GPU arm and the
    reference arm see the same bytes (and print the same sk_mean, rounded to 1e-4)."""
    return sk_synth.make_frame(cfg.with_(T=min(cfg.T, 8 * M), M=M, cw_block_inputs=None, cw_freqs=(),
                                         burst_fraction=0.0, sine_freqs=()), frame=777)


def timed_replays(torch, graph, stream, seconds, step_s_estimate, steps_per_replay, barrier, sampler=None):
    """Replay the K-step graph back to back for about `seconds` inside ONE CUDA-event pair on the
    launching stream.  Returns (ms, replays, clock summary of exactly that window)."""
    reps = max(1, int(round(seconds / max(step_s_estimate * steps_per_replay, 1e-7))))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_lo = time.perf_counter()
    if sampler is not None:
        sampler.window = (t_lo, None)
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(reps):
            graph.replay()
        e1.record(stream)
    barrier()
    t_hi = time.perf_counter()
    clocks = None
    if sampler is not None:
        sampler.window = (t_lo, t_hi)
        clocks = sampler.summary()
    return e0.elapsed_time(e1), reps, clocks


def run_sweep(args, sk, sk_synth, torch, dev):
    """--workload cfg3 --sweep: BASELINE.json config 3, throughput at each (M, N): M in {64..1024} x
    N in {16..2048} (the first N inputs).  Inputs beyond N are never read, so next to the frame's
    samples/s the line gives the bytes actually moved and the GB/s on those."""
    cfg = workload("cfg3")
    nbuf = 2                                              # 2 x 512 MiB > 4 x L2
    bufs = [sk_synth.make_frame(cfg, device=dev, frame=i) for i in range(nbuf)]
    stream = torch.cuda.Stream(device=dev)
    peak, peak_src = peaks()
    K = args.steps
    points, launches = [], 0
    for M in (64, 128, 256, 512, 1024):
        sk_mean = null_mean(sk, sk_synth, cfg, dev, M)
        B = cfg.T // M
        for N in (16, 64, 256, 1024, 2048):
            with torch.cuda.stream(stream):
                ws = sk.workspace_for(cfg.T, cfg.F, cfg.E, M, dev, stream.cuda_stream)
                out = sk.sk_frame(bufs[0], M, first_n=N, n_sigma=3.0, sk_mean=sk_mean, workspace=ws, stream=stream)
            torch.cuda.synchronize()

            def step(i):
                sk.sk_frame(bufs[i % nbuf], M, first_n=N, n_sigma=3.0, sk_mean=sk_mean, out=out, workspace=ws,
                            stream=stream, inputs_ready=True)
            n0 = sk.sk_launch_count()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=stream):
                for i in range(K):
                    step(i)
            launches += sk.sk_launch_count() - n0
            with torch.cuda.stream(stream):
                graph.replay()
            torch.cuda.synchronize()
            ms, reps, _ = timed_replays(torch, graph, stream, args.sweep_seconds, 1e-4, K, torch.cuda.synchronize)
            ms, reps, _ = timed_replays(torch, graph, stream, args.sweep_seconds, ms * 1e-3 / (reps * K), K,
                                        torch.cuda.synchronize)
            step_s = ms * 1e-3 / (reps * K)
            lanes, slabs, chunk, bpu = sk.sk_frame_plan(cfg.T, cfg.F, cfg.E, M, first_n=N, inputs_ready=True)
            alg = cfg.T * cfg.F * N + B * cfg.F * 5                                  # N/E of the frame + outputs
            moved = cfg.T * cfg.F * min(cfg.E, slabs * 16 * lanes) + B * cfg.F * 5   # whole slabs are fetched
            skv = out.SK.double()
            points.append({"M": M, "N": N, "us_per_frame": step_s * 1e6,
                           "frame_samples_per_s": cfg.nbytes / step_s,
                           "bytes_algorithmic": alg, "gbs_algorithmic": alg / step_s / 1e9,
                           "bytes_moved": moved, "gbs_on_bytes_moved": moved / step_s / 1e9,
                           "frac_of_measured_peak": moved / step_s / 1e9 / peak,
                           "plan": {"slab_bytes": 16 * lanes, "slabs": slabs, "chunk_rows": chunk, "blocks_per_unit": bpu},
                           "sk_mean": float(skv.mean().item()),
                           "var_over_first_order": float(skv.var().item()) / (4.0 / (M * N))})
            del graph
    full = [p for p in points if p["N"] == cfg.E]
    line = {"metric": METRIC, "value": sum(p["frame_samples_per_s"] for p in full) / len(full), "unit": UNIT,
            "n_gpus": 1, "steps": K, "warmup": 1, "ms_per_step": sum(p["us_per_frame"] for p in full) / len(full) * 1e-3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8->u32/f64", "data": "synthetic",
            "config": {"workload": cfg.name + " (M, N) sweep", "E": cfg.E, "F": cfg.F, "T": cfg.T,
                       "value_is": "mean over the five N = 2048 points",
                       "l2": f"rotating over {nbuf} distinct frames of 512 MiB",
                       "launch": "per point: one CUDA graph of K sk_frame calls replayed for ~%.1f s, "
                                 "SK_FRAME_INPUTS_READY" % args.sweep_seconds,
                       "bytes_algorithmic": "T*F*N + 5 B per cell (N/E of the frame)",
                       "bytes_moved": "T*F*(slabs*slab_bytes) + 5 B per cell: whole slabs are fetched, slabs beyond "
                                      "first_n are never read",
                       "sweep": points},
            "roofline": {"bound": "hbm", "unit": "GB/s", "peak": peak, "peak_source": peak_src,
                         "achieved": min(p["gbs_on_bytes_moved"] for p in full),
                         "frac": min(p["frac_of_measured_peak"] for p in full), "traffic": None,
                         "note": "the slowest of the five N = 2048 points; per-point figures in config.sweep"},
            "gpu_launches": int(launches)}
    print(json.dumps(line))


def run_multi(args):
    """--op multi: sk_frame_multi: SK and mask at M, 2M, 4M, 8M from ONE pass
    over a config-2 frame, against the single-length sk_frame on the same frames."""
    import torch
    import paper_1808_10365_b200 as sk
    import sk_synth
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cfg = workload("cfg2")
    nlev = 4
    nbuf = 4
    bufs = [sk_synth.make_frame(cfg, device=dev, frame=i) for i in range(nbuf)]
    means = [null_mean(sk, sk_synth, cfg, dev, cfg.M << l) for l in range(nlev)]
    stream = torch.cuda.Stream(device=dev)
    K = args.steps
    with torch.cuda.stream(stream):
        ws = sk.workspace_for(cfg.T, cfg.F, cfg.E, cfg.M, dev, stream.cuda_stream, nlev)
        out = sk.sk_frame_multi(bufs[0], cfg.M, nlev, n_sigma=5.0, sk_means=means, workspace=ws, stream=stream)
    torch.cuda.synchronize()
    n0 = sk.sk_launch_count()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=stream):
        for i in range(K):
            sk.sk_frame_multi(bufs[i % nbuf], cfg.M, nlev, n_sigma=5.0, sk_means=means, out=out, workspace=ws,
                              stream=stream, inputs_ready=True)
    launches = sk.sk_launch_count() - n0
    with torch.cuda.stream(stream):
        graph.replay()
    torch.cuda.synchronize()
    ms, reps, _ = timed_replays(torch, graph, stream, 0.3, 2e-4, K, torch.cuda.synchronize)
    sampler = ClockSampler(0)
    sampler.start()
    ms, reps, clocks = timed_replays(torch, graph, stream, 1.0, ms * 1e-3 / (reps * K), K, torch.cuda.synchronize, sampler)
    sampler.stop_flag = True
    step_s = ms * 1e-3 / (reps * K)
    cells = sum((cfg.B >> l) * cfg.F for l in range(nlev))
    alg = cfg.nbytes + 5 * cells
    peak, peak_src = peaks()
    print(json.dumps({
        "op": "multi", "metric": METRIC, "value": cfg.nbytes / step_s, "unit": UNIT, "n_gpus": 1, "steps": K,
        "warmup": 1, "ms_per_step": step_s * 1e3, "higher_is_better": True, "data": "synthetic", "dtype": "u8->u32/f64",
        "config": {"workload": cfg.name, "E": cfg.E, "F": cfg.F, "T": cfg.T, "M": cfg.M, "lengths": [cfg.M << l for l in range(nlev)],
                   "sk_means": means, "flagged_fraction": [float(m.float().mean().item()) for m in out.mask],
                   "launch": f"one CUDA graph of K sk_frame_multi calls replayed {reps}x (~1 s), SK_FRAME_INPUTS_READY"},
        "roofline": {"bound": "hbm", "achieved": alg / step_s / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": alg / step_s / 1e9 / peak, "traffic": stored_traffic("multi"), "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": alg},
        "clocks": clocks, "gpu_launches": int(launches)}))


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    if args.op == "sim":
        return run_sim(args)
    if args.op == "cm":
        return run_cm(args)
    if args.op == "multi":
        return run_multi(args)
    if args.op == "ceiling":
        return run_ceiling(args)
    if args.op == "fig5":
        return run_fig5(args)
    if args.op == "fig6":
        return run_fig6(args)
    if args.op == "firstpass":
        return run_firstpass(args)
    if args.op == "memonly":
        return run_memonly(args)
    if args.op == "eager":
        return run_eager(args)
    if args.op != "frame":
        return run_aux(args)

    import torch
    import torch.distributed as dist

    import paper_1808_10365_b200 as sk
    import sk_synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the SK path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    sk.lib()
    if args.path == "ldg" or args.lanes:
        sk.plan_override(sk.SK_PLAN_LDG if args.path == "ldg" else sk.SK_PLAN_AUTO, args.lanes)
    if args.sweep:
        if world > 1:
            raise SystemExit("--sweep is a single-GPU line")
        return run_sweep(args, sk, sk_synth, torch, dev)

    cfg = workload(args.workload)
    K, W = args.steps, max(args.warmup, 3)
    frame_bytes = cfg.nbytes
    # distinct frames so that no step re-reads L2-resident data: > 4x the 126 MB L2, or 10 frames
    l2 = 126 * 1024 * 1024
    nbuf = 10 if frame_bytes > l2 else max(4, -(-5 * l2 // frame_bytes))
    free = torch.cuda.mem_get_info()[0]
    nbuf = max(2, min(nbuf, int(free * 0.8) // frame_bytes))
    # every rank draws its own frames (weak scaling: independent frames per GPU, no collective)
    bufs = [sk_synth.make_frame(cfg, device=dev, frame=fid) for fid in frame_ids(rank, nbuf)]
    sk_mean = null_mean(sk, sk_synth, cfg, dev)
    n_sigma = 5.0
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):              # workspace and outputs belong to the timed stream
        ws = sk.workspace_for(cfg.T, cfg.F, cfg.E, cfg.M, dev, stream.cuda_stream)
        out = sk.sk_frame(bufs[0], cfg.M, n_sigma=n_sigma, sk_mean=sk_mean, workspace=ws, stream=stream)
    torch.cuda.synchronize()

    # Every frame is resident and complete before the timed region starts.  Without --zero no step
    # writes any frame, so the SK_FRAME_INPUTS_READY promise (include/sk_b200.h) holds for every step.
    # With --zero every step excises its own frame and the frames recur every nbuf steps: step
    # i + nbuf reads what step i wrote.  The promise covers only what was written before the last call
    # made WITHOUT the flag, so the first step of every pass over the ring (i % nbuf == 0) is made
    # without it: that kernel waits for all earlier ones (the previous pass's excisions included)
    # before its first read, and the nbuf - 1 steps after it read frames last written before it.
    def step(i):
        ready = not args.serialize and not (args.zero and i % nbuf == 0)
        sk.sk_frame(bufs[i % nbuf], cfg.M, n_sigma=n_sigma, sk_mean=sk_mean, zero_flagged=args.zero,
                    out=out, workspace=ws, stream=stream, inputs_ready=ready)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(W):                           # W untimed warm-up steps (with --zero they excise the frames)
        step(i)
    if args.zero:
        for i in range(W, nbuf):
            step(i)
    torch.cuda.synchronize()
    flagged = float(out.mask.float().mean().item())

    # the graph holds a whole number of K-step passes (>= 200 steps), so that the pipeline bubble at
    # a graph boundary (the first kernel of a replay does not overlap the last of the previous one)
    # is amortised the same way whatever K is
    passes = max(1, -(-200 // K))
    G = K * passes
    n0 = sk.sk_launch_count()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=stream):
        for i in range(G):
            step(i)
    launches_per_replay = sk.sk_launch_count() - n0
    with torch.cuda.stream(stream):
        graph.replay()                           # one untimed replay (graph upload)
    torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()
    # ---- burst: the first ~20 ms after an idle pause.  The kernel draws enough power to reach
    # the 1 kW cap after ~40 ms of uninterrupted work; before that the SM clock is 1965 MHz.  This is
    # the counterpart of MEASURED_PEAKS.json's best-of-10 copy; it is NOT the headline.
    burst = None
    if args.burst_seconds > 0 and world == 1:
        ms0, reps0, _ = timed_replays(torch, graph, stream, 0.002, 2e-5 * max(1, frame_bytes >> 26), G, barrier)
        time.sleep(args.cooldown)
        bms, breps, bclk = timed_replays(torch, graph, stream, args.burst_seconds, ms0 * 1e-3 / (reps0 * G), G,
                                         barrier, sampler)
        burst = {"value": frame_bytes * G * breps / (bms * 1e-3), "unit": UNIT, "ms_per_step": bms / (G * breps),
                 "seconds": bms * 1e-3, "timed_steps": G * breps, "clocks": bclk,
                 "protocol": f"{args.cooldown} s idle, then the {G}-step graph replayed {breps}x"}
    # ---- steady state (the headline): settle for half the window, then time >= `--seconds` of
    # back-to-back replays inside one CUDA-event pair; the clocks reported are this window's.
    ms0, reps0, _ = timed_replays(torch, graph, stream, args.seconds / 2, 2e-5 * max(1, frame_bytes >> 26), G, barrier)
    ms, reps, clocks = timed_replays(torch, graph, stream, args.seconds, ms0 * 1e-3 / (reps0 * G), G, barrier, sampler)
    ms = max_over_ranks(ms, world, dev)
    steps_timed = G * reps
    launches = launches_per_replay * reps

    # ---- end to end through the C ABI with host buffers (copies inside the timed region)
    Ke = args.e2e_steps or min(K, 20)
    h_frames = [bufs[i % nbuf].cpu().pin_memory() for i in range(min(2, nbuf))]
    h_SK = torch.empty(cfg.B, cfg.F, dtype=torch.float32).pin_memory()
    h_mask = torch.empty(cfg.B, cfg.F, dtype=torch.uint8).pin_memory()
    d_stage = torch.empty_like(bufs[0])

    def e2e_step(i):
        sk.sk_frame_host(h_frames[i % len(h_frames)], cfg.M, h_SK, h_mask, d_stage, out.SK, out.mask,
                         n_sigma=n_sigma, sk_mean=sk_mean, zero_flagged=False, workspace=ws, stream=stream)

    e2e_step(0)
    barrier()
    t0 = time.perf_counter()
    for i in range(Ke):
        e2e_step(i)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, world, dev)
    # the same Ke frames as ONE sk_frames_host call: every step still uploads its own frame from pinned host
    # memory and reads its own SK and mask back, but the host waits once, not after every frame
    e2e_q = None
    try:
        hq_SK = torch.empty(Ke, cfg.B, cfg.F, dtype=torch.float32).pin_memory()
        hq_mask = torch.empty(Ke, cfg.B, cfg.F, dtype=torch.uint8).pin_memory()
        queue = [h_frames[i % len(h_frames)] for i in range(Ke)]
        sk.sk_frames_host(queue[:2], cfg.M, hq_SK[:2], hq_mask[:2], d_stage, out.SK, out.mask, n_sigma=n_sigma,
                          sk_mean=sk_mean, workspace=ws, stream=stream)
        barrier()
        t0 = time.perf_counter()
        sk.sk_frames_host(queue, cfg.M, hq_SK, hq_mask, d_stage, out.SK, out.mask, n_sigma=n_sigma, sk_mean=sk_mean,
                          workspace=ws, stream=stream)
        torch.cuda.synchronize()
        e2e_q = max_over_ranks(time.perf_counter() - t0, world, dev)
        if not (torch.equal(hq_SK[0], h_SK) or torch.equal(hq_SK[1], h_SK)):
            e2e_q = None                                   # never report a number from a call whose results differ
    except Exception as ex:                                # the extra can never cost the JSON line
        print("sk_frames_host e2e skipped:", ex, file=sys.stderr)
    sampler.stop_flag = True
    sampler.join(timeout=2)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = job_value(frame_bytes, world, steps_timed, ms)
    cells = cfg.B * cfg.F
    out_bytes = cells * 5
    flagged_bytes = int(flagged * frame_bytes) if args.zero else 0
    alg_bytes = frame_bytes + out_bytes + flagged_bytes          # per launch (1 B/sample read)
    peak, peak_src = peaks()
    achieved = alg_bytes / (ms * 1e-3 / steps_timed) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / steps_timed, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u8->u32/f64", "data": "synthetic",
        "config": {"workload": cfg.name, "E": cfg.E, "F": cfg.F, "T": cfg.T, "M": cfg.M, "N": cfg.E,
                   "n_sigma": n_sigma, "sk_mean": sk_mean, "zero_flagged": bool(args.zero),
                   "frame_bytes": frame_bytes, "flagged_fraction": flagged,
                   "l2": f"rotating over {nbuf} distinct frames ({nbuf * frame_bytes >> 20} MiB > 126 MB L2)",
                   "launch": f"one CUDA graph of {passes} x K = {G} sk_frame calls"
                             + ("" if args.serialize else ", SK_FRAME_INPUTS_READY (programmatic dependent launch)"),
                   "timed_region": f"steady state: the graph replayed {reps}x back to back inside one "
                                   f"CUDA-event pair ({ms * 1e-3:.2f} s, {steps_timed} steps), after "
                                   f"{args.seconds / 2:.2f} s of the same to settle the clocks",
                   "timed_steps": steps_timed, "replays": reps,
                   "parallelism": f"{world} independent replicas (no collective)"},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": stored_traffic(cfg.name + ("_zero" if args.zero else "")),
                     "peak_source": peak_src,
                     "frac_of_nominal_8000": achieved / 8000.0, "kernel": "sk_stream_kernel",
                     "algorithmic_bytes_per_launch": alg_bytes},
        "e2e": {"value": job_value(frame_bytes, world, Ke, (e2e_q or e2e_s) * 1e3), "unit": UNIT,
                "h2d_bytes_per_step": frame_bytes, "d2h_bytes_per_step": out_bytes, "steps": Ke,
                "api": ("sk_frames_host (C ABI, pinned host buffers): one call for the %d frames, every frame uploaded and "
                        "its SK and mask read back inside the timed region, one wait at the end" % Ke) if e2e_q
                       else "sk_frame_host (C ABI, pinned host buffers)",
                "per_frame_call": {"value": job_value(frame_bytes, world, Ke, e2e_s * 1e3), "unit": UNIT,
                                   "api": "sk_frame_host: one call and one wait per frame"}},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if world == 1:
        try:                                             # an extra: never let it cost the line
            line["roofline"]["sm_ceiling"] = sm_ceiling(sk, torch, dev, (clocks or {}).get("sm_mhz"),
                                                        (clocks or {}).get("sm_max_mhz"), value)
        except Exception as e:
            line["roofline"]["sm_ceiling"] = {"unavailable": str(e)}
    if args.zero:
        line["config"]["zero_note"] = ("the warm-up excises every frame once; the timed passes flag the same cells "
                                       "(their SK is 0) and overwrite them again: the traffic of a first pass")
    if burst is not None:
        burst["roofline_frac"] = burst["value"] * alg_bytes / frame_bytes / 1e9 / peak
        ceil = line["roofline"].get("sm_ceiling")
        if ceil and "subpartition_cycles_per_32_samples" in ceil and (burst["clocks"] or {}).get("sm_mhz"):
            burst["frac_of_sm_ceiling"] = burst["value"] * ceil["subpartition_cycles_per_32_samples"] / (
                ceil["subpartitions"] * 32 * burst["clocks"]["sm_mhz"] * 1e6)
        line["burst"] = burst

    if not args.no_cpu_baseline:
        from oracle import sk_oracle
        host = h_frames[0].numpy()
        max_bytes = 100 * 1024 * 1024
        blocks = max(1, min(cfg.B, max_bytes // (cfg.M * cfg.F * cfg.E)))
        host = host[: blocks * cfg.M]
        n, t0 = 0, time.perf_counter()
        while True:
            sk_oracle.frame(host, cfg.M, n_sigma=n_sigma, sk_mean=sk_mean)
            n += 1
            if time.perf_counter() - t0 >= args.cpu_seconds:
                break
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": host.size * n / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{n} passes over {blocks} of {cfg.B} blocks of {cfg.name} "
                                          f"({host.size} samples each), {dt:.1f} s, single thread; "
                                          f"host has {os.cpu_count()} cores"}
        # SURVEY 8(d)'s optional second baseline: the same oracle, unchanged, on every host core at once (one
        # thread per core, each on its own slab of whole blocks; ctypes releases the GIL around the C call)
        cores = os.cpu_count() or 1
        if cores > 1 and blocks >= cores:
            from concurrent.futures import ThreadPoolExecutor
            per = blocks // cores
            slabs = [host[i * per * cfg.M:(i + 1) * per * cfg.M] for i in range(cores)]
            secs = max(1.0, args.cpu_seconds / 2)
            t0 = time.perf_counter()

            def passes(h):
                k = 0
                while True:
                    sk_oracle.frame(h, cfg.M, n_sigma=n_sigma, sk_mean=sk_mean)
                    k += 1
                    if time.perf_counter() - t0 >= secs:
                        return k * h.size

            with ThreadPoolExecutor(cores) as ex:
                done = sum(ex.map(passes, slabs))
            dt = time.perf_counter() - t0
            line["cpu_baseline"]["all_cores"] = {"value": done / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                                 "sample": f"{cores} threads, each repeating its own {per}-block slab of the "
                                                           f"same frame for {dt:.1f} s"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
