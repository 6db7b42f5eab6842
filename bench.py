"""bench.py -- throughput of the PVFinder hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--precision tf32|bf16|fp16|fp32] [--events E] [--model run3|pileup] [--channels C]

One "step" = one pass of the whole hot path (interval sort, FC + segmented sum, UNet, peak finder:
SURVEY.md section 8a rows a0-a4) over one batch of synthetic events (BASELINE.json config 2: 16000
events of the Run-3-shaped model).  Prints ONE JSON line on rank 0.

* ``value``      events/s, inputs already resident in HBM, whole job (all ranks), device-timed.
* ``e2e``        same metric through pvf_run_host: host buffers (pinned), H2D + D2H inside the timing.
* ``roofline``   the UNet kernel (dominant): algorithmic FLOPs / its CUDA-event duration vs the
                 measured tensor peak of MEASURED_PEAKS.json (scaled to the precision used).
* ``cpu_baseline`` the CPU oracle, as it stands, on a bounded sample (rank 0, N = 1 only).
* ``--impl reference``: the oracle alone (this tier's reference arm), host cores only.

Multi-GPU: events are independent -> one replica per rank, each with its own
batch of E events, no data-path collective ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from pvf_inputs import make_events, make_weights, select_events  # noqa: E402

UNET_FLOP_PER_EVENT = {64: 2.5196e9, 32: 0.65562e9, 16: 0.17677e9}
SEEDS = {"run3": 1002, "pileup": 1003, "single": 1000}
METRIC = "PVFinder events/s (whole hot path) on B200"


def _config_id(args):
    """Which BASELINE.json config the flags correspond to (label only)."""
    if args.model == "single":
        return "0"
    if args.model == "pileup":
        return "3"
    if args.channels != 64 or args.precision in ("bf16", "fp16"):
        return "4"
    return "1" if args.events == 1000 else "2"


def _peaks_file():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled DURING the timed regions (B200_PROFILING.md); one background
    process for the whole run, summarised per wall-clock window."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw.instant,power.limit")

    def __init__(self, index=0):
        self.rows, self.proc, self.thread, self.index = [], None, None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def window(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        sm, mx, reasons, pw, plim = [], None, set(), [], None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in list(self.rows) if t0 <= t <= t1 + 0.1] or [r for (_, r) in list(self.rows)[-1:]]
        for r in rows:
            p = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(p[0])); mx = float(p[1])
            except Exception:
                continue
            for n, v in zip(names, p[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
            try:                                  # instantaneous board power: what sw_power_cap is about (the steps are power-bound)
                pw.append(float(p[6])); plim = float(p[7])
            except Exception:
                pass
        out = {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx,
               "reasons": sorted(reasons), "samples": len(sm)}
        if pw:
            out["power_w"] = float(np.median(pw))    # instantaneous samples (100 ms apart) inside the window: median and maximum
            out["power_w_max"] = float(np.max(pw))
            out["power_limit_w"] = plim
        return out

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()


def rank_seed(model, rank):
    """Every rank is a replica with its OWN batch (events are independent): no collective
    on the data path, weak scaling."""
    return SEEDS[model] + rank


def max_over_ranks(values, dist, device):
    """Device-timed durations -> the slowest rank's (the job is as fast as its slowest replica)."""
    import torch
    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_rate(world, events_per_rank, steps, ms):
    """Whole-job events/s: all ranks' events over the max-over-ranks time."""
    return world * events_per_rank * steps / (ms * 1e-3)


def run_oracle_sample(ev, w, n_sample):
    """Oracle timed as it stands on the first n_sample events, stage by stage: the same functions in the same
    16-event chunks as oracle.run.  Returns (events/s, seconds, threads, {stage: seconds})."""
    from oracle import pvf_oracle as O   # bench.py's cpu_baseline / reference legs may execute oracle/
    sub = select_events(ev, range(min(n_sample, ev.n_events)))
    off = sub.event_offsets.astype(np.int64)
    st = {"fc_hist": 0.0, "unet": 0.0, "peaks": 0.0}
    probs = np.zeros((sub.n_events, 4000), np.float32)
    t_all = time.perf_counter()
    for lo in range(0, sub.n_events, 16):
        hi = min(lo + 16, sub.n_events)
        t0 = time.perf_counter()
        H, _ = O.histogram(sub.feat[:, off[lo]:off[hi]], off[lo:hi + 1] - off[lo], w.fc_w, w.fc_b)
        t1 = time.perf_counter()
        probs[lo:hi] = O.unet_probs(H, w.conv_w, w.conv_b)
        st["fc_hist"] += t1 - t0
        st["unet"] += time.perf_counter() - t1
    t0 = time.perf_counter()
    O.find_peaks(probs)
    st["peaks"] = time.perf_counter() - t0
    dt = time.perf_counter() - t_all
    try:
        import threadpoolctl
        thr = max([p.get("num_threads", 1) for p in threadpoolctl.threadpool_info()] or [1])
    except Exception:
        thr = os.cpu_count() or 1
    return sub.n_events / dt, dt, int(thr), st


def main_reference(args, rank, world):
    """This tier's reference arm: the CPU oracle on host cores; rank 0 only."""
    if rank != 0:
        return
    ev = make_events(args.model, args.events, SEEDS[args.model])
    w = bench_weights(args.weights, args.channels)
    n_sample = args.ref_sample
    for _ in range(args.warmup):
        run_oracle_sample(ev, w, n_sample)
    t0 = time.perf_counter()
    thr = 1
    for _ in range(args.steps):
        _, _, thr, _ = run_oracle_sample(ev, w, n_sample)
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    sample = f"first {n_sample} of {args.events} events per step, oracle.run (numpy float64) as it stands"
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json config 2: {args.events} events, model {args.model}, "
                               f"UNet {args.channels} ch (bounded sample per step)", "sample_events": n_sample},
        "cpu_baseline": {"value": value, "unit": "events/s", "cores": thr, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


def nonempty_intervals(ev):
    """Number of (event, interval) pairs that hold at least one in-range track (bookkeeping for byte / FLOP
    accounting only; same float32 recipe as DESIGN.md reading R2)."""
    z = ev.feat[0]
    iv = np.floor((z.astype(np.float32) + np.float32(200.0)) * np.float32(0.1)).astype(np.int64)
    evi = np.repeat(np.arange(ev.n_events), np.diff(ev.event_offsets))
    ok = np.isfinite(z) & (iv >= 0) & (iv < 40)
    return int(np.unique(evi[ok] * 40 + iv[ok]).size)


def tensor_peak(peaks, peaks_src, prec, tf32_measured, sustained=True):
    """(peak TFLOP/s, note) for the UNet roofline: MEASURED_PEAKS.json's bf16 figure for the 16-bit modes; for TF32 the
    figure this run measured (torch.matmul 8192^3, TF32 allowed -- measurement only), the derived one kept beside it."""
    key = "bf16_tflops_sustained" if sustained else "bf16_tflops"
    if prec in ("bf16", "fp16"):
        return peaks[key], f"{peaks_src} {key} {peaks[key]} TFLOP/s (MEASURED_PEAKS.json)"
    if tf32_measured is not None:
        k = "sustained" if sustained else "burst"
        return tf32_measured[k], f"measured in this run: torch.matmul 8192^3 TF32, {k}"
    return peaks[key] * 1.1 / 2.25, f"{peaks_src} {key} {peaks[key]} x nominal tf32/bf16 ratio 1.1/2.25 (derived)"


def measure_tf32_peak(torch, seconds=4.0):
    """cuBLAS TF32 matmul 8192^3, the way MEASURED_PEAKS.json measures bf16: best of 10 (burst) and back to back
    for `seconds` (sustained).  Measurement only -- never on the product path, outside every timed region."""
    n = 8192
    old = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = True
    try:
        a = torch.randn(n, n, device="cuda")
        b = torch.randn(n, n, device="cuda")
        c = torch.empty(n, n, device="cuda")
        for _ in range(3):
            torch.matmul(a, b, out=c)
        torch.cuda.synchronize()
        flop = 2.0 * n ** 3
        best = 0.0
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            torch.matmul(a, b, out=c)
            e1.record()
            e1.synchronize()
            best = max(best, flop / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0, reps = time.time(), 0
        e0.record()
        while time.time() - t0 < seconds:
            for _ in range(20):
                torch.matmul(a, b, out=c)
            reps += 20
            torch.cuda.synchronize()
        e1.record()
        e1.synchronize()
        sustained = reps * flop / (e0.elapsed_time(e1) * 1e-3) / 1e12
        del a, b, c
        return {"burst": best, "sustained": sustained, "how": f"torch.matmul {n}^3 fp32 inputs, allow_tf32; best of 10 / {reps} back to back"}
    finally:
        torch.backends.cuda.matmul.allow_tf32 = old


def bench_weights(kind, channels):
    """make_weights, plus the diagnostic kind "zero-conv": `peaky` with every conv weight and bias set to zero, so that
    every MMA operand of the UNet is zero.  The launch sequence and the executed instructions are identical; what changes is
    the switching activity of the data paths -- the difference in stage time is the data-dependent share of the power the
    1 kW cap charges (profiles/r02_experiments.md, section on the power cap).  Never a headline configuration."""
    w = make_weights("peaky" if kind == "zero-conv" else kind, 1, channels)
    if kind == "zero-conv":
        w.conv_w = [np.zeros_like(a) for a in w.conv_w]
        w.conv_b = [np.zeros_like(a) for a in w.conv_b]
    return w


class Workload:
    """One configuration of the hot path on the device: events + weights + handle + output buffers."""

    def __init__(self, torch, PVFinder, *, model, events, seed, precision, channels=64, split_mask=None, elide=False,
                 cta_pair=True, margin=0.0, weights="peaky", host_io=False, l2_chunk_events=0, stage_timing=True):
        self.torch = torch
        self.ev = make_events(model, events, seed)
        self.w = bench_weights(weights, channels)
        self.E, self.precision, self.channels, self.elide = events, precision, channels, elide
        self.split = split_mask if split_mask is not None else (1 if precision == "tf32" else 0)
        extra = {}
        if l2_chunk_events:
            extra["l2_chunk_events"] = int(l2_chunk_events)
        self.stage_timing = stage_timing
        self.pvf = PVFinder(self.w, max_events=events, max_tracks=max(self.ev.n_tracks, 1), precision=precision,
                            split_mask=self.split, stage_timing=stage_timing, host_io=host_io, elide_empty=elide,
                            cta_pair=bool(cta_pair), boundary_margin_mm=margin, **extra)
        self.feat = torch.from_numpy(self.ev.feat).cuda()
        self.off = torch.from_numpy(self.ev.event_offsets).cuda()
        self.probs = torch.empty(events, 4000, device="cuda")
        self.pk = self.pvf.alloc_peaks(events)
        self.stream = torch.cuda.Stream()

    def run(self):
        self.pvf.run(self.feat, self.off, self.E, self.probs, self.pk, stream=self.stream)

    def timed(self, steps, warmup, barrier=None):
        """(total ms over `steps` runs, mean stage ms [sort, fc+sum, unet, peaks], wall window)."""
        torch = self.torch
        for _ in range(warmup):
            self.run()
        self.stream.synchronize()
        try:
            self.pvf.stage_times_ms()            # reset the stage-time ring
        except Exception:
            pass
        if barrier:
            barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.time()
        e0.record(self.stream)
        for _ in range(steps):
            self.run()
        e1.record(self.stream)
        self.stream.synchronize()
        t1 = time.time()
        if barrier:
            barrier()
        return e0.elapsed_time(e1), (self.pvf.stage_times_ms() if self.stage_timing else None), (t0, t1)

    def close(self):
        self.pvf.destroy()
        del self.feat, self.off, self.probs, self.pk


def run_variants(torch, PVFinder, args, sampler, peaks, peaks_src, tf32_measured):
    """Every other named configuration of BASELINE.json on the same line (3 warm-ups + 5 steps each): config 2 in
    BF16 / FP16, config 3, config 4 at C = 32 / 16, config 1 (1000 events), config 0 (one event: latency), the FP32
    path, and the separate modes (empty-interval elision, L2-resident histogram chunks)."""
    V = []
    specs = [
        dict(name="config2_bf16", model="run3", events=16000, seed=SEEDS["run3"], precision="bf16"),
        dict(name="config2_fp16", model="run3", events=16000, seed=SEEDS["run3"], precision="fp16"),
        # FP16 operands with the e1 layer split into two FP16 pieces: meets north_star's TF32 tolerance (1e-3), tests fp16s
        dict(name="config2_fp16_e1split", model="run3", events=16000, seed=SEEDS["run3"], precision="fp16", split_mask=1),
        dict(name="config3_tf32", model="pileup", events=16000, seed=SEEDS["pileup"], precision="tf32"),
        dict(name="config4_bf16_c32", model="run3", events=16000, seed=1004, precision="bf16", channels=32),
        dict(name="config4_bf16_c16", model="run3", events=16000, seed=1004, precision="bf16", channels=16),
        dict(name="config1_tf32", model="run3", events=1000, seed=1001, precision="tf32"),
        dict(name="config2_tf32_elide_empty", model="run3", events=16000, seed=SEEDS["run3"], precision="tf32", elide=True),
        dict(name="config2_tf32_l2_chunks_1024", model="run3", events=16000, seed=SEEDS["run3"], precision="tf32",
             l2_chunk_events=1024),
        dict(name="config2_fp32", model="run3", events=16000, seed=SEEDS["run3"], precision="fp32"),
        dict(name="config2_fp32_cuda_cores", model="run3", events=4000, seed=SEEDS["run3"], precision="fp32", cta_pair=False),
        # diagnostic, never a headline: the same launches with all-zero UNet operands do not reach the 1 kW cap -- the
        # stage time at the maximum clock, i.e. what the power cap costs (profiles/r02_experiments.md section 8)
        dict(name="config2_tf32_zero_operands_power_cap_diagnostic", model="run3", events=16000, seed=SEEDS["run3"],
             precision="tf32", weights="zero-conv"),
    ]
    for sp in specs:
        name = sp.pop("name")
        try:
            wl = Workload(torch, PVFinder, **sp)
            ms, stage, win = wl.timed(5, 3)
            E, ch, prec = wl.E, wl.channels, wl.precision
            flop = UNET_FLOP_PER_EVENT[ch] * E
            rec = {"name": name, "events": E, "tracks": wl.ev.n_tracks, "precision": prec, "channels": ch,
                   "events_per_s": E * 5 / (ms * 1e-3), "ms_per_step": ms / 5, "us_per_event": ms * 1e3 / (5 * E),
                   "stage_ms": {"sort": stage[0], "fc_hist": stage[1], "unet": stage[2], "peaks": stage[3]},
                   "split_mask": wl.split, "steps": 5, "warmup": 3, "clocks": sampler.window(*win)}
            if wl.elide:
                ne = nonempty_intervals(wl.ev) / (E * 40.0)
                rec["nonempty_interval_fraction"] = ne
                flop *= ne                                         # executed-FLOP accounting: a separate mode
            if prec == "fp32" and not sp.get("cta_pair", True):
                pk_, note = 148 * 128 * 2 * 1.965e9 / 1e12, "FP32 FMA peak: 148 SM x 128 lanes x 2 x 1.965 GHz"
            else:
                pk_, note = tensor_peak(peaks, peaks_src, prec, tf32_measured, sustained=E >= 4000)
                if prec == "fp32":
                    note += ("; FP32-accurate mode: nominal FLOPs against the TF32 peak -- every product costs one kind::tf32 "
                             "and one kind::f16 MMA (2/3 and 1/3 of the executed tensor time), so 0.67 is this mode's ceiling")
            if sp.get("weights") == "zero-conv":
                pk_, note = 1100.0, ("nominal dense TF32 peak at 1.965 GHz (this run is not power-capped: compare the "
                                                  "clocks entry with the headline's)")
            rec["unet_tflops"] = flop / (stage[2] * 1e-3) / 1e12
            rec["unet_frac"] = rec["unet_tflops"] / pk_
            rec["unet_peak"] = pk_
            rec["unet_peak_source"] = note
            wl.close()
            V.append(rec)
        except Exception as exc:   # a variant must never take the headline line down
            V.append({"name": name, "error": repr(exc)[:200]})
        torch.cuda.empty_cache()
    # config 0: one event, per-call latency (sub-400 us budget per event)
    for tag, prec, split in (("tf32", "tf32", None), ("fp16", "fp16", None), ("fp16_e1split", "fp16", 1), ("fp32", "fp32", None)):
        try:
            wl = Workload(torch, PVFinder, model="single", events=1, seed=SEEDS["single"], precision=prec, split_mask=split)
            n = 200
            _, stage, _ = wl.timed(n, 20)                          # per-stage split: stage timing on (kernels not chained)
            wl.close()
            wl = Workload(torch, PVFinder, model="single", events=1, seed=SEEDS["single"], precision=prec, split_mask=split,
                          stage_timing=False)
            ms, _, win = wl.timed(n, 20)                           # the latency: no events between the kernels, PDL chain
            iso = []
            for _ in range(30):                                    # isolated calls: launch gaps included
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(wl.stream)
                wl.run()
                e1.record(wl.stream)
                e1.synchronize()
                iso.append(e0.elapsed_time(e1) * 1e3)
            # the same call captured once in a CUDA graph (pvf_run allocates nothing and never synchronises; the
            # programmatic dependent launches become programmatic edges) and replayed: what a per-event caller would do
            graph_us, graph_iso = None, None
            try:
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=wl.stream):
                    wl.run()
                with torch.cuda.stream(wl.stream):
                    for _ in range(20):
                        g.replay()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(wl.stream)
                    for _ in range(n):
                        g.replay()
                    e1.record(wl.stream)
                    e1.synchronize()
                    graph_us = e0.elapsed_time(e1) * 1e3 / n
                    gi = []
                    for _ in range(30):
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record(wl.stream)
                        g.replay()
                        e1.record(wl.stream)
                        e1.synchronize()
                        gi.append(e0.elapsed_time(e1) * 1e3)
                    graph_iso = float(np.median(gi))
                del g
            except Exception:
                pass
            V.append({"name": f"config0_{tag}_latency", "events": 1, "tracks": wl.ev.n_tracks, "precision": prec,
                      "split_mask": wl.split, "channels": 64, "latency_graph_us": graph_us,
                      "latency_graph_isolated_us_median": graph_iso, "latency_us": ms * 1e3 / n, "latency_isolated_us_median": float(np.median(iso)),
                      "how": f"{n} back-to-back pvf_run calls on one stream (device time / call), kernels chained by programmatic "
                             "dependent launch; 30 isolated calls; stage_us from a second handle with stage timing (no PDL)",
                      "stage_us": {"sort": stage[0] * 1e3, "fc_hist": stage[1] * 1e3, "unet": stage[2] * 1e3,
                                   "peaks": stage[3] * 1e3},
                      "launches_per_run": wl.pvf.launches_per_run(1), "clocks": sampler.window(*win)})
            wl.close()
        except Exception as exc:
            V.append({"name": f"config0_{tag}_latency", "error": repr(exc)[:200]})
    return V


def main_ours(args, rank, world, local_rank):
    import torch
    from paper_2602_19959_b200 import PVFinder   # raises if libpvf.so is missing: no CPU fallback

    if not torch.cuda.is_available():
        raise SystemExit("bench.py (impl ours) needs a CUDA device; there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    E = args.events
    split = args.split_mask if args.split_mask >= 0 else None
    wl = Workload(torch, PVFinder, model=args.model, events=E, seed=rank_seed(args.model, rank), precision=args.precision,
                  channels=args.channels, split_mask=split, elide=args.elide_empty, cta_pair=args.cta_pair,
                  margin=args.boundary_margin, weights=args.weights, host_io=True, l2_chunk_events=args.l2_chunk_events)
    ev, w, pvf, stream = wl.ev, wl.w, wl.pvf, wl.stream

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident timing (inputs in HBM; 107 MB features + 2 GB H: larger than L2)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(1.0)
    ms, stage, win = wl.timed(args.steps, args.warmup, barrier)
    clocks = sampler.window(*win) if rank == 0 else None
    launches = pvf.launches_per_run(E) * args.steps

    # ---------------- end to end through pvf_run_host: pinned host buffers, H2D + D2H inside, every step timed
    hfeat = torch.from_numpy(ev.feat).pin_memory()
    hoff = torch.from_numpy(ev.event_offsets).pin_memory()
    hprobs = torch.empty(E, 4000).pin_memory()
    hpk = pvf.alloc_peaks(E, pinned=True)
    pvf.run_host(hfeat, hoff, E, hprobs, hpk, stream=stream)
    barrier()
    n_e2e = max(1, min(args.steps, args.e2e_steps))
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(n_e2e + 1)]
    marks[0].record(stream)
    for k in range(n_e2e):
        pvf.run_host(hfeat, hoff, E, hprobs, hpk, stream=stream)   # synchronises the stream itself
        marks[k + 1].record(stream)
    stream.synchronize()
    barrier()
    ms_e2e = marks[0].elapsed_time(marks[-1])
    e2e_steps_ms = [marks[k].elapsed_time(marks[k + 1]) for k in range(n_e2e)]
    h2d = int(hfeat.numel() * 4 + hoff.numel() * 4)
    d2h = int(hprobs.numel() * 4 + sum(v.numel() * v.element_size() for v in hpk.values()))
    del hfeat, hprobs

    ms, ms_e2e = max_over_ranks([ms, ms_e2e], dist, "cuda")
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    value = whole_job_rate(world, E, args.steps, ms)
    e2e_value = whole_job_rate(world, E, n_e2e, ms_e2e)

    peaks, peaks_src = _peaks_file()
    nonempty = nonempty_intervals(ev)
    flop = UNET_FLOP_PER_EVENT[args.channels] * E
    if args.elide_empty:
        flop *= nonempty / (E * 40.0)     # executed-FLOP accounting: only the intervals that hold a track go through the UNet
    tf32_measured = None
    variants = None
    if world == 1 and not args.no_variants:
        wl.close()
        torch.cuda.empty_cache()
        try:
            tf32_measured = measure_tf32_peak(torch)
        except Exception as exc:
            tf32_measured = None
            print(f"bench: TF32 peak measurement failed: {exc!r}", file=sys.stderr)
        variants = run_variants(torch, PVFinder, args, sampler, peaks, peaks_src, tf32_measured)
    sampler.stop()
    unet_s = stage[2] * 1e-3
    if args.precision == "fp32" and not args.cta_pair:
        bound, peak = "alu", 148 * 128 * 2 * 1.965e9 / 1e12
        peak_note = "FP32 FMA: 148 SM x 128 lanes x 2 FLOP x 1.965 GHz (B200_PROFILING.md unit counts)"
    else:
        bound = "tensor"
        peak, peak_note = tensor_peak(peaks, peaks_src, args.precision, tf32_measured, sustained=E >= 4000)
    achieved = flop / unet_s / 1e12
    traffic, tensor_pct, traffic_src = None, None, None
    for fn in ("r02_roofline_traffic.json.txt", "r01_roofline_traffic.json.txt"):
        try:
            with open(os.path.join(ROOT, "profiles", fn)) as f:
                rec = json.load(f)[f"{args.precision}_c{args.channels}"]
            traffic = rec["bytes_per_event"] * E
            tensor_pct = rec.get("tensor_pipe_active_pct")
            traffic_src = f"profiles capture (profiles/{fn}: ncu --set full on a 4000-event batch) x events; not observed in this run"
            break
        except Exception:
            continue
    # FC + sum: bytes the stage must move.  The tensor-core FC kernel writes only the intervals that hold a track
    # (the UNet takes the others as zeros), so its bytes are features + non-empty histograms; the canonical figure
    # of SURVEY.md 8(d) (all 40 intervals written) is kept beside it.
    fc_s = stage[1] * 1e-3
    bytes_alg = ev.n_tracks * 36 + E * 40 * 800 * 4
    bytes_moved = ev.n_tracks * 36 + (nonempty if (args.precision != "fp32" or args.cta_pair) else E * 40) * 800 * 4
    roof = {"kernel": "unet", "bound": bound, "achieved": achieved, "peak": peak,
            "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
            "peak_source": peak_note,
            # BASELINE.json's metric also asks for the UNet tensor-pipe utilisation: a profiler counter, so it is
            # the value of the committed ncu capture (profiles/), not something measured in this run
            "tensor_pipe_active_pct_ncu": tensor_pct, "tensor_pipe_source": traffic_src}
    roof["frac_vs_nominal_dense_peak"] = achieved / {"tf32": 1100.0, "bf16": 2250.0, "fp16": 2250.0, "fp32": 1100.0}[args.precision] \
        if bound == "tensor" else None      # B200_PROFILING.md nominal dense peaks at the maximum clock, for context
    if args.precision == "tf32":
        d_s = peaks["bf16_tflops_sustained"] * 1.1 / 2.25
        d_b = peaks["bf16_tflops"] * 1.1 / 2.25
        roof["peak_measured_tf32"] = tf32_measured
        roof["frac_vs_derived_sustained"] = achieved / d_s      # bf16 sustained x nominal 1.1/2.25 (round 1's denominator)
        roof["frac_vs_derived_burst"] = achieved / d_b
        if tf32_measured is not None:
            roof["frac_vs_measured_burst"] = achieved / tf32_measured["burst"]
    out = {
        "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": {"fp32": "f32", "tf32": "tf32", "bf16": "bf16", "fp16": "f16"}[args.precision],
        "data": "synthetic",
        "config": {"workload": f"BASELINE.json config {_config_id(args)}: {E} events/GPU, "
                               f"model {args.model}, {ev.n_tracks} tracks, UNet {args.channels} ch, weights {args.weights}",
                   "precision": args.precision, "split_mask": wl.split,
                   "elide_empty_intervals": bool(args.elide_empty), "unet_cta_pair": bool(args.cta_pair), "boundary_margin_mm": args.boundary_margin,
                   "l2_chunk_events": args.l2_chunk_events, "nonempty_interval_fraction": nonempty / (E * 40.0),
                   "cache": ("inputs larger than L2 (107 MB features, 2 GB histogram per step)" if E >= 2000 else
                             "small batch: inputs fit in L2 (latency-style measurement)")},
        "us_per_event": ms * 1e3 / (args.steps * E),
        "stage_ms": {"sort": stage[0], "fc_hist": stage[1], "unet": stage[2], "peaks": stage[3]},
        "stage_us_per_event": {k: v * 1e3 / E for k, v in zip(("sort", "fc_hist", "unet", "peaks"), stage)},
        "roofline": roof,
        "roofline_fc_hist": {"bound": "hbm", "achieved": bytes_moved / fc_s / 1e9,
                             "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": bytes_moved / fc_s / 1e9 / peaks["hbm_gbs"],
                             "bytes": "features 36 B/track + histograms of the non-empty intervals (what this kernel writes)",
                             "achieved_canonical": bytes_alg / fc_s / 1e9,
                             "frac_canonical": bytes_alg / fc_s / 1e9 / peaks["hbm_gbs"],
                             "bytes_canonical": "SURVEY.md 8(d): features + all 40 intervals x 800 floats per event"},
        # the FC + sum stage is bound by its 1600 SFU operations per track (800 x (ex2 + lg2)), not by HBM (DESIGN.md
        # section 4.2): 148 SMs x 16 SFU lanes x 1.965 GHz = 4.65 Tops/s
        "roofline_fc_hist_alu": {"bound": "alu", "achieved": ev.n_tracks * 1600 / fc_s / 1e12,
                                 "peak": 148 * 16 * 1.965e9 / 1e12, "unit": "T SFU-op/s",
                                 "frac": ev.n_tracks * 1600 / fc_s / (148 * 16 * 1.965e9),
                                 "peak_source": "148 SMs x 16 SFU lanes/clk x 1.965 GHz max SM clock (guide unit counts)"},
        "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": n_e2e, "api": "pvf_run_host (pinned host buffers)",
                "ms_per_step_min_mean_max": [min(e2e_steps_ms), ms_e2e / n_e2e, max(e2e_steps_ms)]},
        "gpu_launches": launches, "clocks": clocks,
    }
    if variants is not None:
        out["variants"] = variants
    if world == 1 and not args.no_cpu_baseline:
        v, dt, thr, st = run_oracle_sample(ev, w, args.cpu_sample)
        n_s = min(args.cpu_sample, E)
        out["cpu_baseline"] = {"value": v, "unit": "events/s", "cores": thr, "kind": "oracle",
                               "sample": f"first {n_s} events of the batch, {dt:.1f} s",
                               "stage_s": st, "stage_us_per_event": {k: 1e6 * x / n_s for k, x in st.items()},
                               "stages": "fc_hist = interval assignment + FC + histogram sum; unet incl. sigmoid; peaks"}
    print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--precision", default=os.environ.get("PVF_BENCH_PRECISION", "tf32"), choices=["fp32", "tf32", "bf16", "fp16"])
    ap.add_argument("--split-mask", type=int, default=-1)
    ap.add_argument("--events", type=int, default=16000)
    ap.add_argument("--model", default="run3", choices=["run3", "pileup", "single"])
    ap.add_argument("--weights", default="peaky", choices=["peaky", "rand", "zero-conv"])
    ap.add_argument("--channels", type=int, default=64, choices=[64, 32, 16])
    ap.add_argument("--cpu-sample", type=int, default=192)   # ~13 s of oracle time on 16 host threads
    ap.add_argument("--ref-sample", type=int, default=16)
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-variants", action="store_true",
                    help="skip the other named configurations and the TF32 peak measurement (N = 1 only anyway)")
    ap.add_argument("--boundary-margin", type=float, default=0.0,
                    help="NEXT-1 mode (mm): boundary tracks contribute to two intervals, PAPER.md:49")
    ap.add_argument("--cta-pair", type=int, default=1, choices=[0, 1],
                    help="UNet as clusters of two CTAs sharing every MMA (cta_group::2)")
    ap.add_argument("--l2-chunk-events", type=int, default=0,
                    help="NEXT-2 mode: histograms through a chunk-sized, L2-resident buffer (pvf_config.l2_chunk_events)")
    ap.add_argument("--elide-empty", action="store_true",
                    help="NEXT-2 mode: UNet only over non-empty intervals (reported with executed-FLOP accounting)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        main_reference(args, rank, world)
    else:
        main_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
