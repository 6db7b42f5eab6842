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
    """nvidia-smi clocks + throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

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

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.1] or [r for (_, r) in self.rows]
        for r in rows:
            p = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(p[0])); mx = float(p[1])
            except Exception:
                continue
            for n, v in zip(names, p[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx,
                "reasons": sorted(reasons), "samples": len(sm)}


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
    """Oracle timed as it stands on the first n_sample events.  Returns (events/s, seconds, threads)."""
    from oracle import pvf_oracle as O   # bench.py's cpu_baseline / reference legs may execute oracle/
    sub = select_events(ev, range(min(n_sample, ev.n_events)))
    t0 = time.perf_counter()
    O.run(sub.feat, sub.event_offsets, w)
    dt = time.perf_counter() - t0
    try:
        import threadpoolctl
        thr = max([p.get("num_threads", 1) for p in threadpoolctl.threadpool_info()] or [1])
    except Exception:
        thr = os.cpu_count() or 1
    return sub.n_events / dt, dt, int(thr)


def main_reference(args, rank, world):
    """This tier's reference arm: the CPU oracle on host cores; rank 0 only."""
    if rank != 0:
        return
    ev = make_events(args.model, args.events, SEEDS[args.model])
    w = make_weights(args.weights, 1, args.channels)
    n_sample = args.ref_sample
    for _ in range(args.warmup):
        run_oracle_sample(ev, w, n_sample)
    t0 = time.perf_counter()
    thr = 1
    for _ in range(args.steps):
        _, _, thr = run_oracle_sample(ev, w, n_sample)
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
    ev = make_events(args.model, E, rank_seed(args.model, rank))
    w = make_weights(args.weights, 1, args.channels)
    split = args.split_mask if args.split_mask >= 0 else (1 if args.precision == "tf32" else 0)
    pvf = PVFinder(w, max_events=E, max_tracks=ev.n_tracks, precision=args.precision, split_mask=split,
                   stage_timing=True, host_io=True, elide_empty=args.elide_empty,
                   cta_pair=bool(args.cta_pair) and args.precision != "fp32",
                   boundary_margin_mm=args.boundary_margin)
    feat = torch.from_numpy(ev.feat).cuda()
    off = torch.from_numpy(ev.event_offsets).cuda()
    probs = torch.empty(E, 4000, device="cuda")
    pk = pvf.alloc_peaks(E)
    stream = torch.cuda.Stream()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident timing (inputs in HBM; 107 MB features + 2 GB H: larger than L2)
    for _ in range(args.warmup):
        pvf.run(feat, off, E, probs, pk, stream=stream)
    stream.synchronize()
    try:
        pvf.stage_times_ms()            # reset the stage-time ring
    except Exception:
        pass
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(1.0)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_wall0 = time.time()
    e0.record(stream)
    for _ in range(args.steps):
        pvf.run(feat, off, E, probs, pk, stream=stream)
    e1.record(stream)
    stream.synchronize()
    t_wall1 = time.time()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    stage = pvf.stage_times_ms()        # mean over the timed runs: sort, FC+sum, UNet, peaks
    launches = pvf.launches_per_run(E) * args.steps

    # ---------------- end to end through pvf_run_host: pinned host buffers, H2D + D2H inside
    hfeat = torch.from_numpy(ev.feat).pin_memory()
    hoff = torch.from_numpy(ev.event_offsets).pin_memory()
    hprobs = torch.empty(E, 4000).pin_memory()
    hpk = pvf.alloc_peaks(E, pinned=True)
    pvf.run_host(hfeat, hoff, E, hprobs, hpk, stream=stream)
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_e2e = max(1, min(args.steps, args.e2e_steps))
    f0.record(stream)
    for _ in range(n_e2e):
        pvf.run_host(hfeat, hoff, E, hprobs, hpk, stream=stream)   # synchronises the stream itself
    f1.record(stream)
    stream.synchronize()
    barrier()
    ms_e2e = f0.elapsed_time(f1)
    h2d = int(hfeat.numel() * 4 + hoff.numel() * 4)
    d2h = int(hprobs.numel() * 4 + sum(v.numel() * v.element_size() for v in hpk.values()))

    ms, ms_e2e = max_over_ranks([ms, ms_e2e], dist, "cuda")
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    value = whole_job_rate(world, E, args.steps, ms)
    e2e_value = whole_job_rate(world, E, n_e2e, ms_e2e)

    peaks, peaks_src = _peaks_file()
    flop = UNET_FLOP_PER_EVENT[args.channels] * E
    nonempty = None
    if args.elide_empty:
        # executed-FLOP accounting: only the intervals that hold a track go through the UNet
        z = ev.feat[0]
        iv = np.floor((z.astype(np.float32) + np.float32(200.0)) * np.float32(0.1)).astype(np.int64)   # bookkeeping only
        evi = np.repeat(np.arange(E), np.diff(ev.event_offsets))
        ok = np.isfinite(z) & (iv >= 0) & (iv < 40)
        nonempty = float(np.unique(evi[ok] * 40 + iv[ok]).size) / (E * 40)
        flop *= nonempty
    unet_s = stage[2] * 1e-3
    if args.precision == "fp32":
        bound, peak = "alu", 148 * 128 * 2 * 1.965e9 / 1e12
        peak_note = "FP32 FMA: 148 SM x 128 lanes x 2 FLOP x 1.965 GHz (B200_PROFILING.md unit counts)"
    else:
        ratio = 1.0 if args.precision in ("bf16", "fp16") else 1.1 / 2.25
        bound, peak = "tensor", peaks["bf16_tflops_sustained"] * ratio
        peak_note = (f"{peaks_src} bf16 sustained {peaks['bf16_tflops_sustained']} TFLOP/s"
                     + ("" if ratio == 1.0 else " x nominal tf32/bf16 ratio 1.1/2.25"))
    achieved = flop / unet_s / 1e12
    traffic = None   # DRAM bytes per launch from the committed ncu --set full capture (per event x E)
    tensor_pct = None
    try:
        with open(os.path.join(ROOT, "profiles", "r01_roofline_traffic.json.txt")) as f:
            rec = json.load(f)[f"{args.precision}_c{args.channels}"]
            traffic = rec["bytes_per_event"] * E
            tensor_pct = rec.get("tensor_pipe_active_pct")
    except Exception:
        pass
    hbm_bytes_fc = (ev.n_tracks * 36 + E * 40 * 800 * 4)
    out = {
        "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": {"fp32": "f32", "tf32": "tf32", "bf16": "bf16", "fp16": "f16"}[args.precision],
        "data": "synthetic",
        "config": {"workload": f"BASELINE.json config {_config_id(args)}: {E} events/GPU, "
                               f"model {args.model}, {ev.n_tracks} tracks, UNet {args.channels} ch, weights {args.weights}",
                   "precision": args.precision, "split_mask": split,
                   "elide_empty_intervals": bool(args.elide_empty), "unet_cta_pair": bool(args.cta_pair) and args.precision != "fp32", "boundary_margin_mm": args.boundary_margin, "nonempty_interval_fraction": nonempty,
                   "cache": ("inputs larger than L2 (107 MB features, 2 GB histogram per step)" if E >= 2000 else
                             "small batch: inputs fit in L2 (latency-style measurement)")},
        "us_per_event": ms * 1e3 / (args.steps * E),
        "stage_ms": {"sort": stage[0], "fc_hist": stage[1], "unet": stage[2], "peaks": stage[3]},
        "stage_us_per_event": {k: v * 1e3 / E for k, v in zip(("sort", "fc_hist", "unet", "peaks"), stage)},
        "roofline": {"kernel": "unet", "bound": bound, "achieved": achieved, "peak": peak,
                     "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic, "peak_source": peak_note,
                     # BASELINE.json's metric also asks for the UNet tensor-pipe utilisation: a profiler counter, so it is
                     # the value of the committed ncu capture (profiles/), not something measured in this run
                     "tensor_pipe_active_pct_ncu": tensor_pct},
        "roofline_fc_hist": {"bound": "hbm", "achieved": hbm_bytes_fc / (stage[1] * 1e-3) / 1e9,
                             "peak": peaks["hbm_gbs"], "unit": "GB/s",
                             "frac": hbm_bytes_fc / (stage[1] * 1e-3) / 1e9 / peaks["hbm_gbs"]},
        # the FC + sum stage is bound by its 1600 SFU operations per track (800 x (ex2 + lg2)), not by HBM (DESIGN.md
        # section 4.2): 148 SMs x 16 SFU lanes x 1.965 GHz = 4.65 Tops/s
        "roofline_fc_hist_alu": {"bound": "alu", "achieved": ev.n_tracks * 1600 / (stage[1] * 1e-3) / 1e12,
                                 "peak": 148 * 16 * 1.965e9 / 1e12, "unit": "T SFU-op/s",
                                 "frac": ev.n_tracks * 1600 / (stage[1] * 1e-3) / (148 * 16 * 1.965e9),
                                 "peak_source": "148 SMs x 16 SFU lanes/clk x 1.965 GHz max SM clock (guide unit counts)"},
        "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": n_e2e, "api": "pvf_run_host (pinned host buffers)"},
        "gpu_launches": launches, "clocks": clocks,
    }
    if world == 1 and not args.no_cpu_baseline:
        v, dt, thr = run_oracle_sample(ev, w, args.cpu_sample)
        out["cpu_baseline"] = {"value": v, "unit": "events/s", "cores": thr, "kind": "oracle",
                               "sample": f"first {args.cpu_sample} events of the batch, {dt:.1f} s"}
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
    ap.add_argument("--weights", default="peaky", choices=["peaky", "rand"])
    ap.add_argument("--channels", type=int, default=64, choices=[64, 32, 16])
    ap.add_argument("--cpu-sample", type=int, default=192)   # ~13 s of oracle time on 16 host threads
    ap.add_argument("--ref-sample", type=int, default=16)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--boundary-margin", type=float, default=0.0,
                    help="NEXT-1 mode (mm): boundary tracks contribute to two intervals, PAPER.md:49")
    ap.add_argument("--cta-pair", type=int, default=1, choices=[0, 1],
                    help="UNet as clusters of two CTAs sharing every MMA (cta_group::2)")
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
