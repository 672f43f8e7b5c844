#!/usr/bin/env python
"""bench.py -- templates/s of the whole per-template hot path on BASELINE.json's metric workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--log2n 23]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

Workload (config.workload): BASELINE.json configs[4] (the throughput sweep the metric is quoted
on) at N = 2^23 samples, tsamp = 64 us: a seeded N(0,1) series and 256 circular + 256 elliptical
(e~U[0,0.1]) random templates (paper_2112_11991_b200/workloads.py::config5).  One "step" = one
pass of the whole hot path over that bank: tb_search_templates on 512
templates + tb_get_candidates.  value = templates/s with the series resident in HBM; e2e = the
same with the series in pinned HOST memory, copied in (tb_plan_set_series) every step, candidates
copied back every step, timed by wall clock around the C-ABI calls.

Multi-GPU (N>1): templates are independent (Alg. 1), so every rank searches its own
512-template shard of a 512*N bank on its own copy of the series; no data-path collective; weak
scaling; time = max over ranks.

--impl reference times the CPU oracle (oracle/tb_oracle.py) on this box's host cores on a bounded
sample of the same workload -- a deliberately plain program, reported as a baseline, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "orbital templates/sec at 2^23 samples (circ & ellip)"
UNIT = "templates/s"
FOLDS = (0, 1, 2, 3, 4)
SIGMA = 6.0


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------- oracle legs
def _oracle_one(args):
    series, tsamp, tmpl, tid = args
    from oracle import tb_oracle as orc
    t0 = time.perf_counter()
    c = orc.search_template(series, tsamp, tmpl, tid, FOLDS, SIGMA)
    return len(c), time.perf_counter() - t0


def oracle_rate(wl, n_templates, cores, pool):
    """Templates/s of the oracle on `cores` processes over n_templates (half circ, half ellip)."""
    k = len(wl.templates) // 2
    ids = [(i // 2) if i % 2 == 0 else k + i // 2 for i in range(n_templates)]
    jobs = [(wl.series, wl.tsamp, wl.templates[i], i) for i in ids]
    t0 = time.perf_counter()
    pool.map(_oracle_one, jobs, chunksize=1)
    return n_templates / (time.perf_counter() - t0)


def host_cores():
    """Every core this process may run on (one oracle process per core)."""
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def source_digest():
    """sha256 (first 16 hex digits) over the CUDA sources: ties profiles/traffic.json to a build."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2112_11991_b200", "csrc")
    for name in sorted(os.listdir(d)):
        with open(os.path.join(d, name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def run_reference(args, wl):
    import multiprocessing as mp
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = host_cores()
    per_step = cores                               # one template per core per step
    with mp.get_context("fork").Pool(cores) as pool:
        for _ in range(args.warmup):
            oracle_rate(wl, per_step, cores, pool)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            oracle_rate(wl, per_step, cores, pool)
        dt = time.perf_counter() - t0
    value = per_step * args.steps / dt
    sample = f"{per_step} templates/step ({per_step - per_step // 2} circular + {per_step // 2} elliptical) of the 512"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(wl, None),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "cpu_model": cpu_model(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def workload_config(wl, chunk):
    return {"workload": f"BASELINE configs[4] throughput sweep at N=2^{int(np.log2(wl.n_samples))}: "
                        f"N(0,1) series, tsamp=64us, {len(wl.templates) // 2} circular + "
                        f"{len(wl.templates) // 2} elliptical (e~U[0,0.1]) templates per GPU",
            "n_samples": wl.n_samples, "tsamp_s": wl.tsamp, "templates_per_gpu": len(wl.templates),
            "folds": list(FOLDS), "sigma_threshold": SIGMA, "median_window": 1024,
            "chunk_templates": chunk,
            "l2": "per-step working set (chunk scratch, >5 GB) exceeds the 126 MB L2; the 32 MB series is "
                  "shared by all templates and L2-resident by design"}


# ---------------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        os.unlink(self.f.name)
        busy = [s for s in sm if s > 0.5 * max(sm)] if sm else []
        return {"sm_mhz": statistics.median(busy) if busy else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------- our arm
def run_ours(args, wl):
    import torch
    import torch.distributed as dist
    from paper_2112_11991_b200 import build
    build.build()
    from paper_2112_11991_b200 import tb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    from paper_2112_11991_b200 import dist as tbd

    def max_over_ranks(v):
        return tbd.max_over_ranks(v, "cuda")

    N, K = wl.n_samples, len(wl.templates)
    first_id = rank * K                                   # this rank's shard of the K*world bank
    stream = torch.cuda.Stream()
    pinned = torch.from_numpy(wl.series).pin_memory()
    host_series = pinned.numpy()
    # the headline plan records no stage events: nothing but the search itself is inside the timed region
    plan = tb.Plan(host_series, wl.tsamp, device=local, stream=stream.cuda_stream, enable_timings=False,
                   chunk_templates=args.chunk, fft_path=args.fft_path, whiten=args.whiten)
    chunk = plan.info()["chunk_templates"]
    stage_keys = ["ms_delay", "ms_resample", "ms_fft", "ms_spectrum", "ms_hsum", "ms_total"]

    def step():
        plan.search(wl.templates, first_id, FOLDS, SIGMA)
        return plan.candidates()

    # ---- device-resident timing (value) ----
    for _ in range(max(args.warmup, 3)):
        step()
    sampler = ClockSampler(local)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_cands = 0
    ev0.record(stream)
    for _ in range(args.steps):
        cands, n = step()
        n_cands = n
    ev1.record(stream)
    barrier()
    ms = max_over_ranks(ev0.elapsed_time(ev1))
    clocks = sampler.stop()
    value = world * K * args.steps / (ms * 1e-3)
    tm = plan.timings()                                   # after the timed region: launch count and path of one step
    launches = tm["n_kernel_launches"] * args.steps
    path_used = tm["fft_path_used"]

    # ---- end to end: series from pinned host memory every step, wall clock ----
    def e2e_step():
        plan.set_series(host_series)
        plan.search(wl.templates, first_id, FOLDS, SIGMA)
        return plan.candidates()

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        c, n = e2e_step()
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    e2e = {"value": world * K * args.steps / e2e_s, "unit": UNIT,
           "h2d_bytes_per_step": 4 * N + 80 * K, "d2h_bytes_per_step": 8 + 24 * int(n)}

    plan.close()

    # ---- per-stage breakdown: a second plan with the stage events on, same steps, outside the headline ----
    plan = tb.Plan(host_series, wl.tsamp, device=local, stream=stream.cuda_stream, enable_timings=True,
                   chunk_templates=args.chunk, fft_path=args.fft_path, whiten=args.whiten)
    stages = {k: 0.0 for k in stage_keys}
    step()
    for _ in range(args.steps):
        step()
        tm = plan.timings()
        for k in stage_keys:
            stages[k] += tm[k]

    # ---- circular / elliptical split (outside the timed region) ----
    detail = {}
    for name, sl in (("circular", slice(0, K // 2)), ("elliptical", slice(K // 2, K))):
        t = []
        for _ in range(3):
            plan.search(wl.templates[sl], 0, FOLDS, SIGMA)
            plan.candidates()
            t.append(plan.timings()["ms_total"])
        detail[f"{name}_templates_per_s"] = (K // 2) / (min(t) * 1e-3)
    plan.close()

    # ---- roofline ----
    peak, peak_src = measured_peaks()
    per_t = {k: stages[k] / (K * args.steps) * 1e-3 for k in stage_keys}          # seconds per template
    # algorithmic bytes each kernel must move per template
    if path_used == 2:
        model = {"ms_delay": 0, "ms_resample": 4 * N + 4 * N // chunk, "ms_fft": 8 * N, "ms_spectrum": 6 * N, "ms_hsum": 2 * N}
        log2n = int(np.log2(N))
        p1 = "P1 k_fft_cols32" if 18 <= log2n <= 24 or log2n == 26 else "P1 k_fft_cols"
        p2 = "P2 k_fft_rows_t" if log2n <= 23 else "P2 k_fft_rows_wide" if log2n <= 25 else "P2 k_fft_cols<DIRECT> + k_fft_rows_scatter"
        names = {"ms_delay": "K0 k_delay_segments (a2 knots)", "ms_resample": p1 + " (a2+a3, a4 pass 1)",
                 "ms_fft": p2 + " (a4 pass 2)", "ms_spectrum": "k_spectrum_t (a4 unpack, a5+a6+a7)",
                 "ms_hsum": "k_hsum_tile (a8+a9)"}
    else:
        model = {"ms_delay": 0, "ms_resample": 4 * N + 4 * N // chunk, "ms_fft": 8 * N, "ms_spectrum": 6 * N, "ms_hsum": 2 * N}
        names = {"ms_delay": "(unused)", "ms_resample": "k_resample (a2+a3)", "ms_fft": "cuFFT R2C batched (a4)",
                 "ms_spectrum": "k_spectrum_median (a5+a6+a7)", "ms_hsum": "k_hsum_tile (a8+a9)"}
    stage_report = {}
    for k in stage_keys[:-1]:
        gbs = model[k] / per_t[k] / 1e9 if per_t[k] > 0 else 0.0
        stage_report[names[k]] = {"us_per_template": per_t[k] * 1e6, "model_bytes": model[k],
                                  "achieved_gbs": gbs, "frac": gbs / peak,
                                  "share_of_step": per_t[k] / per_t["ms_total"] if per_t["ms_total"] else 0.0}
        if k == "ms_delay" and path_used == 2:
            # K0 of chunk i+1 runs on a side stream under P2 / the spectrum former of chunk i: its time is the span it
            # was resident for (it trickles in beside them), not additive; alone it takes 1.6 us per template.  It is
            # therefore left out of the shares (the other four sum to about 1)
            stage_report[names[k]]["overlapped"] = True
            stage_report[names[k]]["share_of_step"] = None
    dom = max(stage_keys[1:-1], key=lambda k: per_t[k])
    dom_gbs = model[dom] / per_t[dom] / 1e9 * 1.0
    # DRAM bytes per launch of the dominant kernel from the last ncu --set full capture
    # (profiles/traffic.json).  A profiler cannot run inside the timed program, so the figure is
    # only reported when the capture was taken on THIS build of the CUDA sources; otherwise null.
    traffic, traffic_note = None, "no capture for this build"
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as f:
            tj = json.load(f)
        if N != 1 << 23 or chunk != 64:
            traffic_note = "the capture is of the N = 2^23, 64-template launch only"
        elif tj.get("_csrc_sha256_16") == source_digest():
            traffic = tj.get(names[dom].split(" (")[0])
            traffic_note = tj.get("_source", "")
        else:
            traffic_note = f"profiles/traffic.json was captured on another build ({tj.get('_csrc_sha256_16')})"
    roofline = {"bound": "hbm", "kernel": names[dom], "achieved": dom_gbs, "peak": peak, "unit": "GB/s",
                "frac": dom_gbs / peak, "traffic": traffic, "traffic_source": traffic_note, "peak_source": peak_src,
                "launches_timed": int(args.steps * -(-K // chunk)),
                # one clock: the same CUDA-event time the headline `value` comes from (per GPU)
                "pipeline": {"model_bytes_per_template": 22 * N,
                             "achieved": 22 * N * (value / world) / 1e9,
                             "frac": 22 * N * (value / world) / 1e9 / peak,
                             "frac_of_8TBs_nominal": 22 * N * (value / world) / 1e9 / 8000.0},
                "stage_timer_ms_per_step": stages["ms_total"] / args.steps,
                "stages": stage_report}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f32 (delay model f64)", "data": "synthetic",
           "config": dict(workload_config(wl, chunk), whiten=bool(args.whiten)), "samples_per_s": value * N, "candidates_per_step": int(n_cands),
           "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "detail": detail, "roofline": roofline}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import multiprocessing as mp
        cores = host_cores()
        with mp.get_context("fork").Pool(cores) as pool:
            v = oracle_rate(wl, cores, cores, pool)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "cpu_model": cpu_model(), "kind": "oracle",
                               "sample": f"{cores} templates ({cores - cores // 2} circular + {cores // 2} elliptical) "
                                         f"of the 512, one per core, full N=2^{int(np.log2(N))}"}
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--log2n", type=int, default=23)
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--fft-path", type=int, default=0, help="tb_plan_opts.fft_path (0 auto, 1 cuFFT, 2 hand-written or error)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--whiten", action="store_true",
                    help="SURVEY 8(f) f2 mode: whiten the series once per plan (every set_series), one constant normalisation per "
                         "template instead of block medians; NOT the default path the metric is quoted on")
    args = ap.parse_args()

    from paper_2112_11991_b200 import workloads
    wl = workloads.config5(log2n=args.log2n)
    if args.impl == "reference":
        run_reference(args, wl)
    else:
        run_ours(args, wl)


if __name__ == "__main__":
    main()
