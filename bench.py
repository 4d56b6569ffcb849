#!/usr/bin/env python
"""bench.py -- headline measurement of the OS-TV hot path (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload 3|2|1]

A "step" is one pass of the whole hot path over one batch of synthetic input: one complete
reconstruction of the workload (config 3 by default: 512x512, 800 x 738, 20 ordered subsets, 500
subset iterations, beta = 0.005) = 500 x (K1 forward+residual+monitor+step rule, K2 back+TV+update).
`value` = subset iterations per second over the whole job, inputs resident in HBM; `e2e` = the same
through osiv_reconstruct_host (host buffers, H2D + D2H inside the timed region).  With N > 1 (torchrun)
every rank reconstructs its own slice (weak scaling, no data-path collective); time = max over ranks.

`--impl reference` times the float64 CPU oracle (oracle/) as it stands on the host cores, one bounded
sample of the same workload per step; only that leg and `cpu_baseline` execute anything under oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth_inputs as si  # noqa: E402

METRIC = "os_tv_iterations_per_s"
UNIT = "iterations/s"
FP32_FLOP_PER_NNZ = 6          # q (FMA, 2) + half-width minus |q| (1) + clamp (1) + accumulate (FMA, 2)
NNZ_PER_RAY_PER_N = 1.193      # measured non-zeros per ray / N when the fan spans the inscribed circle
SM_COUNT, FP32_LANES_PER_SM = 148, 128
# per-launch instruction / wavefront / sector / DRAM-byte counts of the two hot kernels at config 3: read from the
# committed ncu capture of this code (profiles/<NCU_COUNTS>.csv, written by `python -m paper_1903_10088_b200.ncu_summary`
# from ncu's raw page; the .md beside it names the ncu command).  Counts do not depend on timing; the times they are
# divided by are measured live in this run.
NCU_COUNTS = {"3": "r2_ncu_config3_counts.csv", "5a": "r2_ncu_config5a_counts.csv", "5b": "r2_ncu_config5b_counts.csv"}


def load_ncu_counts(workload):
    """{'k_forward': {...}, 'k_back': {...}} from the committed capture, or {} when there is none for this workload"""
    import csv
    name = NCU_COUNTS.get(workload)
    path = os.path.join(ROOT, "profiles", name) if name else None
    if not path or not os.path.exists(path):
        return {}, None
    out = {}
    for row in csv.DictReader(open(path)):
        key = "k_forward" if row["kernel"].startswith("k_forward") else "k_back" if row["kernel"].startswith("k_back") else None
        if key and key not in out:
            out[key] = {k: float(v) for k, v in row.items() if k != "kernel"}
            out[key]["name"] = row["kernel"]
    return out, "profiles/" + name


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d, "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def workload_desc(cfg, beta, batch):
    return {"workload": f"config{cfg.name}: {cfg.nx}x{cfg.ny} image, {cfg.n_views}x{cfg.n_channels} fan sinogram, "
                        f"{cfg.n_subsets} ordered subsets, {cfg.n_iters} subset iterations, beta={beta}, "
                        f"Poisson(I0={cfg.i0:g}) counts of a seeded {cfg.n_ellipses}-ellipse phantom",
            "slices_per_gpu": batch, "image": [cfg.ny, cfg.nx], "views": cfg.n_views, "channels": cfg.n_channels,
            "subsets": cfg.n_subsets, "iterations_per_step": cfg.n_iters, "beta": beta,
            "l2": "flushed between steps (256 MiB memset, outside the per-step events)",
            "parallelism": f"{batch} slice(s) per GPU, no collective"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    # started BEFORE the warm-up steps (the start-up of nvidia-smi itself stalls the driver for a few hundred milliseconds:
    # inside the timed region it showed up as 27.8 ms of wall clock per 8.85 ms step); only the samples whose timestamp
    # falls between mark_begin() and mark_end() -- the timed region -- are used, the warm-up ones if there are none
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.path = None
        self.t0 = self.t1 = None

    def mark_begin(self):
        import datetime
        self.t0 = datetime.datetime.now()

    def mark_end(self):
        import datetime
        self.t1 = datetime.datetime.now()

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        import datetime
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = []
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    ts = datetime.datetime.strptime(f[0], "%Y/%m/%d %H:%M:%S.%f")
                    rows.append((ts, float(f[1]), float(f[2]), [n for n, v in zip(names, f[5:9]) if v.lower().startswith("active")]))
                except ValueError:
                    continue
            os.unlink(self.path)
        except Exception:
            pass
        inside = [r for r in rows if self.t0 and self.t1 and self.t0 <= r[0] <= self.t1]
        used = inside if inside else rows
        if used:
            out.update(sm_mhz=float(np.median([r[1] for r in used])), sm_max_mhz=float(max(r[2] for r in used)), samples=len(used),
                       window="timed region" if inside else "warm-up and timed region (no sample fell inside the timed region)")
        out["reasons"] = sorted({n for r in used for n in r[3]})
        return out


def oracle_sample(cfg, beta, counts, n_iters):
    """Time the oracle, as it stands, on the first n_iters subset iterations of the workload."""
    import oracle
    og = oracle.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.dgamma_rad,
                         cfg.channel_offset, cfg.theta0_rad)
    prm = oracle.Params(beta=beta, n_subsets=cfg.n_subsets, n_iters=n_iters)
    t0 = time.perf_counter()
    img, trace, status = oracle.reconstruct(og, counts, cfg.i0, prm)
    dt = time.perf_counter() - t0
    return dt, oracle.num_threads(), img


def run_reference(args, cfg, beta):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    _, _, counts = si.make_case(cfg)
    n_sample = min(cfg.n_iters, cfg.n_subsets)            # one pass over all subsets per step
    for _ in range(args.warmup):
        oracle_sample(cfg, beta, counts, n_sample)
    t = 0.0
    cores = 1
    for _ in range(args.steps):
        dt, cores, _ = oracle_sample(cfg, beta, counts, n_sample)
        t += dt
    value = n_sample * args.steps / t
    sample = f"first {n_sample} of {cfg.n_iters} subset iterations of the workload per step (float64 oracle, OpenMP)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_desc(cfg, beta, 1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args, cfg, beta):
    import torch
    import torch.distributed as dist
    import paper_1903_10088_b200 as osiv
    from paper_1903_10088_b200 import sharding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    osiv.lib()

    geom = osiv.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.sdd_mm,
                         cfg.dgamma_rad, cfg.channel_offset, cfg.theta0_rad)
    batch = args.slices if args.slices > 0 else (64 if args.workload == "4" else 1)
    lo, hi = sharding.slice_range(rank, world, world * batch)     # weak scaling: `batch` slices per rank
    counts_np = np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(lo, hi)])
    prm = osiv.Params(beta=beta, n_subsets=cfg.n_subsets, n_iters=cfg.n_iters)
    h = osiv.Handle(geom, max_batch=batch, device=local)
    counts = torch.from_numpy(counts_np).to(dev)
    out = torch.empty((batch, cfg.ny, cfg.nx), dtype=torch.float32, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    pin_counts = torch.from_numpy(counts_np).pin_memory()
    pin_out = torch.empty((batch, cfg.ny, cfg.nx), dtype=torch.float32).pin_memory()

    def step():
        h.reconstruct(counts, cfg.i0, prm, out=out)

    def step_e2e():
        h.reconstruct_host(pin_counts, cfg.i0, prm, out=pin_out)

    sampler = ClockSampler(local)
    sampler.start()
    step_e2e()
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    # ---- timed region: K steps, device events per step, L2 flushed in between ----
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sharding.barrier()
    torch.cuda.synchronize()
    n0 = h.launch_count()
    sampler.mark_begin()
    wall0 = time.perf_counter()
    for a, b in ev:
        flush.zero_()
        a.record()
        step()
        b.record()
    torch.cuda.synchronize()
    sharding.barrier()
    wall = time.perf_counter() - wall0
    sampler.mark_end()
    launches = h.launch_count() - n0
    t_dev = sum(a.elapsed_time(b) for a, b in ev) * 1e-3
    t_dev = sharding.max_over_ranks(t_dev, dev)
    clocks = sampler.stop()

    # ---- end-to-end: host buffers through osiv_reconstruct_host (one more untimed call first: the second call with these
    # arguments is the one that captures the graph) ----
    step_e2e()
    sharding.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step_e2e()
    torch.cuda.synchronize()
    t_e2e = sharding.max_over_ranks(time.perf_counter() - t0, dev)

    # ---- per-kernel durations for the roofline (2 extra profiled steps; events around every launch) ----
    h.set_profiling(True)
    for _ in range(2):
        flush.zero_()
        step()
    ms_f, n_f, ms_b, n_b = h.get_profile()
    h.set_profiling(False)

    total_iters = world * batch * cfg.n_iters * args.steps
    value = total_iters / t_dev
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks, peak_kind = load_peaks()
    sm_mhz_peak = float(peaks.get("sm_max_mhz", 1965.0))
    alu_peak_derived = SM_COUNT * FP32_LANES_PER_SM * 2 * sm_mhz_peak * 1e6 / 1e12
    # the binding units' peaks, measured in this process (csrc/osiv_probes.cu; MEASURED_PEAKS.json has HBM and bf16 only)
    probe = osiv.probe_peaks(local)
    alu_peak_tflops = float(probe["ffma_tflops"])
    ncu, ncu_file = load_ncu_counts(cfg.name if batch == 1 else "")
    vs = cfg.n_views // cfg.n_subsets
    nnz = NNZ_PER_RAY_PER_N * max(cfg.nx, cfg.ny) * vs * cfg.n_channels * batch       # per launch, fwd = back
    kernels = {}
    for name, ms, n in (("k_forward<1>", ms_f, n_f), ("k_back<1>", ms_b, n_b)):
        us = 1e3 * ms / max(n, 1)
        tf = nnz * FP32_FLOP_PER_NNZ / (us * 1e-6) / 1e12
        kernels[name] = {"avg_us": us, "achieved_tflops": tf, "frac": tf / alu_peak_tflops, "launches": n}
    # Inside the timed region the two kernels are chained by dependent launches and no event can sit between them, so a
    # kernel's average duration THERE is the region's time per iteration times the kernel's share of the profiled
    # (stand-alone) per-launch times -- the share ncu's launch list shows too (profiles/r2_launches_config3.md).
    us_iter = 1e6 * t_dev / args.steps / cfg.n_iters
    for name in kernels:
        share = kernels[name]["avg_us"] / sum(k["avg_us"] for k in kernels.values())
        us_in = us_iter * share
        tf_in = nnz * FP32_FLOP_PER_NNZ / (us_in * 1e-6) / 1e12
        kernels[name]["in_region"] = {"share": share, "avg_us": us_in, "achieved_tflops": tf_in, "frac": tf_in / alu_peak_tflops}
    dom = max(kernels, key=lambda k: kernels[k]["avg_us"])
    # issue / L1 / L2 / DRAM fractions: counts per launch from the committed ncu capture of this code over the live time
    for name in kernels:
        c = ncu.get("k_forward" if name.startswith("k_forward") else "k_back")
        if not c:
            continue
        t = kernels[name]["avg_us"] * 1e-6
        l1_bytes = c["l1_wavefronts_per_sm"] * 128.0 * SM_COUNT
        kernels[name].update({
            "ncu_kernel": c["name"],
            "issue": {"warp_instructions": c["warp_instructions"], "achieved_ginst_s": c["warp_instructions"] / t / 1e9,
                      "peak_ginst_s": probe["issue_ginst_per_s"], "frac": c["warp_instructions"] / t / 1e9 / probe["issue_ginst_per_s"]},
            "l1": {"wavefronts_per_sm": c["l1_wavefronts_per_sm"], "achieved_gbs": l1_bytes / t / 1e9,
                   "peak_gbs": probe["l1_read_gbs"], "frac": l1_bytes / t / 1e9 / probe["l1_read_gbs"],
                   "note": "data-pipe wavefronts x 128 B (global and shared memory share the pipe)"},
            "l2": {"sectors": c["l2_sectors"], "achieved_gbs": c["l2_sectors"] * 32.0 / t / 1e9,
                   "peak_gbs": probe["l2_read_gbs"], "frac": c["l2_sectors"] * 32.0 / t / 1e9 / probe["l2_read_gbs"]},
            "dram_bytes": c["dram_bytes"]})
        ti = kernels[name]["in_region"]["avg_us"] * 1e-6
        kernels[name]["in_region"].update({"issue_frac": c["warp_instructions"] / ti / 1e9 / probe["issue_ginst_per_s"],
                                           "l1_frac": l1_bytes / ti / 1e9 / probe["l1_read_gbs"],
                                           "l2_frac": c["l2_sectors"] * 32.0 / ti / 1e9 / probe["l2_read_gbs"]})
    # compulsory HBM bytes per launch: everything is L2-resident, so this is a floor
    hbm_bytes = {"k_forward<1>": (cfg.nx * cfg.ny * 4 + 2 * vs * cfg.n_channels * 4 + vs * cfg.n_channels * 32) * batch,
                 # + K2's candidate-interval table: one int per (view of the subset, 2x2 tile of the base quadrant)
                 "k_back<1>": (cfg.nx * cfg.ny * 4 * 3 + vs * cfg.n_channels * 16) * batch + vs * (cfg.nx // 4) * (cfg.ny // 4) * 4}
    chain_t = t_dev / args.steps / (2 * cfg.n_iters)
    roof = {"bound": "alu", "kernel": dom, "achieved": kernels[dom]["in_region"]["achieved_tflops"], "peak": alu_peak_tflops,
            "unit": "TFLOP/s", "frac": kernels[dom]["in_region"]["frac"],
            "achieved_note": "algorithmic flops per launch / the kernel's average duration inside the timed region = region time per "
                             "iteration x the kernel's share of the per-launch times (kernels[*].in_region); `standalone` is the same "
                             "kernel timed alone between two events (cold start, no overlap with its neighbours), the figure "
                             "earlier bench lines of this repository carried as `frac`",
            "standalone": {"avg_us": kernels[dom]["avg_us"], "achieved": kernels[dom]["achieved_tflops"], "frac": kernels[dom]["frac"]},
            "traffic": kernels[dom].get("dram_bytes"),
            "traffic_source": (ncu_file + ": dram__bytes_read.sum + dram__bytes_write.sum per launch, cold caches") if ncu_file else None,
            "peak_source": f"FP32 FFMA probe run in this process (csrc/osiv_probes.cu); derived 148 SMs x 128 lanes x 2 flop x "
                           f"{sm_mhz_peak:.0f} MHz = {alu_peak_derived:.1f} TFLOP/s",
            "probe_peaks": probe,
            "issue": kernels[dom].get("issue"), "l1": kernels[dom].get("l1"), "l2": kernels[dom].get("l2"),
            "counts_source": ncu_file,
            "algorithmic_flop_per_launch": nnz * FP32_FLOP_PER_NNZ, "nnz_per_launch": nnz,
            "timing": "kernels[*].avg_us: CUDA events around every launch on the launching stream, 2 extra steps after the timed "
                      "region; an event between two launches serialises them, so these are stand-alone kernel durations "
                      "(in the timed region K1 and K2 overlap their prologues through programmatic dependent launch); "
                      "kernels[*].in_region: the timed region's events, apportioned by those durations' shares",
            "kernels": kernels,
            # in the timed region K1 and K2 are chained by dependent launches: the step's time over its hot launches
            "chain": {"us_per_launch": 1e6 * chain_t,
                      "achieved_tflops": nnz * FP32_FLOP_PER_NNZ / chain_t / 1e12,
                      "frac": nnz * FP32_FLOP_PER_NNZ / chain_t / 1e12 / alu_peak_tflops,
                      "issue_frac": (sum(c["warp_instructions"] for c in ncu.values()) / 2.0 / chain_t / 1e9 / probe["issue_ginst_per_s"]) if len(ncu) == 2 else None,
                      # the memory level that binds: L1 / shared-memory data-pipe wavefronts x 128 B of both kernels over the timed region
                      "l1_gbs": (sum(c["l1_wavefronts_per_sm"] for c in ncu.values()) / 2.0 * 128.0 * SM_COUNT / chain_t / 1e9) if len(ncu) == 2 else None,
                      "l1_frac": (sum(c["l1_wavefronts_per_sm"] for c in ncu.values()) / 2.0 * 128.0 * SM_COUNT / chain_t / 1e9 / probe["l1_read_gbs"]) if len(ncu) == 2 else None},
            "hbm": {"compulsory_bytes_per_launch": hbm_bytes[dom],
                    "achieved_gbs": hbm_bytes[dom] / (kernels[dom]["avg_us"] * 1e-6) / 1e9,
                    "peak_gbs": float(peaks["hbm_gbs"]), "peak_kind": peak_kind,
                    "frac": hbm_bytes[dom] / (kernels[dom]["avg_us"] * 1e-6) / 1e9 / float(peaks["hbm_gbs"])}}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * t_dev / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_desc(cfg, beta, batch),
            "seconds_per_500_iter_recon": (t_dev / args.steps) * 500.0 / cfg.n_iters,
            "slices_per_s": world * batch * args.steps / t_dev,
            "wall_ms_per_step_incl_flush": 1e3 * wall / args.steps,
            "wall_note": "host clock around the timed region: includes the L2 flushes and whatever the nvidia-smi clock sampler "
                         "(one query per 100 ms) stalls; a loop without sampler and flush runs at the device time (DESIGN.md section 6)",
            "paper_context": {"gtx1080ti_s_per_slice_thinning_1_20": 3.71, "iterations_per_s": 134.8,
                              "source": "PAPER.md:156,164 Table I (other hardware, real data; context only)"},
            "clocks": clocks,
            "e2e": {"value": world * batch * cfg.n_iters * args.steps / t_e2e, "unit": UNIT,
                    "h2d_bytes_per_step": int(pin_counts.numel() * 4), "d2h_bytes_per_step": int(pin_out.numel() * 4),
                    "ms_per_step": 1e3 * t_e2e / args.steps},
            "gpu_launches": int(launches),
            "roofline": roof}

    # the other workloads of BASELINE.json inside the same JSON line (one line per run; these are not the headline)
    if world == 1 and args.workload == "3" and batch == 1 and not args.no_extra:
        del h, counts, out, flush
        torch.cuda.empty_cache()
        extra = {}
        extra["config4"] = batch_throughput(osiv, si.scan_config("4"), 0.005, 64, 2, 1, dev)
        for name in ("5a", "5b"):
            pa = argparse.Namespace(steps=5, warmup=3)
            extra["config" + name] = projector_pair(pa, si.scan_config(name))
        # the paper's Table I: seconds per 512 x 512 slice against the thinning parameter 1/M
        paper_gpu = {1: 11.00, 2: 7.76, 5: 5.37, 10: 4.30, 20: 3.71, 40: 3.39}
        t1 = {}
        for M in (1, 2, 5, 10, 20, 40):
            r = batch_throughput(osiv, si.scan_config("3", n_subsets=M), 0.005, 1, 2, 1, dev)
            t1[f"1/{M}"] = {"seconds_per_slice": r["ms_per_step"] * 1e-3, "iterations_per_s": r["iterations_per_s"],
                            "views_per_iteration": cfg.n_views // M, "plan": r["plan"], "paper_gtx1080ti_seconds": paper_gpu[M]}
        extra["table1"] = {"workload": "config 3's slice at the paper's six thinning parameters, 500 subset iterations each "
                                       "(the paper does not print its iteration count per column; context only, other hardware, real data)",
                           "source": "PAPER.md:158-164 Table I", "thinning": t1}
        for b2 in (0.001, 0.02):                    # config 3's beta sweep: same launches, other data
            extra[f"config3_beta{b2}"] = batch_throughput(osiv, cfg, b2, 1, 3, 1, dev)
        line["extra"] = extra
    if not args.no_cpu_baseline:
        n_sample = min(cfg.n_iters, 10 * cfg.n_subsets)
        dt, cores, _ = oracle_sample(cfg, beta, counts_np[0], n_sample)
        line["cpu_baseline"] = {"value": n_sample / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"first {n_sample} of {cfg.n_iters} subset iterations of slice 0 "
                                          f"({dt:.1f} s, float64 oracle with OpenMP)"}
        if args.cpu_plan != "none":
            line["cpu_baseline"]["plan"] = cpu_plan(args, args.cpu_plan == "full")
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def projector_pair(args, cfg):
    """Config 5 (BASELINE.json): forward A and adjoint A^T alone, all views, on a uniform-random image / sinogram.
    Not the headline metric: one extra JSON line with ms per pass, nnz/s ("rays.pixels/s" = ray-pixel intersections),
    algorithmic GB/s against the measured HBM peak and the adjoint-identity error of the fp32 outputs."""
    import torch
    import paper_1903_10088_b200 as osiv
    torch.cuda.set_device(0)
    geom = osiv.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.sdd_mm)
    img_np, sino_np = si.uniform_image(cfg), si.uniform_sinogram(cfg)
    img, sino = torch.from_numpy(img_np)[None].cuda(), torch.from_numpy(sino_np)[None].cuda()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    h = osiv.Handle(geom, max_batch=1, device=0)
    out = {}
    for name, fn in (("forward", lambda: h.forward(img)), ("back", lambda: h.backward(sino))):
        for _ in range(max(args.warmup, 3)):
            res = fn()
        ts = []
        for _ in range(args.steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); res = fn(); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        out[name] = (float(np.median(ts)), res.cpu().numpy()[0].astype(np.float64))
    nnz = NNZ_PER_RAY_PER_N * max(cfg.nx, cfg.ny) * cfg.n_views * cfg.n_channels
    bytes_alg = 4.0 * (cfg.nx * cfg.ny + cfg.n_views * cfg.n_channels)          # image + sinogram, once each
    peaks, kind = load_peaks()
    lhs = float(np.dot(out["forward"][1].ravel(), sino_np.astype(np.float64).ravel()))
    rhs = float(np.dot(img_np.astype(np.float64).ravel(), out["back"][1].ravel()))
    line = {"metric": "projector_pair", "workload": f"config{cfg.name}: {cfg.nx}x{cfg.ny}, {cfg.n_views}x{cfg.n_channels}, all views",
            "n_gpus": 1, "steps": args.steps, "dtype": "f32", "data": "synthetic", "nnz_per_pass": nnz,
            "adjoint_rel_error": abs(lhs - rhs) / abs(lhs), "l2": "flushed between passes"}
    ncu, ncu_file = load_ncu_counts(cfg.name)
    probe = osiv.probe_peaks(0)
    for name in ("forward", "back"):
        ms = out[name][0]
        line[name] = {"ms_per_pass": ms, "nnz_per_s": nnz / (ms * 1e-3), "algorithmic_gbs": bytes_alg / (ms * 1e-3) / 1e9,
                      "hbm_frac": bytes_alg / (ms * 1e-3) / 1e9 / float(peaks["hbm_gbs"]), "hbm_peak_kind": kind,
                      "alu_frac": nnz * FP32_FLOP_PER_NNZ / (ms * 1e-3) / 1e12 / probe["ffma_tflops"]}
        # the pass is two launches (layout kernel + projector); the projector's counts per launch from the committed capture
        c = ncu.get("k_forward" if name == "forward" else "k_back")
        if c:
            t = ms * 1e-3
            line[name].update({"issue_frac": c["warp_instructions"] / t / 1e9 / probe["issue_ginst_per_s"],
                               "l1_gbs": c["l1_wavefronts_per_sm"] * 128.0 * SM_COUNT / t / 1e9,
                               "l1_frac": c["l1_wavefronts_per_sm"] * 128.0 * SM_COUNT / t / 1e9 / probe["l1_read_gbs"],
                               "l2_gbs": c["l2_sectors"] * 32.0 / t / 1e9, "l2_frac": c["l2_sectors"] * 32.0 / t / 1e9 / probe["l2_read_gbs"],
                               "dram_gbs_cold": c["dram_bytes"] / t / 1e9, "counts_source": ncu_file})
    return line


def run_projector_pair(args, cfg):
    print(json.dumps(projector_pair(args, cfg)))
    return 0


def batch_throughput(osiv, cfg, beta, batch, steps, warmup, dev):
    """slices/s of `batch` slices per launch (config 4): CUDA events around whole reconstructions, L2 flushed in between"""
    import torch
    geom = osiv.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.sdd_mm,
                         cfg.dgamma_rad, cfg.channel_offset, cfg.theta0_rad)
    counts = torch.from_numpy(np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(batch)])).to(dev)
    prm = osiv.Params(beta=beta, n_subsets=cfg.n_subsets, n_iters=cfg.n_iters)
    out = torch.empty((batch, cfg.ny, cfg.nx), dtype=torch.float32, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
    with osiv.Handle(geom, max_batch=batch, device=dev.index or 0) as h:
        for _ in range(warmup):
            h.reconstruct(counts, cfg.i0, prm, out=out)
        ts = []
        for _ in range(steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); h.reconstruct(counts, cfg.i0, prm, out=out); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        plan = h.plan(cfg.n_subsets, batch)
    ms = float(np.mean(ts))
    vs = cfg.n_views // cfg.n_subsets
    nnz = NNZ_PER_RAY_PER_N * max(cfg.nx, cfg.ny) * vs * cfg.n_channels * batch
    us_launch = 1e3 * ms / (2 * cfg.n_iters)
    return {"workload": f"config{cfg.name}: {batch} slices of {cfg.nx}x{cfg.ny}, {cfg.n_views}x{cfg.n_channels}, {cfg.n_subsets} subsets, "
                        f"{cfg.n_iters} iterations, beta={beta}", "steps": steps, "warmup": warmup, "ms_per_step": ms,
            "slices_per_s": batch / (ms * 1e-3), "iterations_per_s": batch * cfg.n_iters / (ms * 1e-3),
            "us_per_slice_iteration": 1e3 * ms / (batch * cfg.n_iters), "plan": plan,
            "achieved_tflops": nnz * FP32_FLOP_PER_NNZ / (us_launch * 1e-6) / 1e12}


def cpu_plan(args, full):
    """the float64 oracle, as it stands, on the host cores (never inside a timed GPU region):
    configs 1 and 2 in full, one projector pass of 5a; with --cpu-plan full also config 3's 500 iterations, 5b and two slices
    of config 4 (scaled to 64 and labelled so)."""
    import oracle
    out = {"cores": oracle.num_threads(), "kind": "oracle"}
    for name in ("1", "2") + (("3",) if full else ()):
        c = si.scan_config(name)
        _, _, cnt = si.make_case(c)
        beta = 0.005 if name == "3" else c.betas[0]
        dt, _, _ = oracle_sample(c, beta, cnt, c.n_iters)
        out["config" + name] = {"seconds": dt, "iterations": c.n_iters, "iterations_per_s": c.n_iters / dt, "sample": "full reconstruction"}
    if full:
        c = si.scan_config("4")
        dts = [oracle_sample(c, 0.005, si.make_case(c, slice_index=s)[2], c.n_iters)[0] for s in range(2)]
        out["config4"] = {"seconds_64_slices_scaled": 32.0 * sum(dts), "seconds_2_slices": sum(dts),
                          "slices_per_s": 2.0 / sum(dts), "sample": "2 slices x 500 iterations, scaled x32 (labelled as scaled)"}
    for name in ("5a",) + (("5b",) if full else ()):
        c = si.scan_config(name)
        og = oracle.Geometry(c.nx, c.ny, c.pixel_mm, c.n_views, c.n_channels, c.sad_mm)
        img, sino = si.uniform_image(c), si.uniform_sinogram(c)
        t0 = time.perf_counter(); oracle.forward(og, img); t1 = time.perf_counter(); oracle.backward(og, sino); t2 = time.perf_counter()
        nnz = NNZ_PER_RAY_PER_N * max(c.nx, c.ny) * c.n_views * c.n_channels
        out["config" + name] = {"forward_s": t1 - t0, "back_s": t2 - t1, "forward_nnz_per_s": nnz / (t1 - t0), "back_nnz_per_s": nnz / (t2 - t1),
                                "sample": "one forward and one back pass over all views"}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="3", choices=["1", "2", "3", "4", "5a", "5b"])
    ap.add_argument("--slices", type=int, default=0, help="slices per GPU (default 1; 64 for workload 4)")
    ap.add_argument("--beta", type=float, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the config 4 / 5a / 5b / beta-sweep figures inside the line")
    ap.add_argument("--cpu-plan", default="short", choices=["none", "short", "full"],
                    help="BASELINE.md section 3 oracle timings next to cpu_baseline: short = configs 1, 2, 5a; full = + 3, 4, 5b (minutes)")
    ap.add_argument("--probe", action="store_true", help="print the measured FP32 / issue / L2 / shared-memory / L1 peaks and exit")
    args = ap.parse_args()
    if args.probe:
        import paper_1903_10088_b200 as osiv
        print(json.dumps({"probe_peaks": osiv.probe_peaks(0), "how": "csrc/osiv_probes.cu: saturating loops, CUDA events, best of 5"}))
        return 0
    cfg = si.scan_config(args.workload)
    beta = args.beta if args.beta is not None else (0.005 if args.workload == "3" else (cfg.betas[0] if cfg.betas else 0.0))
    if args.workload in ("5a", "5b"):
        return run_projector_pair(args, cfg)
    if args.impl == "reference":
        return run_reference(args, cfg, beta)
    return run_ours(args, cfg, beta)


if __name__ == "__main__":
    sys.exit(main())
