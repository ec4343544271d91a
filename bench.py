#!/usr/bin/env python
"""bench.py -- posterior evaluations/s of the BioEM hot path on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config paper] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic images: bioem_push_images (a0) +
bioem_run (a1-a7) for the named config.  The default is the LARGEST single-GPU configuration of BASELINE.json,
"paper" (configs[2]: 224^2 px -- the paper's own box size, P:229 -- 1024 images, 4096 orientations x 32 CTFs x 61^2
shifts = 4.99e11 evaluations per step, about 5 s); BASELINE.json quotes its metric on no particular config, and the
other four are parity-test cases (`--config` still runs them).  `value` is timed with the images already resident in
HBM; `e2e` is the same step through the C ABI with HOST buffers (H2D of the image stack and D2H of the results inside
the timed region).  One process per GPU (torchrun for N > 1): the path shards over images with no data-path
collective (paper: P:199): the global stack of N x 1024 images goes through shard.score_block_and_gather
(every rank scores its contiguous block, one all_gather of the per-image results inside the timed region) ->
"scaling": "weak".  `--impl reference` times the FP64 CPU oracle (the only reference there is) on a bounded sample
of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import bioem_workloads as W  # noqa: E402

METRIC = "posterior evaluations/s (image x orientation x CTF x shift)"
UNIT = "evaluations/s"
SM_COUNT, FP32_LANES = 148, 128
KERNEL_NAMES = {1: "k_fused", 2: "k_fused_pk", 3: "k_fused_c2", 4: "k_fused_tm", 5: "k_fused_dft", 6: "k_realspace"}


def ncu_table(workload):
    """Per-launch DRAM traffic and executed flops of the fused kernel from the committed ncu captures: the row of
    profiles/fused_kernel_ncu.csv for this workload (the .md beside it names the capture commands), or None."""
    f = ROOT / "profiles" / "fused_kernel_ncu.csv"
    if not f.exists():
        return None
    rows = [r.split(",") for r in f.read_text().splitlines() if r and not r.startswith("#")]
    hdr = rows[0]
    for r in rows[1:]:
        d = dict(zip(hdr, r))
        if d.get("workload") == workload:
            return d
    return None


def algorithmic_flops_per_pair(N: int, D: int) -> float:
    """SURVEY 8(d) / DESIGN 7: conj-multiply 6H + pruned inverse transform ((N/2+1) column FFTs of 5 N log2 N,
    (2D+1) c2r row FFTs of 2.5 N log2 N) + 30 flops per shift for the closed form."""
    H = N * (N // 2 + 1)
    S = (2 * D + 1) ** 2
    lg = math.log2(N)
    return 6 * H + (N // 2 + 1) * 5 * N * lg + (2 * D + 1) * 2.5 * N * lg + 30 * S


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        return json.loads(p.read_text()), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                       "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [r.split(",") for r in Path(self.f.name).read_text().splitlines() if r.count(",") >= 6]
        os.unlink(self.f.name)
        clk, reasons, mx = [], set(), None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                clk.append(float(r[0])); mx = float(r[1])
            except ValueError:
                continue
            for nm, v in zip(names, r[3:7]):
                if v.strip().lower() == "active":
                    reasons.add(nm)
        if clk:
            out.update(sm_mhz=float(np.median(clk)), sm_max_mhz=mx, reasons=sorted(reasons), samples=len(clk))
        return out


def build_inputs(config, rank, orient_stride=1):
    spec = W.get_spec(config)
    if orient_stride > 1:
        from dataclasses import replace
        spec = replace(spec, name=f"{spec.name}/orient_stride{orient_stride}", orient_stride=spec.orient_stride * orient_stride)
    if rank:
        from dataclasses import replace
        spec = replace(spec, index=spec.index + 100 * rank)      # other ranks: same config, different image seeds
    return W.build_workload(spec)


def oracle_sample_rate(wl, n_img, n_orient, n_ctf):
    """The oracle as it stands on a bounded sample (first images / orientations / CTFs of the workload)."""
    import oracle
    s = wl["spec"]
    oracle.build()
    oracle.lib()
    t0 = time.perf_counter()
    for m in wl["models"][:1]:
        oracle.run_model(m, s.n_pix, s.pixel_A, s.max_shift, wl["quats"][:n_orient], wl["ctfs"][:n_ctf], wl["images"][:n_img])
    dt = time.perf_counter() - t0
    pairs = n_img * n_orient * n_ctf
    return pairs * s.n_shifts / dt, dt, oracle.num_threads(), f"{n_img} images x {n_orient} orientations x {n_ctf} CTFs x {s.n_shifts} shifts of '{s.name}' (direct summation, model 0)"


def oracle_sample_shape(wl, target_s):
    """Size the bounded sample for about `target_s` seconds of oracle time: all CTFs, up to 16 images (the oracle's OpenMP
    loop runs over images), and as many orientations as a one-orientation probe says fit."""
    s = wl["spec"]
    ni, nc = min(s.n_images, 16), s.n_ctf
    oracle_sample_rate(wl, ni, 1, nc)                             # build / load / page in / thread start-up, untimed
    _, dt, _, _ = oracle_sample_rate(wl, ni, 1, nc)
    no = int(max(1, min(s.n_orient, target_s / max(dt, 1e-6))))
    return ni, no, nc


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = build_inputs(args.config, 0)
    s = wl["spec"]
    ni, no, nc = oracle_sample_shape(wl, 6.0)                    # ~6 s of oracle time per step
    for _ in range(args.warmup):
        oracle_sample_rate(wl, 1, 1, 1)
    t_tot, ev = 0.0, 0.0
    for _ in range(args.steps):
        rate, dt, cores, sample = oracle_sample_rate(wl, ni, no, nc)
        t_tot += dt
        ev += rate * dt
    value = ev / t_tot
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": s.name, "n_pix": s.n_pix, "note": "FP64 CPU oracle, bounded sample per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1609_06634_b200 import BioEM, shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    local = local % torch.cuda.device_count()                                 # --backend gloo may put several ranks on one GPU (functional check only)
    torch.cuda.set_device(local)
    if world > 1:
        if args.backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # rank r holds block r of the global stack of world x n_images images (same config, its own image seeds)
    wl = build_inputs(args.config, rank, args.orient_stride)
    s = wl["spec"]
    n_global = s.n_images * world
    img_host = torch.from_numpy(wl["images"]).pin_memory()
    img_dev = img_host.cuda()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")          # > 126 MB L2
    b = BioEM(device=local)
    b.load_workload(wl, images=False)

    def step_device():
        flush.zero_()                                                          # L2 flush between iterations
        b.invalidate_precompute()                                              # a1-a3 run in every step (nothing cached across steps)
        if world > 1:                                                          # block -> results -> one all_gather (shard.py)
            return shard.score_block_and_gather(b, img_dev, n_global)
        b.push_images(img_dev)
        b.run()

    def step_e2e():
        flush.zero_()
        b.invalidate_precompute()
        if world > 1:
            return shard.score_block_and_gather(b, img_host, n_global)
        b.push_images(img_host)                                                # H2D inside the step
        b.run()
        return dict(logp=b.get_log_posterior(), **b.get_best())                # D2H inside the step

    for _ in range(max(args.warmup, 1)):
        step_device()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    fused_ms, launches = [], 0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step_device()
        launches += b.get_launch_count()[0]                                    # kernels of push_images + run
        fused_ms.append(b.get_timing()[1])                                     # CUDA events around the fused kernel, on the context's stream
    e1.record()
    barrier()
    clocks = sampler.stop() if sampler else None
    fused_ms = float(np.mean(fused_ms))                                        # average launch duration over the timed region
    total_ms_last = b.get_timing()[0]
    kern, oc = b.get_run_plan()
    t_dev = e0.elapsed_time(e1) * 1e-3

    # ---- end to end through the C ABI with host buffers
    res = step_e2e()
    barrier()
    t0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        res = step_e2e()
    e1.record()
    barrier()
    t_e2e = max(e0.elapsed_time(e1) * 1e-3, time.perf_counter() - t0)
    h2d = int(img_host.numel() * 4)
    d2h = int(sum(np.asarray(v).nbytes for v in res.values())) // world       # this rank's share of the results

    if world > 1:
        t = torch.tensor([t_dev, t_e2e], device="cuda" if args.backend == "nccl" else "cpu", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_dev, t_e2e = float(t[0]), float(t[1])
    evals_job = float(s.n_evaluations) * world * args.steps
    if rank == 0:
        peaks, peak_src = measured_peaks()
        fp32_peak = SM_COUNT * FP32_LANES * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12          # TFLOP/s, DESIGN 7
        fma_meas, _ = b.measure_fp32_peak()
        fpp = algorithmic_flops_per_pair(s.n_pix, s.max_shift)
        fl = fpp * s.n_pairs
        achieved = fl / (fused_ms * 1e-3) / 1e12
        hbm_bytes = s.n_pairs * 8.0 * s.n_pix * (s.n_pix // 2 + 1)               # streaming Ohat once per pair
        ncu = ncu_table(s.name) or {}
        ex = float(ncu["executed_flops_per_pair"]) if ncu.get("executed_flops_per_pair") else None
        roof = {
            "bound": "alu", "kernel": KERNEL_NAMES.get(kern, str(kern)) + " (a4+a5+a6)", "orientations_per_work_item": oc,
            "achieved": achieved, "peak": fp32_peak, "unit": "TFLOP/s",
            "frac": achieved / fp32_peak, "traffic": float(ncu["dram_bytes_per_launch"]) if ncu.get("dram_bytes_per_launch") else None,
            "traffic_source": ncu.get("capture"),
            "peak_source": f"148 SM x 128 lanes x 2 x {peaks.get('sm_max_mhz', 1965.0):.0f} MHz (formula, {peak_src})",
            "measured_ffma_tflops": fma_meas, "frac_of_measured_ffma": achieved / fma_meas,
            "kernel_ms": fused_ms, "step_ms_on_device": total_ms_last, "flops_per_pair": fpp,
            "executed_flops_per_pair": ex, "executed_tflops": (ex * s.n_pairs / (fused_ms * 1e-3) / 1e12) if ex else None,
            "hbm_alt": {"bytes_per_launch_if_streamed": hbm_bytes, "gbs_equivalent": hbm_bytes / (fused_ms * 1e-3) / 1e9,
                        "peak_gbs": peaks.get("hbm_gbs")},
        }
        ni, no, nc = oracle_sample_shape(wl, 24.0)               # lands at 10-30 s of oracle time (the one-orientation probe overestimates)
        rate, dt, cores, sample = oracle_sample_rate(wl, ni, no, nc)
        line = {
            "metric": METRIC, "value": evals_job / t_dev, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_dev / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": s.name, "n_pix": s.n_pix, "n_images_per_gpu": s.n_images, "n_models": s.n_models,
                       "n_orient": s.n_orient, "n_ctf": s.n_ctf, "max_shift": s.max_shift, "evaluations_per_step_per_gpu": s.n_evaluations,
                       "cache": "L2 flushed between iterations (256 MiB write); projection spectra are regenerated every step",
                       "precision": "hot loop FP32, precompute and top-8 re-scoring FP64",
                       "parallelism": f"images sharded, dp{world}" + (", results all_gathered every step" if world > 1 else "")},
            "e2e": {"value": evals_job / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": launches, "clocks": clocks, "roofline": roof,
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": dt},
        }
        print(json.dumps(line), flush=True)
    b.close()
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """Shapes of the paper's Fig. 4 (time against the number of images; linear above 128-256) and Fig. 2 (time against the
    number of displacements for the Fourier-space and the real-space variant; the Fourier route is almost flat and wins beyond a
    handful of displacements) on the `small` grid with every 16th orientation.
    One JSON line per point: device time of bioem_run (CUDA events inside the library), median of 3."""
    import torch
    from paper_1609_06634_b200 import BioEM
    wl = build_inputs("small", 0, 16)
    s = wl["spec"]
    pts = ([("images", n, s.max_shift, 0) for n in (1, 2, 4, 8, 16, 32, 64, 128, 256)] if args.sweep == "images"
           else [("shifts", s.n_images, d, 0) for d in (0, 1, 2, 4, 8, 12, 16)] + [("shifts", s.n_images, d, 1) for d in (0, 1, 2, 3, 4)])
    with BioEM(device=0) as b:
        b.load_workload(wl, images=False)
        for kind, n_img, D, variant in pts:
            b.set_shift_range(D)
            b.set_displacement_variant(variant)
            b.push_images(wl["images"][:n_img])
            ms = []
            for _ in range(4):
                b.invalidate_precompute()
                b.run()
                b.get_log_posterior()
                ms.append(b.get_timing())
            tot, fused = np.median([m[0] for m in ms[1:]]), np.median([m[1] for m in ms[1:]])
            pairs = n_img * s.n_orient * s.n_ctf
            print(json.dumps({"sweep": kind, "variant": "real space, cropping" if variant else "Fourier space, circular", "n_images": n_img,
                              "max_shift": D, "n_shifts": (2 * D + 1) ** 2, "pairs": pairs, "run_ms": float(tot), "scoring_ms": float(fused),
                              "ns_per_pair": 1e6 * float(tot) / pairs}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="paper", choices=sorted(W.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="torch.distributed backend for N > 1 (gloo: functional check of the multi-rank path, e.g. two ranks on one GPU)")
    ap.add_argument("--orient-stride", type=int, default=1,
                    help="profiling aid: keep every k-th orientation of the grid (the workload name in the JSON line says so)")
    ap.add_argument("--sweep", choices=["images", "shifts"], help="Fig. 4 / Fig. 2 shaped sweeps on one GPU (one JSON line per point)")
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
