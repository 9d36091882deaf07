#!/usr/bin/env python
"""Benchmark of the measurement operator hot path (BASELINE.json metric: visibilities/s for Phi and
Phi^dagger at M = 1e8 on one B200; % of HBM roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4] [--M m]

A "step" is one pass of the whole hot path, Phi^dagger Phi (S+Z, F, W G, G^dagger W^dagger,
F^dagger, Z^dagger S^dagger) over the config's visibility set; for N > 1 every
rank owns its own M visibilities (the paper's data-parallel scheme) and the step
ends with the all-reduce of the image (Eq. 38).  value = (visibilities all ranks processed) / time.
Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle (the only reference there
is: the paper ships no code) on a bounded sample, on the host cores.
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

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "visibilities/sec for Phi^dagger Phi (one Phi + one Phi^dagger per step)"
UNIT = "visibilities/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--M", type=int, default=0, help="override the number of visibilities (debug)")
    ap.add_argument("--cpu-sample", type=int, default=4_000_000, help="visibilities in the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except Exception:
                self.p.kill()
        try:
            self.f.flush()
            rows = [r.strip().split(",") for r in open(self.f.name) if r.strip()]
            sm, mx, reasons = [], [], set()
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            for r in rows:
                if len(r) < 7:
                    continue
                try:
                    sm.append(float(r[0])); mx.append(float(r[1]))
                except ValueError:
                    continue
                for nme, val in zip(names, r[3:7]):
                    if val.strip().lower() == "active":
                        reasons.add(nme)
            if sm:
                out = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                       "samples": len(sm)}
        except Exception:
            pass
        finally:
            try:
                os.unlink(self.f.name)
            except OSError:
                pass
        return out


# ----------------------------------------------------------------------------------- oracle timing
def time_oracle(cfg, x, uv, w, sample: int):
    """The CPU oracle as it stands on a bounded sample: the K x K stages (pad, FFT, inverse FFT, crop)
    at full size, the O(M J^2) stages (degrid, grid) on the first `sample` visibilities, extrapolated
    linearly in M (operator time is linear in M)."""
    import oracle
    ms = min(sample, len(uv))
    uvs = uv[:ms].astype(np.float64)
    ws = w[:ms].astype(np.float64)
    mode = cfg.kernel_mode
    prec = 32 if cfg.dtype == "c64" else 64
    t0 = time.perf_counter()
    B = oracle.fft2(oracle.pad(x, cfg.J), -1)
    t1 = time.perf_counter()
    y = oracle.degrid_from_grid(B, uvs, ws, cfg.J, mode, cfg.table_R, prec)
    t2 = time.perf_counter()
    Bp = oracle.grid_to_grid(y, uvs, ws, cfg.K, cfg.J, mode, cfg.table_R, prec)
    t3 = time.perf_counter()
    oracle.crop(oracle.fft2(Bp, +1), cfg.J)
    t4 = time.perf_counter()
    fixed = (t1 - t0) + (t4 - t3)
    per_vis = ((t2 - t1) + (t3 - t2)) / ms
    return {"fixed_s": fixed, "degrid_s": t2 - t1, "grid_s": t3 - t2, "per_vis_s": per_vis, "sample": ms,
            "cores": oracle.num_threads()}


def cpu_baseline_entry(cfg, M, res):
    full = res["fixed_s"] + M * res["per_vis_s"]
    return {"value": M / full, "unit": UNIT, "cores": res["cores"], "kind": "oracle",
            "sample": (f"oracle/ (fp64 C++, OpenMP): pad+FFT+iFFT+crop at full {cfg.K}x{cfg.K} "
                       f"({res['fixed_s']:.2f} s) + degrid ({res['degrid_s']:.2f} s) and grid ({res['grid_s']:.2f} s) "
                       f"on the first {res['sample']} of {M} visibilities, extrapolated linearly in M "
                       f"to {full:.1f} s per Phi^dagger Phi")}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from inputs import synth
    cfg = synth.CONFIGS[args.config]
    M = args.M or cfg.M
    ms = min(args.cpu_sample, M)
    x = synth.make_image(cfg.n, cfg.seed, cfg.dtype)
    uv = synth.make_uv(cfg, ms)
    w = synth.make_weights(cfg, ms)
    runs = []
    for i in range(args.warmup + args.steps):
        r = time_oracle(cfg, x, uv, w, ms)
        if i >= args.warmup:
            runs.append(r)
    fixed = statistics.mean(r["fixed_s"] for r in runs)
    per_vis = statistics.mean(r["per_vis_s"] for r in runs)
    full = fixed + M * per_vis
    agg = dict(runs[-1], fixed_s=fixed, per_vis_s=per_vis)
    value = args.gpus * M / full if args.gpus > 1 else M / full
    line = {"impl": "reference", "metric": METRIC, "value": M / full, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": full * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload(cfg, M, args.gpus),
            "cpu_baseline": cpu_baseline_entry(cfg, M, agg),
            "e2e": {"value": M / full, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    del value
    print(json.dumps(line), flush=True)


def alu_roofline(cfg, M, stage_ms):
    """fp32 FMA work of W G / G^dagger W^dagger per visibility (ANALYTIC mode): the J x J complex-times-real MACs
    (2 J^2 + 2 J FMA for degridding, 2 J^2 + 2 J + 2 for gridding) plus the paired even/odd Horner chains of the
    kernel weights, 2 axes x J/2 pairs x (deg + 1) FMA + 6; TABLE mode: the MACs only.  Peak: nominal plain-ALU fp32."""
    if cfg.dtype != "c64":
        return None
    J = cfg.J
    deg = 8 if J == 4 else 7
    wts = 0 if cfg.kernel_mode == "table" else 2 * (J // 2) * (deg + 1) + 6
    fma = {"degrid": 2 * J * J + 2 * J + 2 + wts, "grid": 2 * J * J + 2 * J + 2 + wts}
    peak = 148 * 128 * 2 * 1.965e9 / 1e12
    out = {"bound": "alu", "unit": "TFLOP/s", "peak": peak,
           "peak_source": "nominal: 148 SMs x 128 fp32 lanes x 2 flop x 1.965 GHz (DESIGN.md 5)"}
    for k, f in fma.items():
        if stage_ms.get(k):
            ach = 2.0 * f * M / (stage_ms[k] * 1e-3) / 1e12
            out[k] = {"fma_per_visibility": f, "achieved": ach, "frac": ach / peak}
    return out


def workload(cfg, M, gpus):
    return {"workload": f"BASELINE.json configs[{cfg.index - 1}] ({cfg.name}): {cfg.n}x{cfg.n} image, "
                        f"{cfg.K}x{cfg.K} grid, Kaiser-Bessel J={cfg.J}, M={M} visibilities per GPU, "
                        f"uv={cfg.uv}, {cfg.dtype}, kernel={cfg.kernel_mode}",
            "n": cfg.n, "K": cfg.K, "J": cfg.J, "M_per_gpu": M, "M_total": M * gpus, "uv": cfg.uv,
            "kernel_mode": cfg.kernel_mode, "y_order": "native (tile-sorted) inside Phi^dagger Phi",
            "l2": (f"inputs exceed L2 (no flush needed): every step streams {M * (20 if cfg.dtype == 'c64' else 40) / 1e9:.2f} GB of "
                   f"visibility data + the {cfg.K * cfg.K * (8 if cfg.dtype == 'c64' else 16) / 1e6:.0f} MB grid"
                   if M * 20 > 126e6 else "working set fits L2: times are L2-resident, no roofline claim"),
            "parallelism": f"dp{gpus} over visibilities, all-reduce of the image after Phi^dagger" if gpus > 1 else "single GPU"}


# ----------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist

    from inputs import synth
    from paper_1903_04502_b200 import ANALYTIC, C64, C128, TABLE, PurifyOp
    from paper_1903_04502_b200 import dist as pdist

    rank, local_rank, world = pdist.world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    cfg = synth.CONFIGS[args.config]
    M = args.M or cfg.M
    dt = C64 if cfg.dtype == "c64" else C128
    cbytes = 8 if cfg.dtype == "c64" else 16
    rbytes = cbytes // 2
    # every rank draws its OWN visibility set (weak scaling): seed offset by rank
    rcfg = pdist.rank_config(cfg, rank)
    t_gen = time.perf_counter()
    x = synth.make_image(cfg.n, cfg.seed, cfg.dtype)
    uv = synth.make_uv(rcfg, M)
    w = synth.make_weights(rcfg, M)
    t_gen = time.perf_counter() - t_gen

    x_pin = torch.from_numpy(x).pin_memory()
    out_pin = torch.empty_like(x_pin).pin_memory()
    x_dev = x_pin.cuda()
    out_dev = torch.empty_like(x_dev)
    t_create = time.perf_counter()
    op = PurifyOp(cfg.n, cfg.J, torch.from_numpy(uv).cuda(), torch.from_numpy(w).cuda(), dtype=dt,
                  kernel_mode=TABLE if cfg.kernel_mode == "table" else ANALYTIC,
                  table_samples_per_unit=cfg.table_R if cfg.kernel_mode == "table" else 0, time_stages=True)
    torch.cuda.synchronize()
    t_create = time.perf_counter() - t_create
    info = op.info()
    torch.cuda.empty_cache()

    def step():
        op.normal(x_dev, out_dev)
        pdist.allreduce_image(out_dev)                          # Eq. (38): sum of the per-rank dirty images

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank) if rank == 0 else None
    if sampler:
        time.sleep(0.5)                      # let nvidia-smi start sampling before the GPU gets busy
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    e0.record()
    marks[0].record()
    for i in range(args.steps):
        step()
        marks[i + 1].record()          # per-step marks (no synchronisation): mean / std / min as the paper reports
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    per_step = [marks[i].elapsed_time(marks[i + 1]) for i in range(args.steps)]
    launches = op.last_launch_count() * args.steps
    ms_total = pdist.max_over_ranks(ms_total, device="cuda")
    ms_step = ms_total / args.steps

    # ---- per-stage breakdown (separate pass; each step followed by a sync to read the stage events)
    stages = {}
    for _ in range(args.steps):
        op.normal(x_dev, out_dev)
        for k, v in op.stage_times_ms().items():
            stages.setdefault(k, []).append(v)
    stage_ms = {k: statistics.mean(v) for k, v in stages.items()}
    clocks = sampler.stop() if sampler else None

    # ---- Phi alone and Phi^dagger alone (native order), and caller order
    def timed(fn, reps):
        fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    y_dev = op.degrid(x_dev, native=True)
    reps = max(3, args.steps // 2)
    ms_phi = timed(lambda: op.degrid(x_dev, y_dev, native=True), reps)
    ms_phit = timed(lambda: op.grid(y_dev, out_dev, native=True), reps)
    y_call = op.permute_from_native(y_dev)
    ms_phi_caller = timed(lambda: op.degrid(x_dev, y_call, native=False), reps)
    ms_phit_caller = timed(lambda: op.grid(y_call, out_dev, native=False), reps)
    del y_call

    # ---- f2: power method on Phi^dagger Phi, 10 iterations from the all-ones vector
    op.norm(None, max_iter=1, rel_tol=0.0)               # warm-up: workspace allocation happens here
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    lam, its = op.norm(None, max_iter=10, rel_tol=0.0)
    torch.cuda.synchronize()
    norm_info = {"lambda_after_10_iterations": lam, "ms_per_iteration": (time.perf_counter() - t0) * 1e3 / max(its, 1),
                 "note": "purify_op_norm: Phi^dagger Phi + fp64 norm + scaling per iteration (wall clock of the call / iterations)"}

    # ---- f1: Algorithm 1 lines 3-6 around the operator (fused for complex64 + analytic weights), native-order vectors
    y_obs = op.degrid(x_dev, native=True)
    y_obs.mul_(1.01)
    s_dual = torch.zeros_like(y_obs)
    ms_admm = timed(lambda: op.admm_fidelity_step(x_dev, y_obs, s_dual, 1.0, 0.9, out_dev, want_norm=False), reps)
    admm_info = {"ms": ms_admm, "ms_minus_phi_dagger_phi": ms_admm - ms_step,
                 "note": "purify_admm_fidelity_step: v = Phi x, l2-ball projection, dual update, Phi^dagger (v - r + s)"}
    del y_obs, s_dual

    # ---- end to end through the C ABI with HOST buffers (H2D of x, D2H of the result inside)
    op.normal_host(x_pin, out_pin)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        op.normal_host(x_pin, out_pin)
        if world > 1:
            pass    # the host-buffer path is single-GPU; the image all-reduce is in the device arm
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / args.steps
    e2e_s = pdist.max_over_ranks(e2e_s, device="cuda")

    if rank == 0:
        peak, peak_src = measured_peak()
        K = cfg.K
        per_vis = 2 * rbytes + rbytes + cbytes                       # uv + w + y  (20 B / 40 B)
        alg_bytes = M * per_vis + K * K * cbytes                      # + the grid, once
        dom = "degrid" if stage_ms.get("degrid", 0) >= stage_ms.get("grid", 0) else "grid"
        dom_ms = stage_ms[dom]
        achieved = alg_bytes / (dom_ms * 1e-3) / 1e9
        traffic = None
        try:    # measured DRAM traffic of the dominant kernel (ncu capture under profiles/), same workload only
            tr = json.load(open(os.path.join(ROOT, "profiles", "r1f_traffic.json.txt")))
            traffic = tr.get(f"config{cfg.index}_M{M}", {}).get(dom)
        except Exception:
            traffic = None
        kname = f"{dom}_x_kernel" if info["layout"] == 1 else f"{dom}_kernel"
        line = {
            "metric": METRIC, "value": world * M / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
            "ms_per_step_stats": {"mean": statistics.mean(per_step), "std": statistics.pstdev(per_step), "min": min(per_step),
                                  "max": max(per_step), "note": "rank 0, per-step CUDA events inside the timed region"},
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if cfg.dtype == "c64" else "f64", "data": "synthetic",
            "config": workload(cfg, M, world),
            "e2e": {"value": world * M / e2e_s, "unit": UNIT, "ms_per_step": e2e_s * 1e3,
                    "h2d_bytes_per_step": int(x_pin.numel() * cbytes), "d2h_bytes_per_step": int(out_pin.numel() * cbytes),
                    "api": "purify_normal_host (pinned host x in, host x out)"},
            "gpu_launches": launches,
            "roofline": {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "peak_source": peak_src, "traffic": traffic,
                         "note": "HBM fraction of the ALGORITHMIC bytes; the kernel itself is fp32-FMA bound (profiles/r1f_summary.md)",
                         "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": dom_ms,
                         "frac_of_8TBs": achieved / 8000.0,
                         "other_kernel": {k: {"ms": stage_ms[k], "achieved": alg_bytes / (stage_ms[k] * 1e-3) / 1e9,
                                              "frac": alg_bytes / (stage_ms[k] * 1e-3) / 1e9 / peak}
                                          for k in ("degrid", "grid") if k != dom}},
            # the same kernels against the plain-ALU fp32 ceiling (they are FMA-bound, not HBM-bound):
            # algorithmic flops = M x (4 J^2 + 4 J complex-times-real MAC flops + weight evaluation), peak = 148 SMs x
            # 128 fp32 lanes x 2 flop x 1.965 GHz
            "roofline_alu": alu_roofline(cfg, M, stage_ms),
            "stage_ms": stage_ms,
            "operators": {"phi_ms": ms_phi, "phi_vis_per_s": M / (ms_phi * 1e-3),
                          "phi_dagger_ms": ms_phit, "phi_dagger_vis_per_s": M / (ms_phit * 1e-3),
                          "phi_caller_order_ms": ms_phi_caller, "phi_dagger_caller_order_ms": ms_phit_caller},
            "operator_norm": norm_info,
            "admm_fidelity_step": admm_info,
            "clocks": clocks,
            "setup": {"generate_s": t_gen, "create_s": t_create, "n_items": info["n_items"],
                      "n_tiles_nonempty": info["n_tiles_nonempty"], "max_tile_count": info["max_tile_count"],
                      "device_bytes": info["device_bytes"], "M_native": info["M_native"],
                      "padding_ratio": info["M_native"] / max(M, 1), "n_batches": info["n_batches"]},
        }
        if world == 1 and not args.no_cpu_baseline:
            ms = min(args.cpu_sample, M)
            res = time_oracle(cfg, x, uv[:ms], w[:ms], ms)
            line["cpu_baseline"] = cpu_baseline_entry(cfg, M, res)
        print(json.dumps(line), flush=True)
    op.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
