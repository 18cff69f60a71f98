#!/usr/bin/env python
"""bench.py — one JSON line for the doubly-periodic Stokes mobility product on B200.

A "step" is ONE mobility product (U, Omega) = M (F, tau): all hot-path stages (bin, spread, xy FFT, per-wavenumber
solve, inverse FFT, interpolate) over one batch of synthetic particles.  Default workload = BASELINE.json configs[4]
("cfg5": bottom wall, 1,048,576-particle microroller monolayer, 4320 x 4320 x 32 grid, forces + torques), the
configuration the metric is quoted on; it fits one GPU (57 GB of grids).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl reference] [--no-cpu-baseline]

N > 1 (under torchrun): N independent replicas, one per GPU, no data-path collective ("replicas only");
value = total particles of all ranks / max-over-ranks device time.
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

import workloads

METRIC = "ms per DP-wall mobility product M·F at N=1M; particles/s; % of HBM roofline"
# kernels of this library launched per product: k_bin_count, k_scan, k_bin_scatter, k_weights, k_spread, k_solve<nz>, k_zero_mode,
# k_interp, plus k_fft_x_fwd, k_fft_y_fwd, k_fft_y_inv, k_fft_x_inv with the library's own FFT passes (else cuFFT's kernels)
MY_KERNELS_PER_STEP = {"own": 12, "cufft": 8}
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, one launch, from the committed ncu --set full capture
# (profiles/r1_d_README.md: 18.83 GB read with 11 of 32 input planes skipped + 29.00 GB written); None where no capture exists
NCU_TRAFFIC_GB = {("k_solve<32>", 5): 47.83}


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def stage_bytes(prob, n, fin, fout, zero_planes=0):
    """Algorithmic (compulsory) bytes per product and stage: every grid value read once and
    written once per stage.  Planes above every footprint hold no force (exactly zero): with ``zero_planes`` of the nz input
    planes skipped, the input side of spread / forward FFT / solve shrinks by that share — the bytes really needed."""
    G = prob.nx * prob.ny * prob.nz
    Kz = (prob.nx // 2 + 1) * prob.ny * prob.nz
    R, C = 8.0 * G, 16.0 * Kz
    a = 1.0 - zero_planes / float(prob.nz)
    return {"spread": a * fin * R + 72.0 * n, "fft_fwd": a * fin * (R + C), "solve": (a * fin + fout) * C,
            "fft_inv": fout * (C + R), "interp": fout * R + 72.0 * n}


def replica_seed(base_seed: int, rank: int) -> int:
    """N > 1 = N independent replicas (the product does not shard): each rank draws its own particles from
    the same recipe; rank 0 keeps the configuration's own seed."""
    return base_seed + 17 * rank


def max_over_ranks(dist, value: float, device) -> float:
    """Device time of the slowest rank (the contract's timing rule); no other collective exists on this path."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(n_per_rank: int, world: int, ms_step: float) -> float:
    """particles/s of all replicas together."""
    return world * n_per_rank / (ms_step * 1e-3)


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        super().__init__(daemon=True)
        self.gpu = gpu_index
        self.stop_flag = threading.Event()
        self.rows = []

    def run(self):
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.splitlines()[0].split(",")])
            except Exception:
                pass
            self.stop_flag.wait(0.1)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows)}


def cpu_sample_problem(cfg: int):
    """Bounded sample of the same workload recipe for the oracle legs: same kernel, heights, drives and area fraction,
    fewer particles (the product is linear-time), sized for ~10-30 s of host work."""
    if cfg in (3, 5):
        return workloads.monolayer_bw(n=32768, seed=1005, name="cfg5-sample-32k")
    if cfg == 4:
        return workloads.monolayer_slit(n=32768, seed=1004, name="cfg4-sample-32k")
    return workloads.config(cfg)


def time_oracle(cfg: int, reps: int = 1):
    import oracle
    prob, pos, F, T = cpu_sample_problem(cfg)
    best = None
    for _ in range(reps):
        t0 = time.perf_counter()
        oracle.mobility_apply(prob, pos, F, T, dft="fft")
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return prob, len(pos), best, oracle.num_threads()


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores; each step = one product of the bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    prob, pos, F, T = cpu_sample_problem(args.config)
    for _ in range(args.warmup):
        oracle.mobility_apply(prob, pos, F, T, dft="fft")
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.mobility_apply(prob, pos, F, T, dft="fft")
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    val = len(pos) / dt
    full = workloads_describe(args.config)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "particles/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": dict(full, note="oracle timed on a bounded sample of this workload"),
            "cpu_baseline": {"value": val, "unit": "particles/s", "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": "%s: N=%d, grid %dx%dx%d, same recipe; xy DFT via numpy.fft (library primitive)" % (
                                 prob.name, len(pos), prob.nx, prob.ny, prob.nz)},
            "e2e": {"value": val, "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def workloads_describe(cfg: int):
    names = {1: "cfg1 bottom wall N=128", 2: "cfg2 slit N=4096", 3: "cfg3 bottom-wall monolayer N=65536",
             4: "cfg4 slit monolayer N=262144", 5: "cfg5 bottom-wall microroller monolayer N=1048576"}
    return {"workload": names[cfg]}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--transfer-fp32", action="store_true", help="time the fp32 spread/interpolate variant as the main number")
    ap.add_argument("--no-fp32-variant", action="store_true", help="skip the extra timing of the fp32 spread/interpolate variant")
    ap.add_argument("--dense-planes", action="store_true", help="transform every plane (do not skip the planes no footprint reaches)")
    ap.add_argument("--fft", choices=["own", "cufft"], default="own", help="xy FFT backend (own shared-memory passes, or cuFFT for comparison)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl != "reference" else args.warmup

    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import paper_2210_01837_b200 as dp
    dp.load_library()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist = dist_mod
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)

    prob, pos, F, T = workloads.config(args.config)
    if world > 1:      # replicas: each rank draws its own particles from the same recipe
        prob, pos, F, T = (workloads.monolayer_bw(n=prob.n, seed=replica_seed(prob.seed, rank), name=prob.name) if args.config in (3, 5)
                           else workloads.config(args.config))
    n = len(pos)
    fin = 6 if T is not None else 3
    fout = fin
    plan = dp.Plan(prob, max_particles=n, use_torques=T is not None, device=local_rank, fft_backend=0 if args.fft == "own" else 1,
                   transfer_fp32=args.transfer_fp32, dense_planes=args.dense_planes)
    fft_backend = plan.fft_backend()
    dpos = torch.from_numpy(pos).to(dev)
    dF = torch.from_numpy(F).to(dev)
    dT = torch.from_numpy(T).to(dev) if T is not None else None
    U = torch.empty((n, 3), dtype=torch.float64, device=dev)
    Om = torch.empty((n, 3), dtype=torch.float64, device=dev) if T is not None else None
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident timing: inputs already in HBM
    plan.set_profiling(True)
    for _ in range(args.warmup):
        plan.mobility_apply(dpos, dF, dT, out_U=U, out_Omega=Om, stream=stream)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_acc = {}
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        plan.mobility_apply(dpos, dF, dT, out_U=U, out_Omega=Om, stream=stream)
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    sampler.stop_flag.set()
    sampler.join(timeout=3)
    # per-stage device times: a second, separately synchronised pass (dp_stage_ms synchronises, so it stays out of the timed loop)
    for _ in range(max(3, min(args.steps, 5))):
        plan.mobility_apply(dpos, dF, dT, out_U=U, out_Omega=Om, stream=stream)
        for k, v in plan.stage_ms().items():
            stage_acc.setdefault(k, []).append(v)
    stage_ms = {k: float(np.median(v)) for k, v in stage_acc.items()}
    assert plan.check() == 0
    zero_planes = plan.zero_planes()
    ms_step = max_over_ranks(dist, ms_total / args.steps, dev)
    value = whole_job_value(n, world, ms_step)

    # ---- end to end: host buffers in (pinned), host buffers out, through dp_mobility_apply_host
    e2e = None
    if not args.no_e2e:
        hp = torch.from_numpy(pos).pin_memory(); hF = torch.from_numpy(F).pin_memory()
        hT = torch.from_numpy(T).pin_memory() if T is not None else None
        hU = torch.empty((n, 3), dtype=torch.float64).pin_memory()
        hO = torch.empty((n, 3), dtype=torch.float64).pin_memory() if T is not None else None
        npv = lambda t: None if t is None else t.numpy()
        for _ in range(2):
            plan.mobility_apply_host(npv(hp), npv(hF), npv(hT), out_U=npv(hU), out_Omega=npv(hO))
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            plan.mobility_apply_host(npv(hp), npv(hF), npv(hT), out_U=npv(hU), out_Omega=npv(hO))   # synchronous
        dt = max_over_ranks(dist, (time.perf_counter() - t0) / args.steps, dev)
        e2e = {"value": world * n / dt, "unit": "particles/s", "ms_per_step": dt * 1e3,
               "h2d_bytes_per_step": int(24 * n * (3 if T is not None else 2)), "d2h_bytes_per_step": int(24 * n * (2 if T is not None else 1))}

    # ---- two more timings of the same product on the same inputs, same rules (3 warm-ups, CUDA events, max over ranks):
    #      the optional fp32 spread/interpolate variant (north_star: "also timed"), and the product with the zero-plane
    #      skipping switched off (every plane spread, transformed and loaded)
    plan_bytes = plan.device_bytes()

    def time_variant(**kw):
        nonlocal plan
        plan.close()
        plan = dp.Plan(prob, max_particles=n, use_torques=T is not None, device=local_rank, **kw)
        plan.set_profiling(True)
        for _ in range(args.warmup):
            plan.mobility_apply(dpos, dF, dT, out_U=U, out_Omega=Om, stream=stream)
        barrier()
        v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        v0.record(stream)
        for _ in range(args.steps):
            plan.mobility_apply(dpos, dF, dT, out_U=U, out_Omega=Om, stream=stream)
        v1.record(stream)
        barrier()
        vms = max_over_ranks(dist, v0.elapsed_time(v1) / args.steps, dev)
        plan.mobility_apply(dpos, dF, dT, out_U=U, out_Omega=Om, stream=stream)
        vst = plan.stage_ms()
        return {"ms_per_step": vms, "value": world * n / (vms * 1e-3), "unit": "particles/s",
                "stage_ms": {k: vst[k] for k in ("spread", "fft_fwd", "solve", "fft_inv", "interp")},
                "plan_device_GB": plan.device_bytes() / 1e9}

    variant = dense = None
    if not args.transfer_fp32 and not args.no_fp32_variant and args.fft == "own":
        variant = time_variant(transfer_fp32=True, dense_planes=args.dense_planes)
        variant["what"] = ("spreading and interpolation accumulate in fp32, real-space grids stored in fp32; FFTs and solves fp64; "
                           "matches the oracle to <= 1e-5 (tests)")
        if not args.dense_planes and zero_planes > 0:
            dense = time_variant(transfer_fp32=False, dense_planes=True)
            dense["what"] = "same fp64 product with dense_planes = 1: the %d planes no footprint reaches are spread, transformed and loaded too" % zero_planes

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src = hbm_peak()
    by = stage_bytes(prob, n, fin, fout, zero_planes)
    by_dense = stage_bytes(prob, n, fin, fout, 0)
    stages = {}
    for k, b in by.items():
        t_ms = stage_ms.get(k, 0.0)
        gbs = b / (t_ms * 1e-3) / 1e9 if t_ms > 0 else None
        stages[k] = {"ms": t_ms, "algorithmic_GB": b / 1e9, "GBps": gbs, "frac": (gbs / peak) if gbs else None}
    stages["bin"] = {"ms": stage_ms.get("bin", 0.0)}
    mine = {k: stages[k] for k in ("spread", "solve", "interp")}
    dom = max(mine, key=lambda k: mine[k]["ms"])
    kernel_name = {"spread": "k_spread", "solve": "k_solve<%d>" % prob.nz, "interp": "k_interp"}[dom]
    mid = sum(by[k] for k in ("fft_fwd", "solve", "fft_inv")) / 1e9
    mid_ms = sum(stage_ms.get(k, 0.0) for k in ("fft_fwd", "solve", "fft_inv"))
    traffic = NCU_TRAFFIC_GB.get((kernel_name, args.config))
    roofline = {"bound": "hbm", "kernel": kernel_name, "achieved": mine[dom]["GBps"], "peak": peak, "unit": "GB/s",
                "frac": mine[dom]["frac"], "traffic": traffic * 1e9 if traffic else None, "peak_source": peak_src,
                "note": "k_solve is co-bound by the fp64 pipe and shared memory (profiles/r1_d_README.md); the fraction is of the HBM roofline",
                "fft_chebyshev_solve_stages": {"algorithmic_GB": mid, "ms": mid_ms, "GBps": mid / (mid_ms * 1e-3) if mid_ms else None,
                                               "frac": (mid / (mid_ms * 1e-3) / peak) if mid_ms else None},
                "whole_product": {"algorithmic_GB": sum(by.values()) / 1e9, "ms": ms_step,
                                  "frac": sum(by.values()) / 1e9 / (ms_step * 1e-3) / peak,
                                  "algorithmic_GB_if_all_planes_dense": sum(by_dense.values()) / 1e9}}

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        sprob, sn, sdt, cores = time_oracle(args.config)
        cpu = {"value": sn / sdt, "unit": "particles/s", "cores": cores, "kind": "oracle", "seconds": sdt,
               "sample": "%s: N=%d, grid %dx%dx%d, same recipe; xy DFT via numpy.fft (library primitive)" % (sprob.name, sn, sprob.nx, sprob.ny, sprob.nz)}

    line = {"metric": METRIC, "value": value, "unit": "particles/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workloads_describe(args.config), n_particles=n, grid=[prob.nx, prob.ny, prob.nz], wall_mode=["bottom_wall", "slit"][prob.wall_mode],
                           fields_in=fin, fields_out=fout, w=prob.w, l2="inputs (%.1f GB of grids per product) far exceed the 126 MB L2" % (sum(by.values()) / 1e9 / 4),
                           parallelism="replicas" if world > 1 else "single GPU", plan_device_GB=plan_bytes / 1e9,
                           fft_backend=fft_backend, transfer_fp32=bool(args.transfer_fp32),
                           zero_planes_skipped=zero_planes, nz=prob.nz),
            "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": MY_KERNELS_PER_STEP[fft_backend] * args.steps,
            "stages": stages, "roofline": roofline, "cpu_baseline": cpu, "fp32_transfer_variant": variant, "all_planes_dense": dense}
    print(json.dumps(line), flush=True)
    plan.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
