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
# kernels of this library launched per product: k_bin_count, k_scan_local, k_scan_add, k_bin_scatter, k_weights, k_tile_lists, k_spread_pipe, k_spread (the tiles that overflow a staged chunk), k_solve_pair<nz> (three grid
# fields each way) or k_solve<nz> (six), k_zero_mode, k_interp, plus k_fft_x_fwd, k_fft_y_fwd, k_fft_y_inv, k_fft_x_inv with the
# library's own FFT passes (else cuFFT's kernels)
MY_KERNELS_PER_STEP = {"own": 15, "cufft": 11}


def ncu_traffic(kernel_prefix: str, cfg: int, torque_mode: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the named kernel, read from the newest committed ncu launch
    list of this configuration and torque mode (profiles/*_launches_dram_cfg<c>_<mode>.csv, written by the command its .md names).
    Returns (bytes or None, file name or None): a capture of an older build is evidence for that build, so the file is named."""
    import csv
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "*_launches_dram_cfg%d_%s.csv" % (cfg, torque_mode))))
    if not files:
        return None, None
    path = files[-1]
    rd = wr = None
    try:
        with open(path, newline="") as f:
            rows = [r for r in csv.reader(f) if len(r) > 10]
        h = rows[0]
        ki, mi, vi, ui = h.index("Kernel Name"), h.index("Metric Name"), h.index("Metric Value"), h.index("Metric Unit")
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
        for r in rows[1:]:
            if kernel_prefix not in r[ki]:
                continue
            v = float(r[vi].replace(",", "")) * scale.get(r[ui], 1.0)
            if r[mi] == "dram__bytes_read.sum" and rd is None:
                rd = v
            if r[mi] == "dram__bytes_write.sum" and wr is None:
                wr = v
    except Exception:
        return None, os.path.basename(path)
    return (rd + wr if rd is not None and wr is not None else None), os.path.basename(path)


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def stage_bytes(prob, n, fin, fout, zero_planes=0):
    """Algorithmic (compulsory) bytes per product and stage: every grid value read once and
    written once per stage.  Planes above every footprint hold no force (exactly zero) and are never interpolated from: with
    ``zero_planes`` of the nz planes skipped, spread / forward FFT / solve loads shrink by that share on the input side and
    solve stores / inverse FFT / interpolation on the output side — the bytes really needed."""
    G = prob.nx * prob.ny * prob.nz
    Kz = (prob.nx // 2 + 1) * prob.ny * prob.nz
    R, C = 8.0 * G, 16.0 * Kz
    a = 1.0 - zero_planes / float(prob.nz)
    return {"spread": a * fin * R + 72.0 * n, "fft_fwd": a * fin * (R + C), "solve": a * (fin + fout) * C,
            "fft_inv": a * fout * (C + R), "interp": a * fout * R + 72.0 * n}


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
    """Workload of the oracle legs.  Configs 1-3 are timed whole (the oracle finishes them in seconds); configs 4, 5 on a bounded
    sample of the same recipe — same kernel, heights, drives and area fraction, fewer particles (the product is linear-time,
    PAPER.md:337) — sized for ~10-30 s of host work.  Returns (problem, pos, F, T, is_whole_config)."""
    if cfg == 5:
        return workloads.monolayer_bw(n=32768, seed=1005, name="cfg5-sample-32k") + (False,)
    if cfg == 4:
        return workloads.monolayer_slit(n=32768, seed=1004, name="cfg4-sample-32k") + (False,)
    return workloads.config(cfg) + (True,)


ORACLE_DFT = "fft"       # the oracle's own plain recursive mixed-radix FFT (validated against its explicit O(n^2) sums in tests/)


def oracle_sample_text(prob, n, whole):
    return "%s: N=%d, grid %dx%dx%d%s; xy DFT: the oracle's own plain recursive FFT (dp_oracle.cpp)" % (
        prob.name, n, prob.nx, prob.ny, prob.nz, " (the whole configuration)" if whole else ", bounded sample of the same recipe")


def time_oracle(cfg: int, torque_mode: str, reps: int = 1):
    import oracle
    prob, pos, F, T, whole = cpu_sample_problem(cfg)
    best = None
    for _ in range(reps):
        t0 = time.perf_counter()
        oracle.mobility_apply(prob, pos, F, T, dft=ORACLE_DFT, torque_mode=torque_mode)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return prob, len(pos), best, oracle.num_threads(), whole


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores; each step = one product of the bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    prob, pos, F, T, whole = cpu_sample_problem(args.config)
    for _ in range(args.warmup):
        oracle.mobility_apply(prob, pos, F, T, dft=ORACLE_DFT, torque_mode=args.torque_mode)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.mobility_apply(prob, pos, F, T, dft=ORACLE_DFT, torque_mode=args.torque_mode)
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    val = len(pos) / dt
    full = workloads_describe(args.config)
    sample = oracle_sample_text(prob, len(pos), whole)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "particles/s", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": dict(full, torque_mode=args.torque_mode, same_config=bool(whole),
                           note="the oracle timed on " + ("this whole configuration" if whole else "a bounded sample of this workload")),
            "cpu_baseline": {"value": val, "unit": "particles/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def workloads_describe(cfg: int):
    names = {1: "cfg1 bottom wall N=128", 2: "cfg2 slit N=4096", 3: "cfg3 bottom-wall monolayer N=65536",
             4: "cfg4 slit monolayer N=262144", 5: "cfg5 bottom-wall microroller monolayer N=1048576"}
    return {"workload": names[cfg]}


def replica_inputs(cfg: int, rank: int):
    """Rank r of an N-replica run draws its own particles from the configuration's recipe (seed + 17 r); rank 0 is the configuration."""
    prob, pos, F, T = workloads.config(cfg)
    if rank == 0:
        return prob, pos, F, T
    seed = replica_seed(prob.seed, rank)
    if cfg == 1:
        return workloads.random_bw(seed=seed)
    if cfg == 2:
        return workloads.random_slit(seed=seed)
    if cfg in (3, 5):
        return workloads.monolayer_bw(n=prob.n, seed=seed, name=prob.name)
    return workloads.monolayer_slit(seed=seed)


KERNELS = ("k_spread", "k_fft_x_fwd", "k_fft_y_fwd", "k_solve", "k_fft_y_inv", "k_fft_x_inv", "k_interp")


def kernel_bytes(prob, n, fin, fout, zero_planes=0):
    """Bytes each kernel of the product must itself move (its compulsory reads + writes): R = one real field,
    C = one half spectrum, a = share of the planes that a footprint reaches (the others hold no force and are never interpolated from).  The two passes of a 2-D transform each read and
    write the whole field once, so the two FFT kernels of a stage together move twice SURVEY.md §8(d)'s per-stage figure."""
    G = prob.nx * prob.ny * prob.nz
    Kz = (prob.nx // 2 + 1) * prob.ny * prob.nz
    R, C = 8.0 * G, 16.0 * Kz
    a = 1.0 - zero_planes / float(prob.nz)
    return {"k_spread": a * fin * R + 72.0 * n, "k_fft_x_fwd": a * fin * (R + C), "k_fft_y_fwd": a * fin * 2 * C,
            "k_solve": a * (fin + fout) * C, "k_fft_y_inv": a * fout * 2 * C, "k_fft_x_inv": a * fout * (C + R), "k_interp": a * fout * R + 72.0 * n}


def measure(dp, torch, prob, pos, F, T, dev, dist, args, *, torque_mode, transfer_fp32=False, dense_planes=False, fft="own",
            e2e=False, clocks=False, steps=None, solve_kernel=0):
    """One timed run: plan, warm-ups, K products between CUDA events on the launching stream (max over ranks), then per-stage and
    per-FFT-pass times from the plan's own events in a separate pass, then (optionally) the end-to-end run through host buffers."""
    steps = steps or args.steps
    n = len(pos)
    use_t = T is not None
    tmode = 1 if (torque_mode == "kernel" and use_t) else 0
    plan = dp.Plan(prob, max_particles=n, use_torques=use_t, device=dev.index, fft_backend=0 if fft == "own" else 1,
                   transfer_fp32=transfer_fp32, dense_planes=dense_planes, torque_mode=tmode, solve_kernel=solve_kernel)
    out = {"torque_mode": (torque_mode if use_t else "none"), "fields": plan.fields, "fft_backend": plan.fft_backend(), "plan_device_GB": plan.device_bytes() / 1e9,
           "solve_kernel": ("k_solve_pair<%d>" if (plan.fields == 3 and plan.solve_kernel() == "pair") else "k_solve<%d>") % prob.nz}
    dpos = torch.from_numpy(pos).to(dev)
    dF = torch.from_numpy(F).to(dev)
    dT = torch.from_numpy(T).to(dev) if use_t else None
    U = torch.empty((n, 3), dtype=torch.float64, device=dev)
    Om = torch.empty((n, 3), dtype=torch.float64, device=dev) if use_t else None
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    plan.set_profiling(True)
    for _ in range(args.warmup):
        plan.mobility_apply(dpos, dF, dT, out_U=U, out_Omega=Om, stream=stream)
    barrier()
    sampler = None
    if clocks:
        sampler = ClockSampler(dev.index)
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(steps):
        plan.mobility_apply(dpos, dF, dT, out_U=U, out_Omega=Om, stream=stream)
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    if sampler is not None:
        sampler.stop_flag.set()
        sampler.join(timeout=3)
        out["clocks"] = sampler.summary()
    # per-stage / per-pass device times: separately synchronised (dp_stage_ms synchronises, so it stays out of the timed loop)
    acc = {}
    for _ in range(max(3, min(steps, 5))):
        plan.mobility_apply(dpos, dF, dT, out_U=U, out_Omega=Om, stream=stream)
        d = plan.stage_ms()
        if out["fft_backend"] == "own":
            d.update(plan.fft_pass_ms())
        for k, v in d.items():
            acc.setdefault(k, []).append(v)
    out["stage_ms"] = {k: float(np.median(v)) for k, v in acc.items()}
    assert plan.check() == 0
    out["zero_planes"] = plan.zero_planes()
    out["ms_per_step"] = max_over_ranks(dist, ms_total / steps, dev)
    if e2e:
        hp = torch.from_numpy(pos).pin_memory(); hF = torch.from_numpy(F).pin_memory()
        hT = torch.from_numpy(T).pin_memory() if use_t else None
        hU = torch.empty((n, 3), dtype=torch.float64).pin_memory()
        hO = torch.empty((n, 3), dtype=torch.float64).pin_memory() if use_t else None
        npv = lambda t: None if t is None else t.numpy()
        for _ in range(2):
            plan.mobility_apply_host(npv(hp), npv(hF), npv(hT), out_U=npv(hU), out_Omega=npv(hO))
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            plan.mobility_apply_host(npv(hp), npv(hF), npv(hT), out_U=npv(hU), out_Omega=npv(hO))   # synchronous
        dt = max_over_ranks(dist, (time.perf_counter() - t0) / steps, dev)
        world = dist.get_world_size() if dist is not None else 1
        out["e2e"] = {"value": world * n / dt, "unit": "particles/s", "ms_per_step": dt * 1e3,
                      "h2d_bytes_per_step": int(24 * n * (3 if use_t else 2)), "d2h_bytes_per_step": int(24 * n * (2 if use_t else 1))}
    plan.close()
    del dpos, dF, dT, U, Om
    return out


def kernel_table(prob, n, run, peak):
    """ms, own compulsory bytes and fraction of the HBM roofline of each of the seven grid kernels of one measured run."""
    fin = fout = run["fields"]
    st = run["stage_ms"]
    ms = {"k_spread": st.get("spread", 0.0), "k_solve": st.get("solve", 0.0), "k_interp": st.get("interp", 0.0),
          "k_fft_x_fwd": st.get("fft_x_fwd"), "k_fft_y_fwd": st.get("fft_y_fwd"), "k_fft_y_inv": st.get("fft_y_inv"), "k_fft_x_inv": st.get("fft_x_inv")}
    need = kernel_bytes(prob, n, fin, fout, run["zero_planes"])
    dense = kernel_bytes(prob, n, fin, fout, 0)
    tab = {}
    for k in KERNELS:
        t = ms[k]
        if not t:
            continue
        gbs = need[k] / (t * 1e-3) / 1e9
        tab[k] = {"ms": t, "algorithmic_GB": need[k] / 1e9, "GBps": gbs, "frac": gbs / peak, "algorithmic_GB_if_all_planes_dense": dense[k] / 1e9}
    return tab


def summarise(prob, n, run, peak, world):
    """stage table (SURVEY.md §8(d) bytes: one read + one write per field and stage), the kernel table, the north_star aggregate"""
    fin = fout = run["fields"]
    by = stage_bytes(prob, n, fin, fout, run["zero_planes"])
    by_dense = stage_bytes(prob, n, fin, fout, 0)
    st = run["stage_ms"]
    stages = {}
    for k, b in by.items():
        t = st.get(k, 0.0)
        gbs = b / (t * 1e-3) / 1e9 if t > 0 else None
        stages[k] = {"ms": t, "algorithmic_GB": b / 1e9, "GBps": gbs, "frac": (gbs / peak) if gbs else None}
    stages["bin"] = {"ms": st.get("bin", 0.0)}
    mid = sum(by[k] for k in ("fft_fwd", "solve", "fft_inv")) / 1e9
    mid_ms = sum(st.get(k, 0.0) for k in ("fft_fwd", "solve", "fft_inv"))
    mid_frac = (mid / (mid_ms * 1e-3) / peak) if mid_ms else None
    agg = {"fft_chebyshev_solve_stages": {"algorithmic_GB": mid, "ms": mid_ms, "GBps": mid / (mid_ms * 1e-3) if mid_ms else None, "frac": mid_frac,
                                          "target_frac": 0.5, "target_met": bool(mid_frac is not None and mid_frac >= 0.5)},
           "whole_product": {"algorithmic_GB": sum(by.values()) / 1e9, "ms": run["ms_per_step"],
                             "frac": sum(by.values()) / 1e9 / (run["ms_per_step"] * 1e-3) / peak,
                             "algorithmic_GB_if_all_planes_dense": sum(by_dense.values()) / 1e9}}
    return stages, agg


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-variants", action="store_true", help="skip the extra timings (other torque mode, fp32 transfer variant, dense planes, Fig. 9 workload)")
    ap.add_argument("--transfer-fp32", action="store_true", help="time the fp32 spread/interpolate variant as the main number")
    ap.add_argument("--no-fp32-variant", action="store_true", help="skip the extra timing of the fp32 spread/interpolate variant")
    ap.add_argument("--dense-planes", action="store_true", help="transform every plane (do not skip the planes no footprint reaches)")
    ap.add_argument("--torque-mode", choices=["fourier", "kernel"], default="kernel",
                    help="torques / Omega through the ES kernel's derivative (3 grid fields each way; the paper's second way, PAPER.md:335) "
                         "or through the curl in Fourier-Chebyshev space (6 fields; its first way)")
    ap.add_argument("--fft", choices=["own", "cufft"], default="own", help="xy FFT backend (own shared-memory passes, or cuFFT for comparison)")
    ap.add_argument("--solve-kernel", choices=["pair", "tile"], default="pair",
                    help="kernel of the per-wavenumber solve for products with three grid fields each way: the register-resident warp-pair "
                         "kernel (default) or the tile kernel (dp_params.solve_kernel = 1; always used with six fields)")
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

    prob, pos, F, T = replica_inputs(args.config, rank)       # replicas: each rank draws its own particles from the same recipe
    n = len(pos)
    M = lambda **kw: measure(dp, torch, prob, pos, F, T, dev, dist, args, **kw)

    # ---- the headline run: device-resident timing, clocks sampled during the timed region, end to end through host buffers
    sk = 0 if args.solve_kernel == "pair" else 1
    main_run = M(torque_mode=args.torque_mode, transfer_fp32=args.transfer_fp32, dense_planes=args.dense_planes, fft=args.fft,
                 e2e=not args.no_e2e, clocks=True, solve_kernel=sk)
    ms_step = main_run["ms_per_step"]
    value = whole_job_value(n, world, ms_step)

    # ---- the same product on the same inputs in its other forms, same rules (3 warm-ups, CUDA events, max over ranks)
    other = variant = dense = fig9 = tile = None
    if not args.no_variants and args.fft == "own":
        if main_run["solve_kernel"].startswith("k_solve_pair"):
            tile = M(torque_mode=args.torque_mode, transfer_fp32=args.transfer_fp32, dense_planes=args.dense_planes, solve_kernel=1)
            tile["what"] = "same product with dp_params.solve_kernel = 1: the tile kernel (solve.cu) instead of the warp-pair kernel (solve_pair.cu) in the solve stage"
        if T is not None:
            om = "fourier" if args.torque_mode == "kernel" else "kernel"
            other = M(torque_mode=om, transfer_fp32=args.transfer_fp32, dense_planes=args.dense_planes)
            other["what"] = ("the same forces + torques -> U, Omega product with the torques taken through " +
                             ("the curl in Fourier-Chebyshev space: six grid fields each way (the paper's first way, PAPER.md:335)" if om == "fourier" else
                              "the derivative of the ES kernel: three grid fields each way (the paper's second way, PAPER.md:335)") +
                             "; the two discretisations agree to the method's 2-3 digits, each matches its own oracle path to <= 1e-10")
        if not args.transfer_fp32 and not args.no_fp32_variant:
            variant = M(torque_mode=args.torque_mode, transfer_fp32=True, dense_planes=args.dense_planes)
            variant["what"] = ("spreading and interpolation accumulate in fp32, real-space grids stored in fp32; FFTs and solves fp64; "
                               "matches the oracle to <= 1e-5 (tests)")
        if not args.dense_planes and main_run["zero_planes"] > 0:
            dense = M(torque_mode=args.torque_mode, transfer_fp32=args.transfer_fp32, dense_planes=True)
            dense["what"] = ("same product with dense_planes = 1: the %d planes no footprint reaches are spread, transformed, solved for and transformed back too"
                             % main_run["zero_planes"])
        if world == 1 and args.config == 5:
            # context for the paper's only published timing (Fig. 9): its own grid and kernel, forces only
            p9, pos9, F9, T9 = workloads.paper_fig9(18)
            r9 = measure(dp, torch, p9, pos9, F9, T9, dev, dist, args, torque_mode="kernel")
            fig9 = {"workload": "paper Fig. 9 / Table III 'M' stand-in: N=%d, forces only, grid %dx%dx%d, m=4, beta/m=1.87, H=9.1 R_h, two-layer heights"
                                % (len(pos9), p9.nx, p9.ny, p9.nz),
                    "ms_per_step": r9["ms_per_step"], "value": len(pos9) / (r9["ms_per_step"] * 1e-3), "unit": "particles/s",
                    "stage_ms": r9["stage_ms"], "plan_device_GB": r9["plan_device_GB"],
                    "paper": "370 ms per mobility solve on a V100 for this case (PAPER.md:505): another machine's number, context only"}

    # ---- other workloads of the same path, same timing rules: what has full-size parity tests but would otherwise have no time
    #      (each: problem, particle count, measured run, description); single GPU, default configuration only
    extras = {}
    if not args.no_variants and args.fft == "own" and world == 1 and args.config == 5:
        def X(key, what, pX, posX, FX, TX, tm):
            extras[key] = (pX, len(posX), measure(dp, torch, pX, posX, FX, TX, dev, dist, args, torque_mode=tm), what)
        p4, pos4, F4, T4 = workloads.config(4)
        for tm in ("kernel", "fourier"):
            X("slit_cfg4_" + tm, "BASELINE.json configs[3]: slit channel H = 6 (two walls, App. A correction, no empty planes), N = 262,144, grid %dx%dx%d, forces + torques, torque mode %s"
              % (p4.nx, p4.ny, p4.nz, tm), p4, pos4, F4, T4, tm)
        del pos4, F4, T4
        pj, posj, Fj, Tj = workloads.monolayer_bw(n=n, seed=prob.seed, name="cfg5-jittered", xy="jittered")
        X("cfg5_jittered_lattice", "config 5 with non-overlapping in-plane positions (jittered square lattice at area fraction 0.4, SURVEY.md §8(d): the closer stand-in "
          "for the paper's hard-sphere tile, PAPER.md:492); same box, grid, heights, drives and torque mode as the headline", pj, posj, Fj, Tj, args.torque_mode)
        del posj, Fj, Tj
        p9d, pos9d, F9d, T9d = workloads.paper_fig9(18, dipole=True)
        for tm in ("kernel", "fourier"):
            X("paper_fig9_MD_" + tm, "paper Table III 'M & D' stand-in (PAPER.md:492-501): N = %d, forces + torques, grid %dx%dx%d, m = 6, beta_M/m = 1.38, beta_D/m = 2.3, H = 9.2 R_h, "
              "torque mode %s (fourier = the paper's 'additional FFTs', kernel = its second way, PAPER.md:335)" % (len(pos9d), p9d.nx, p9d.ny, p9d.nz, tm), p9d, pos9d, F9d, T9d, tm)
        del pos9d, F9d, T9d

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src = hbm_peak()
    stages, agg = summarise(prob, n, main_run, peak, world)
    ktab = kernel_table(prob, n, main_run, peak)
    cand = ktab if ktab else {"k_solve": {"ms": stages["solve"]["ms"], "GBps": stages["solve"]["GBps"], "frac": stages["solve"]["frac"],
                                          "algorithmic_GB": stages["solve"]["algorithmic_GB"], "algorithmic_GB_if_all_planes_dense": None}}
    dom = max(cand, key=lambda k: cand[k]["ms"])
    kname = {"k_solve": main_run["solve_kernel"]}.get(dom, dom)
    traffic, traffic_file = ncu_traffic(dom, args.config, main_run["torque_mode"] if T is not None else "kernel")
    frac_dense = None
    if dense is not None:
        dk = kernel_table(prob, n, dense, peak).get(dom)
        frac_dense = dk["frac"] if dk else None
    roofline = {"bound": "hbm", "kernel": kname, "achieved": cand[dom]["GBps"], "peak": peak, "unit": "GB/s", "frac": cand[dom]["frac"],
                "frac_if_all_planes_dense": frac_dense,
                "traffic": traffic, "traffic_source": ("profiles/%s (ncu capture of the build that file's .md names)" % traffic_file) if traffic_file else None,
                "peak_source": peak_src,
                "bytes": "the kernel's own compulsory reads + writes with the planes no footprint reaches left out (algorithmic_GB); "
                         "frac_if_all_planes_dense: SURVEY.md §8(d)'s dense bytes over the time of the dense_planes = 1 run",
                "note": "the solve kernel is bound by the fp64 pipe and instruction issue, not by HBM (k_solve_pair: about 3.7 k fp64 instructions per "
                        "warp and 16 modes against 64 FMA lanes per clock and SM; profiles/r2_*): the fraction is of the HBM roofline, as the contract asks",
                "kernels": ktab}
    roofline.update(agg)
    # the solve kernel against the fp64 pipe (it is bound by plain fp64 arithmetic, not by HBM): algorithmic FMAs per mode of
    # a product with F fields each way = the folded Chebyshev transforms, 2 (directions) x 2F (real columns) x (NE^2 + NO^2), plus the
    # 2(F + 1) real boundary-value problems of nz - 2 rows at 9 FMAs per row (elimination, back substitution with the two boundary
    # functionals, border update, two integrations); peak = 148 SMs x 64 FMA lanes per clock x 1.965 GHz
    ne, no, fin = (prob.nz + 1) // 2, prob.nz // 2, main_run["fields"]
    fma_mode = 2 * 2 * fin * (ne * ne + no * no) + 2 * (fin + 1) * (prob.nz - 2) * 9
    modes = (prob.nx // 2 + 1) * prob.ny - 1
    t_solve = stages["solve"]["ms"] * 1e-3
    if t_solve > 0:
        ach = 2.0 * fma_mode * modes / t_solve / 1e12
        sms = int(torch.cuda.get_device_properties(dev).multi_processor_count)
        pk = 2 * sms * 64 * 1.965e9 / 1e12
        roofline["solve_fp64"] = {"bound": "alu", "kernel": main_run["solve_kernel"], "achieved": ach, "peak": pk, "unit": "TFLOP/s",
                                  "frac": ach / pk, "algorithmic_fma_per_mode": fma_mode, "modes": modes,
                                  "peak_source": "%d SMs (queried) x 64 fp64 FMA lanes per clock x 1.965 GHz (B200_PROFILING.md unit counts)" % sms}

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        sprob, sn, sdt, cores, whole = time_oracle(args.config, args.torque_mode if T is not None else "fourier")
        cpu = {"value": sn / sdt, "unit": "particles/s", "cores": cores, "kind": "oracle", "seconds": sdt, "sample": oracle_sample_text(sprob, sn, whole)}

    def brief(r):
        if r is None:
            return None
        keep = ("spread", "fft_fwd", "solve", "fft_inv", "interp", "fft_x_fwd", "fft_y_fwd", "fft_y_inv", "fft_x_inv")
        d = {"ms_per_step": r["ms_per_step"], "value": world * n / (r["ms_per_step"] * 1e-3), "unit": "particles/s",
             "fields_each_way": r["fields"], "stage_ms": {k: r["stage_ms"][k] for k in keep if k in r["stage_ms"]},
             "plan_device_GB": r["plan_device_GB"], "what": r.get("what")}
        st2, agg2 = summarise(prob, n, r, peak, world)
        d["fft_chebyshev_solve_stages"] = agg2["fft_chebyshev_solve_stages"]
        d["whole_product_frac"] = agg2["whole_product"]["frac"]
        return d

    def extra_brief(pX, nX, r, what):
        stX, aggX = summarise(pX, nX, r, peak, world)
        return {"what": what, "ms_per_step": r["ms_per_step"], "value": nX / (r["ms_per_step"] * 1e-3), "unit": "particles/s", "fields_each_way": r["fields"],
                "solve_kernel": r["solve_kernel"], "zero_planes_skipped": r["zero_planes"], "plan_device_GB": r["plan_device_GB"],
                "stage_ms": {k: v for k, v in r["stage_ms"].items() if k != "total"}, "kernels": kernel_table(pX, nX, r, peak),
                "fft_chebyshev_solve_stages": aggX["fft_chebyshev_solve_stages"], "whole_product_frac": aggX["whole_product"]["frac"]}

    fin = fout = main_run["fields"]
    by_total = sum(stage_bytes(prob, n, fin, fout, main_run["zero_planes"]).values())
    line = {"metric": METRIC, "value": value, "unit": "particles/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workloads_describe(args.config), n_particles=n, grid=[prob.nx, prob.ny, prob.nz], wall_mode=["bottom_wall", "slit"][prob.wall_mode],
                           fields_in=fin, fields_out=fout, w=prob.w, torque_mode=main_run["torque_mode"],
                           l2="inputs (%.1f GB of grids per product) far exceed the 126 MB L2" % (by_total / 1e9 / 4),
                           parallelism="replicas" if world > 1 else "single GPU", plan_device_GB=main_run["plan_device_GB"],
                           fft_backend=main_run["fft_backend"], solve_kernel=main_run["solve_kernel"], transfer_fp32=bool(args.transfer_fp32),
                           zero_planes_skipped=main_run["zero_planes"], nz=prob.nz),
            "clocks": main_run.get("clocks"), "e2e": main_run.get("e2e"), "gpu_launches": MY_KERNELS_PER_STEP[main_run["fft_backend"]] * args.steps,
            "stages": stages, "roofline": roofline, "cpu_baseline": cpu,
            ("fourier_curl_torques" if args.torque_mode == "kernel" else "kernel_derivative_torques"): brief(other),
            "fp32_transfer_variant": brief(variant), "all_planes_dense": brief(dense), "tile_solve_kernel": brief(tile), "paper_fig9": fig9,
            "other_workloads": {k: extra_brief(*v) for k, v in extras.items()}}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
