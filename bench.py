#!/usr/bin/env python
"""bench.py -- one JSON line for the multi-RHS HISQ Dslash + CG hot path on B200.

A STEP is one pass of the whole hot path on BASELINE.json configs[1] (32^3 x 8, fp64, nRHS = 1): one
`hisq_cg` solve of (m^2 - D_eo D_oe) x = b at m = 0.01 to tol 1e-10 (index maps, gathers, Dslash,
fused A-apply, BLAS-1/reductions, convergence control: SURVEY.md 8(a) rows a1-a7) on seeded synthetic
links and a Gaussian even-site source already resident in HBM.  `value` is the metric BASELINE.json
names, HISQ Dslash GFLOP/s, counted as 1146 flop per output site per RHS over every
Dslash application the solve made, divided by the whole solve time (so BLAS-1 and host polling count
against it).  Beside it:
  dslash     pure Dslash launches (alternating D_oe / D_eo), CUDA-event timed: GFLOP/s, algorithmic GB/s
  roofline   the dominant kernel (Dslash fp64 n=1) against MEASURED_PEAKS.json's HBM copy bandwidth
  sweep      configs[2] (64^3 x 16, fp32) Dslash vs nRHS = 1, 2, 4, 8     (--no-sweep to skip)
  e2e        the same step through hisq_cg_host with pinned HOST buffers (H2D + D2H inside the timing)
  cpu_baseline  the oracle (oracle/, as it stands) on this box's host cores on a bounded sample
`--impl reference` times the oracle instead (this tier's reference arm).
Multi-GPU (torchrun): independent replicas, one per rank, no collective on the data path ("replicas
only"); value = total flops of all ranks / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FLOP_PER_SITE = 1146
# Context denominators measured on this pool's B200 with `python -m paper_2306_01098_b200.peaks`
# (profiles/r1_peaks_microbench.txt); the roofline `peak` itself comes from MEASURED_PEAKS.json.
READ_ONLY_GBS = 7420.0                       # 128-bit read-only stream over 8 GB
FMA_PEAK_GFLOPS = {4: 69600.0, 8: 36900.0}   # plain FFMA / DFMA, all SMs
CONFIGS = {
    "C1": dict(L=(8, 8, 8, 8), prec="fp64", nrhs=1, mass=0.1, tol=1e-10),
    "C2": dict(L=(32, 32, 32, 8), prec="fp64", nrhs=1, mass=0.01, tol=1e-10),
    "C3": dict(L=(64, 64, 64, 16), prec="fp32", nrhs=8, mass=None, tol=None),
    "C4": dict(L=(48, 48, 48, 12), prec="mixed", nrhs=4, mass=0.002, tol=1e-9),
    "C5": dict(L=(96, 96, 96, 24), prec="fp64", nrhs=8, mass=0.005, tol=1e-10),
}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write, burst)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        mx = [int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def aggregate(ms: float, flops: float, dist, device):
    """Whole-job throughput over ranks: (max over ranks of the device time, sum over ranks of the work).
    No collective sits on the data path ("replicas only"): this all-reduce only combines the timings."""
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    f = torch.tensor([flops], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(f, op=dist.ReduceOp.SUM)
    return t.item(), f.item()


def ncu_traffic(config: str, prec: str, nrhs: int):
    """DRAM bytes per launch of the Dslash kernel from the committed ncu captures (profiles/r1_traffic.csv), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "r1_traffic.csv")) as f:
            for line in f:
                k, _, v = line.strip().partition(",")
                if k == f"{config}:{prec}:{nrhs}":
                    return int(v)
    except Exception:
        pass
    return None


def dslash_bytes(Vh: int, nrhs: int, w: int) -> int:
    """Algorithmic (compulsory) bytes of one Dslash application: 16 links of 18 reals per output site,
    each input and each output site's colour vector once: (288 + 12 n) words per site."""
    return (288 + 12 * nrhs) * w * Vh


def time_dslash(ctx, nrhs: int, reps: int, warm: int = 5):
    """Average device time (ms) of one Dslash launch, alternating D_oe / D_eo on fixed inputs,
    one pair of CUDA events on the launching stream around 2*reps back-to-back launches."""
    a, c = ctx.new_field(nrhs), ctx.new_field(nrhs)
    b, d = ctx.new_field(nrhs), ctx.new_field(nrhs)
    a.copy_(torch.randn_like(a))
    c.copy_(torch.randn_like(c))
    for _ in range(warm):
        ctx.dslash(a, 1, out=b)
        ctx.dslash(c, 0, out=d)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        ctx.dslash(a, 1, out=b)
        ctx.dslash(c, 0, out=d)
    e1.record()
    e1.synchronize()
    return e0.elapsed_time(e1) / (2 * reps)


def oracle_sample(cfg, seed: int, budget_s: float):
    """Time the oracle on a bounded sample of the step: `iters` CG iterations of the same workload."""
    import numpy as np
    import oracle
    from paper_2306_01098_b200 import inputs
    L = cfg["L"]
    V = inputs.volume(L)
    s = torch.arange(V, dtype=torch.int64)
    X = inputs.fat_links(L, seed, s).numpy()
    W = inputs.naik_links(L, seed, s).numpy()
    b = inputs.sources(L, seed, s, cfg["nrhs"]).numpy()
    par = oracle.site_parity(L)
    b[:, par == 1, :] = 0
    t0 = time.perf_counter()
    oracle.cg(L, X, W, cfg["mass"], 1e-30, b, max_iter=1)
    t1 = time.perf_counter() - t0
    iters = max(2, min(2000, int(budget_s / max(t1 / 2, 1e-3))))   # 1 iteration = 2 A-applies incl. the final check
    t0 = time.perf_counter()
    oracle.cg(L, X, W, cfg["mass"], 1e-30, b, max_iter=iters)
    dt = time.perf_counter() - t0
    n_dslash = 2 * (iters + 1) * cfg["nrhs"]                         # + the final true-residual application
    gflops = FLOP_PER_SITE * (V // 2) * n_dslash / dt / 1e9
    return gflops, dt, iters, oracle.threads()


def run_reference(args, cfg, rank, world):
    if rank != 0:
        return
    vals, dts = [], []
    for i in range(args.warmup + args.steps):
        g, dt, iters, cores = oracle_sample(cfg, 0, args.ref_budget)
        if i >= args.warmup:
            vals.append(g)
            dts.append(dt)
    v = sum(vals) / len(vals)
    sample = f"{iters} CG iterations (2 Dslash each, + 1 final residual) of the {args.config} solve per step"
    print(json.dumps({
        "impl": "reference", "metric": "hisq_dslash_gflops", "value": v, "unit": "GFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(dts) / len(dts), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, cfg)},
        "cpu_baseline": {"value": v, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def workload_name(name, cfg):
    L = cfg["L"]
    return (f"{name}: {L[0]}x{L[1]}x{L[2]}x{L[3]} {cfg['prec']} nRHS={cfg['nrhs']} CG m={cfg['mass']} tol={cfg['tol']}, "
            "Gaussian fat links (std 0.3), Haar SU(3) Naik x(-1/24), phases folded, antiperiodic t")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C2", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--only", default="all", choices=["all", "dslash", "smear"],
                    help="dslash: time only the Dslash kernel of --config at --nrhs; smear: only hisq_smear on --config's "
                         "lattice (profiling drivers)")
    ap.add_argument("--nrhs", type=int, default=0, help="override the config's nRHS (--only dslash)")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-multishift", action="store_true")
    ap.add_argument("--no-compression", action="store_true")
    ap.add_argument("--no-partition", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--ref-budget", type=float, default=10.0)
    ap.add_argument("--dslash-reps", type=int, default=100)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    cfg = CONFIGS[args.config]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return run_reference(args, cfg, rank, world)
    if args.only == "dslash":
        return run_dslash_only(args, cfg)
    if args.only == "smear":
        return run_smear_only(args, cfg)
    if args.config == "C3":
        raise SystemExit("C3 is a Dslash-only config: use --only dslash")

    from paper_2306_01098_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libhisq has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    L, n = cfg["L"], cfg["nrhs"]
    w = 4 if cfg["prec"] == "fp32" else 8
    big = binding.layout.volume(L) > (1 << 21)
    gen_dev = dev if big else None                      # small lattices: CPU generation, bit-identical to the oracle's inputs
    ctx = binding.Hisq(L, cfg["prec"], n, dev)
    fat, naik = binding.make_links(L, rank, dev, ctx.cdtype, gen_device=gen_dev)
    ctx.set_links(fat, naik)
    del fat, naik
    b_can = binding.make_sources(L, rank, n, 0, dev, ctx.cdtype, gen_device=gen_dev)
    b = ctx.pack(b_can)
    x = ctx.new_field(n)
    b_host = b_can.cpu().pin_memory()
    x_host = torch.empty_like(b_host).pin_memory()
    Vh = ctx.Vh

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- the step, device-resident inputs ----
    for _ in range(args.warmup):
        _, info = ctx.cg(b, cfg["mass"], cfg["tol"], x=x)
    # settle: keep warming up (at most 8 more solves) until two consecutive solves agree to 3 % -- boxes have been
    # seen to run the first seconds after other heavy work up to 1.4x slower with no throttle reason reported
    extra, prev = 0, None
    while extra < 8:
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.cg(b, cfg["mass"], cfg["tol"], x=x)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        extra += 1
        if prev is not None and abs(dt - prev) <= 0.03 * prev:
            break
        prev = dt
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    n_dslash = 0
    for _ in range(args.steps):
        _, info = ctx.cg(b, cfg["mass"], cfg["tol"], x=x)
        n_dslash += 2 * (info["iterations"] + info["reliable_updates"])
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = ctx.launch_count() - l0
    clocks = sampler.stop()
    ms_all, flops_all = aggregate(ms, float(FLOP_PER_SITE) * Vh * n * n_dslash, dist, dev)
    value = flops_all / (ms_all * 1e-3) / 1e9

    # ---- the same step end to end: pinned host buffers through hisq_cg_host ----
    ctx.cg_host(x_host, b_host, cfg["mass"], cfg["tol"])
    barrier()
    t0 = time.perf_counter()
    e0.record()
    nd2 = 0
    for _ in range(args.steps):
        _, info2 = ctx.cg_host(x_host, b_host, cfg["mass"], cfg["tol"])
        nd2 += 2 * (info2["iterations"] + info2["reliable_updates"])
    e1.record()
    barrier()
    ms2 = max(e0.elapsed_time(e1), 0.0)
    ms2_all, f2_all = aggregate(ms2, float(FLOP_PER_SITE) * Vh * n * nd2, dist, dev)
    e2e_val = f2_all / (ms2_all * 1e-3) / 1e9
    field_bytes = b_host.numel() * b_host.element_size()

    # ---- the dominant kernel alone: Dslash, CUDA-event timed ----
    d_ms = min(time_dslash(ctx, n, args.dslash_reps) for _ in range(3))   # best of 3 bursts of 2*reps launches
    peak, peak_src = measured_peaks()
    alg_bytes = dslash_bytes(Vh, n, w)
    achieved = alg_bytes / (d_ms * 1e-3) / 1e9
    dsl = {"ms": d_ms, "gflops": FLOP_PER_SITE * Vh * n / (d_ms * 1e-3) / 1e9, "alg_gbs": achieved,
           "paper_model_gbs": (288 + 102 * n) * w * Vh / (d_ms * 1e-3) / 1e9,
           "frac_of_measured_copy": achieved / peak, "frac_of_8TBs": achieved / 8000.0,
           "frac_of_measured_read_only": achieved / READ_ONLY_GBS,
           "frac_of_fma_peak": FLOP_PER_SITE * Vh * n / (d_ms * 1e-3) / 1e9 / FMA_PEAK_GFLOPS[w], "tiles": ctx.tiles(n)}
    # ---- row f4 (part): the full system (D + m) x = b on both parities, same lattice, mass and tol, one solve ----
    full = None
    if not args.no_multishift and rank == 0:
        bo = ctx.pack(binding.make_sources(L, rank, n, 1, dev, ctx.cdtype, gen_device=gen_dev))
        ctx.solve_M(b, bo, cfg["mass"], cfg["tol"])
        torch.cuda.synchronize()
        e0.record()
        _, _, fi = ctx.solve_M(b, bo, cfg["mass"], cfg["tol"])
        e1.record()
        e1.synchronize()
        full = {"what": "hisq_solve_M: s_e = m b_e - D_eo b_o, CG on the even system, x_o = (b_o - D_oe x_e) / m",
                "solve_ms": e0.elapsed_time(e1), "iterations": fi["iterations"],
                "full_lattice_rel_resid": fi["true_rel_resid"]}
        del bo
    # ---- row f4: HISQ smearing of seeded thin links on the same lattice (set-up work: time and launches, context) ----
    smear = None
    if not args.no_multishift and rank == 0:
        thin = binding.make_thin_links(L, rank, dev, ctx.cdtype, 0.3, gen_device=gen_dev)
        ctx.smear(thin)
        torch.cuda.synchronize()
        l0 = ctx.launch_count()
        e0.record()
        ctx.smear(thin)
        e1.record()
        e1.synchronize()
        smear = {"what": "hisq_smear: fat7 -> U(3) projection -> fat7 + Lepage, Naik product, phases folded",
                 "ms": e0.elapsed_time(e1), "launches": int(ctx.launch_count() - l0),
                 "thin_links": "Gram-Schmidt of 1 + 0.3 x Gaussian (seeded stand-in for a thermalised configuration)"}
        # the chain a production run uses: smeared links (U(3) Naik links, 14-real compression) -> full-system solve
        sfat, snaik, _ = ctx.smear(thin, fat_scale=0.5, naik_scale=-0.5 / 24.0)
        del thin
        sc = binding.Hisq(L, cfg["prec"], n, dev)
        sc.set_option("naik_compress", 1)
        sc.set_links(sfat, snaik)
        del sfat, snaik
        bo = sc.pack(binding.make_sources(L, rank, n, 1, dev, sc.cdtype, gen_device=gen_dev))
        sc.solve_M(b, bo, cfg["mass"], cfg["tol"])
        torch.cuda.synchronize()
        e0.record()
        _, _, si = sc.solve_M(b, bo, cfg["mass"], cfg["tol"])
        e1.record()
        e1.synchronize()
        smear["solve_on_smeared_links"] = {"naik_compressed": bool(sc.naik_compressed()), "solve_ms": e0.elapsed_time(e1),
                                           "iterations": si["iterations"], "full_lattice_rel_resid": si["true_rel_resid"],
                                           "dslash_ms": time_dslash(sc, n, args.dslash_reps)}
        sc.close()
        del sc, bo
    # ---- row f2: the same Dslash and solve with compressed Naik links (14 instead of 18 reals per Naik link) ----
    comp = None
    if not args.no_compression:
        ctx.close()
        ctx = binding.Hisq(L, cfg["prec"], n, dev)
        ctx.set_option("naik_compress", 1)
        fat, naik = binding.make_links(L, rank, dev, ctx.cdtype, gen_device=gen_dev)
        ctx.set_links(fat, naik)
        del fat, naik
        if ctx.naik_compressed():
            c_ms = time_dslash(ctx, n, args.dslash_reps)
            ctx.cg(b, cfg["mass"], cfg["tol"], x=x)
            torch.cuda.synchronize()
            e0.record()
            _, ci = ctx.cg(b, cfg["mass"], cfg["tol"], x=x)
            e1.record()
            e1.synchronize()
            stored = (8 * 18 + 8 * 14 + 12 * n) * w * Vh
            comp = {"format": "Naik links as 14 reals (rows 0,1 and d = det/|row0 x row1|^2; exact for c x U(3)), fat links 18", "dslash_ms": c_ms,
                    "dslash_gflops": FLOP_PER_SITE * Vh * n / (c_ms * 1e-3) / 1e9,
                    "stored_bytes_per_launch": stored, "stored_gbs": stored / (c_ms * 1e-3) / 1e9,
                    "uncompressed_alg_gbs": alg_bytes / (c_ms * 1e-3) / 1e9, "speedup_vs_full": d_ms / c_ms,
                    "cg_solve_ms": e0.elapsed_time(e1), "cg_iterations": ci["iterations"],
                    "cg_true_rel_resid": ci["true_rel_resid"]}
    # ---- row f1: multi-shift CG on the same lattice (10 shifts over 5 decades), one solve ----
    ms = None
    if not args.no_multishift and cfg["prec"] != "mixed" and n == 1:
        import numpy as np
        shifts = [0.0] + [float(v) for v in np.geomspace(1e-4, 5.0, 9)]
        ctx.close()
        ctx = binding.Hisq(L, cfg["prec"], len(shifts), dev)
        fat, naik = binding.make_links(L, rank, dev, ctx.cdtype, gen_device=gen_dev)
        ctx.set_links(fat, naik)
        del fat, naik
        xs = ctx.new_field(len(shifts))
        ctx.cg_multishift(b, cfg["mass"], shifts, cfg["tol"], x=xs)
        torch.cuda.synchronize()
        e0.record()
        _, mi = ctx.cg_multishift(b, cfg["mass"], shifts, cfg["tol"], x=xs)
        e1.record()
        e1.synchronize()
        ms = {"shifts": len(shifts), "solve_ms": e0.elapsed_time(e1), "iterations": mi["iterations"],
              "ms_per_iteration": e0.elapsed_time(e1) / max(mi["iterations"], 1), "max_true_rel_resid": max(mi["true_rel_resid"])}
        del xs
    ctx.close()
    del ctx, b, x
    # ---- row f3: the same solve on a t-partitioned context with ONE rank (ring closed on itself): what the multi-GPU
    # machinery (mailbox halos and all-reduces, unfused updates) costs per iteration on one GPU.  Context, not a scaling number.
    part = None
    if not args.no_partition and cfg["prec"] != "mixed" and rank == 0 and L[3] >= 4 and L[3] % 2 == 0:
        from paper_2306_01098_b200 import partition
        pc = binding.Hisq(L, cfg["prec"], n, dev, part=(0, 1))
        fat, naik = partition.make_links_part(L, rank, 0, 1, dev, pc.cdtype, gen_device=gen_dev)
        pc.set_links(fat, naik)
        del fat, naik
        pb = pc.pack(partition.make_sources_part(L, rank, n, 0, 0, 1, dev, pc.cdtype, gen_device=gen_dev))
        peer = partition.PeerHalo(pc, 0, 1, n)
        px = pc.new_field(n)
        pc.cg(pb, cfg["mass"], cfg["tol"], x=px)
        torch.cuda.synchronize()
        e0.record()
        _, pi = pc.cg(pb, cfg["mass"], cfg["tol"], x=px)
        e1.record()
        e1.synchronize()
        part = {"ranks": 1, "transport": "peer mailboxes (ring closed on the rank)", "solve_ms": e0.elapsed_time(e1),
                "iterations": pi["iterations"], "ms_per_iteration": e0.elapsed_time(e1) / max(pi["iterations"], 1),
                "true_rel_resid": pi["true_rel_resid"]}
        peer.close()
        pc.close()
        del pc, pb, px

    out = {
        "metric": "hisq_dslash_gflops", "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "warmup_extra_settle": extra, "ms_per_step": ms_all / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": {"fp32": "f32", "fp64": "f64", "mixed": "f32+f64"}[cfg["prec"]], "data": "synthetic",
        "config": {"workload": workload_name(args.config, cfg), "l2": "inputs larger than L2 (links %.0f MB)" % (2 * 4 * 2 * Vh * 18 * w / 1e6),
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "cg": {"solve_ms": ms_all / args.steps, "iterations": info["iterations"], "true_residual_checks": info["reliable_updates"],
               "true_rel_resid": info["true_rel_resid"], "ms_per_iteration": ms_all / args.steps / max(info["iterations"], 1)},
        "dslash": dsl,
        "multishift_cg": ms,
        "full_system_solve": full,
        "link_smearing": smear,
        "partitioned_cg": part,
        "naik_compression": comp,
        "roofline": {"bound": "hbm", "kernel": f"dslash_kernel<{'float' if w == 4 else 'double'},NR={min(n, 8 if w == 4 else 4)}>",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": ncu_traffic(args.config, cfg["prec"], n),
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                     "timing": f"CUDA events around {2 * args.dslash_reps} back-to-back hisq_dslash calls (alternating parity), best of 3 bursts; the library launches them with programmatic dependent launch: the head of call i+1 overlaps the tail of call i (~2 us per call)"},
        "e2e": {"value": e2e_val, "unit": "GFLOP/s", "h2d_bytes_per_step": field_bytes, "d2h_bytes_per_step": field_bytes,
                "ms_per_step": ms2_all / args.steps},
        "gpu_launches": int(launches), "clocks": clocks,
    }

    if rank == 0 and not args.no_sweep:
        out["sweep"] = sweep_c3(dev, peak, args.dslash_reps)
    if rank == 0 and not args.no_sweep:
        out["paper_shape_sweep"] = sweep_paper_shape(dev, max(10, args.dslash_reps // 4))
    if rank == 0 and not args.no_cpu_baseline:
        g, dt, iters, cores = oracle_sample(cfg, 0, args.cpu_budget)
        out["cpu_baseline"] = {"value": g, "unit": "GFLOP/s", "cores": cores, "kind": "oracle",
                               "sample": f"{iters} CG iterations (2 Dslash each, + 1 final residual) of the {args.config} solve, {dt:.1f} s"}
    if rank == 0:
        print(json.dumps(out))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_smear_only(args, cfg):
    """Profiling driver: HISQ smearing of seeded thin links on one config's lattice (ncu -k regex:staple_kernel ...)."""
    from paper_2306_01098_b200 import binding
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    L = cfg["L"]
    prec = "fp64" if cfg["prec"] == "mixed" else cfg["prec"]
    ctx = binding.Hisq(L, prec, 1, dev)
    thin = binding.make_thin_links(L, 0, dev, ctx.cdtype, 0.3, gen_device=dev)
    ctx.smear(thin)
    torch.cuda.synchronize()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = max(1, args.steps)
    e0.record()
    for _ in range(reps):
        ctx.smear(thin)
    e1.record()
    e1.synchronize()
    print(json.dumps({"only": "smear", "config": args.config, "L": L, "prec": prec, "ms": e0.elapsed_time(e1) / reps,
                      "launches_per_smearing": int((ctx.launch_count() - l0) // reps)}))
    ctx.close()


def run_dslash_only(args, cfg):
    """Profiling driver: only Dslash launches of one config (ncu -k regex:dslash_kernel ...)."""
    from paper_2306_01098_b200 import binding
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    L = cfg["L"]
    n = args.nrhs if args.nrhs > 0 else cfg["nrhs"]
    prec = "fp64" if cfg["prec"] == "mixed" else cfg["prec"]
    w = 4 if prec == "fp32" else 8
    ctx = binding.Hisq(L, prec, n, dev)
    fat, naik = binding.make_links(L, 0, dev, ctx.cdtype, gen_device=dev)
    ctx.set_links(fat, naik)
    del fat, naik
    ms = time_dslash(ctx, n, args.dslash_reps)
    peak, src = measured_peaks()
    by = dslash_bytes(ctx.Vh, n, w)
    print(json.dumps({"only": "dslash", "config": args.config, "L": L, "prec": prec, "nrhs": n, "ms": ms,
                      "gflops": FLOP_PER_SITE * ctx.Vh * n / (ms * 1e-3) / 1e9, "alg_gbs": by / (ms * 1e-3) / 1e9,
                      "frac_of_measured_copy": by / (ms * 1e-3) / 1e9 / peak, "frac_of_8TBs": by / (ms * 1e-3) / 1e9 / 8000.0,
                      "tiles": ctx.tiles(n), "launches": ctx.launch_count()}))
    ctx.close()


# Table 1 of the paper: Dslash TFLOP/s on a 32^4 lattice, other hardware -- context, not a target
PAPER_TABLE1 = {"nrhs": [1, 2, 3, 4, 6, 8], "A100_fp32": [1.36, 2.36, 2.85, 3.98, 4.97, 4.95], "A100_fp64": [0.70, 1.19, 1.45, 1.92, 2.20, 2.51],
                "MI250x_GCD_fp32": [0.93, 1.65, 2.06, 2.36, 2.96, 2.79], "MI250x_GCD_fp64": [0.45, 0.85, 1.14, 0.97, 0.91, 0.95]}


def sweep_paper_shape(dev, reps):
    """The paper's own benchmark shape (32^4, nRHS = 1,2,3,4,6,8, fp32 and fp64; Fig. 5 / Table 1), on this B200."""
    from paper_2306_01098_b200 import binding
    L = (32, 32, 32, 32)
    res = {"workload": "32x32x32x32 Dslash, TFLOP/s at 1146 flop/site/RHS", "paper_table1_context": PAPER_TABLE1}
    for prec in ("fp32", "fp64"):
        ctx = binding.Hisq(L, prec, 8, dev)
        fat, naik = binding.make_links(L, 0, dev, ctx.cdtype, gen_device=dev)
        ctx.set_links(fat, naik)
        del fat, naik
        res["b200_" + prec] = [round(FLOP_PER_SITE * ctx.Vh * n / (time_dslash(ctx, n, reps) * 1e-3) / 1e12, 3)
                               for n in PAPER_TABLE1["nrhs"]]
        ctx.close()
    return res


def sweep_c3(dev, peak, reps):
    """configs[2]: 64^3 x 16, fp32 operator, nRHS = 1, 2, 4, 8: Dslash throughput vs nRHS."""
    from paper_2306_01098_b200 import binding
    cfg = CONFIGS["C3"]
    L = cfg["L"]
    ctx = binding.Hisq(L, "fp32", 8, dev)
    fat, naik = binding.make_links(L, 0, dev, ctx.cdtype, gen_device=dev)
    ctx.set_links(fat, naik)
    del fat, naik
    rows = []
    for n in (1, 2, 4, 8):
        ms = time_dslash(ctx, n, max(10, reps // 4))
        by = dslash_bytes(ctx.Vh, n, 4)
        rows.append({"nrhs": n, "ms": ms, "gflops": FLOP_PER_SITE * ctx.Vh * n / (ms * 1e-3) / 1e9,
                     "alg_gbs": by / (ms * 1e-3) / 1e9, "frac_of_measured_copy": by / (ms * 1e-3) / 1e9 / peak,
                     "frac_of_8TBs": by / (ms * 1e-3) / 1e9 / 8000.0,
                     "frac_of_fma_peak": FLOP_PER_SITE * ctx.Vh * n / (ms * 1e-3) / 1e9 / FMA_PEAK_GFLOPS[4],
                     "tiles": ctx.tiles(n)})
    ctx.close()
    return {"workload": "C3: 64x64x64x16 fp32 Dslash", "rows": rows}


if __name__ == "__main__":
    main()
