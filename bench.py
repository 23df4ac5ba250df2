#!/usr/bin/env python
"""bench.py -- template-frequency-bins/s of the batched semi-coherent F-statistic on B200.

One "step" = one fstat_eval_batch call = the whole hot path (a1 prologue, a2-a5 fused template + inner
products, a6 epilogue) over one batch of P synthetic particles against resident data.  Default
workload = BASELINE.json configs[1] ("First stage": 2.5 yr, 1 577 880 bins, N_p = 1024, P = 2048).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config first_stage] [--impl reference]

Prints ONE JSON line.  ``--impl reference`` times the CPU oracle as it
stands on the host cores (bounded sample per step).  The CUDA arm never touches oracle/ except for the
separately reported ``cpu_baseline`` leg.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synthetic as syn  # noqa: E402

METRIC = "template_frequency_bins_per_s"
UNIT = "template-bins/s"

# FP64-pipe instructions (DFMA + DMUL + DADD + DSETP) of the two main kernels, per unit of work (DESIGN.md
# "Roofline").  The numerator of the roofline is an EXECUTED-INSTRUCTION model, not a flop count:
#   per template-bin of the interpolating kernel and of the direct kernel: counted in the SASS of the library that
#       is loaded, at run time (sass_fp64_mix below; the constants here are only the fallback when cuobjdump is
#       missing, and tests/test_cabi.py checks them against the SASS);
#   per node interval and per work item of a particle: EXECUTED counts measured with ncu
#       (sm__inst_executed_pipe_fp64.sum at forced strides 8 / 512 and two segment lengths; profiles/ names the build).
FAST_FP64_PER_BIN = 19.0
FAST_FP64_PER_INTERVAL = 648.0
FAST_FP64_PER_ITEM = 842.0
DIRECT_FP64_PER_BIN = 267.0
FP64_COUNTS_BUILD = ("per node interval / per work item: least-squares fit to ncu executed counts (smsp__inst_executed_pipe_fp64.sum) of "
                     "build bd29abd at six settings (automatic strides, forced strides 8 / 64 / 512, another segment length, config 2 "
                     "N_p = 16); the fit reproduces each of the six totals within 0.2 % (profiles/r2.md)")
NOMINAL_FP64_INST_PER_S = 148 * 64 * 1.965e9        # 148 SMs x 64 FP64 lanes x 1.965 GHz (B200_PROFILING.md)
STRIDES = (0, 8, 16, 32, 64, 128, 256, 512)          # index 0 = direct kernel
# dram__bytes_read.sum + dram__bytes_write.sum of one fstat_fast_kernel launch on the default workload, from the
# ncu --set full capture named beside it (None when no capture of the current hot kernel exists)
NCU_DRAM_BYTES_PER_LAUNCH = 222.4e6
# the same capture: smsp__inst_executed.sum = 29.72 warp instructions per template-bin, 23.51 of them on the FP64 pipe
NCU_OTHER_INST_PER_TEMPLATE_BIN = 29.72 - 23.51
NCU_DRAM_CAPTURE = "profiles/r2.md (34.3 MB read + 188.1 MB written), ncu capture of build bd29abd"
# row f2 (fstat_fastband_kernel), per WARP-level unit of work counted by the kernel itself (fstat_plan_band_stats): the
# per-bin and per-interval counts are those of fstat_fast_kernel; a node interval in which some lane has a partition edge
# runs the cut path as well (calibrated on the ncu capture of profiles/r2_bands.md: 9.897e8 FP64 warp-instructions)
BAND_FP64_PER_INTERVAL = 736.0      # fstat_fastband_kernel keeps the four-node sub-block code of round-2 build 1ecb204
BAND_FP64_PER_RUN = 1105.0
BAND_FP64_PER_CUT_INTERVAL = 350.0
NCU_BAND_DRAM_BYTES = 120.6e6     # profiles/r2_bands.md: N_seg = 1024, edges at any bin, config 1 data, build 2d160f1 (84.5 MB read + 36.1 MB written)


def sass_fp64_mix(lib_path):
    """FP64-pipe instruction mix of the per-bin loop of fstat_fast_kernel, from `cuobjdump -sass` of the loaded
    library: {"per_bin": FP64 instructions per bin, "dfma", "dadd", "dmul", "dsetp": each per bin, "all_per_bin":
    instructions of every pipe per bin}.  None when cuobjdump is unavailable.  The per-bin loop is the innermost
    loop that reads the folded data from shared memory (LDS) and holds >= 10 FP64 instructions."""
    import re
    try:
        out = subprocess.run(["cuobjdump", "-sass", lib_path], capture_output=True, text=True, check=True).stdout
    except (OSError, subprocess.CalledProcessError):
        return None
    m = re.search(r"Function : \S*fstat_fast_kernel", out)
    if not m:
        return None
    j = out.find("Function :", m.end())
    ins = []
    for line in out[m.start():j if j > 0 else None].splitlines():
        mm = re.search(r"/\*([0-9a-f]{4,5})\*/\s+(.*?);", line)
        if mm:
            w = mm.group(2).split()
            op = w[1] if w[0].startswith("@") else w[0]
            ins.append((int(mm.group(1), 16), op.split(".")[0], mm.group(2)))
    loops = []
    for a, op, text in ins:
        if op == "BRA":
            t = re.search(r"(0x[0-9a-f]+)\s*$", text)
            if t and int(t.group(1), 16) < a:
                loops.append((int(t.group(1), 16), a))
    best = None
    for lo, hi in loops:
        if any(lo <= l2 and h2 <= hi and (l2, h2) != (lo, hi) for l2, h2 in loops):
            continue
        body = [op for a, op, _ in ins if lo <= a <= hi]
        n_lds = body.count("LDS")
        n64 = sum(body.count(o) for o in ("DFMA", "DADD", "DMUL", "DSETP"))
        if n_lds >= 2 and n64 >= 10 * n_lds:                 # the unrolled 4-bin runs (one LDS.128 per bin)
            cand = {"per_bin": n64 / n_lds, "dfma": body.count("DFMA") / n_lds, "dadd": body.count("DADD") / n_lds,
                    "dmul": body.count("DMUL") / n_lds, "dsetp": body.count("DSETP") / n_lds,
                    "all_per_bin": len(body) / n_lds}
            if best is None or n_lds > best[0]:
                best = (n_lds, cand)
    return best[1] if best else None


# ------------------------------------------------------------------------------------------ utilities
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return float(d.get("hbm_gbs", 6650.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="first_stage", help="tiny | first_stage | middle_stages | final_coherent | wide_band")
    ap.add_argument("--n-part", type=int, default=None, help="override N_p (default: the config's first)")
    ap.add_argument("--particles", type=int, default=None, help="override P (default: the config's first)")
    ap.add_argument("--force-level", type=int, default=-2, help="plan option force_level (-2 automatic stride)")
    ap.add_argument("--max-segment-bins", type=int, default=0, help="plan option max_segment_bins (0 automatic)")
    ap.add_argument("--interp-tol", type=float, default=1.0, help="plan option interp_tol")
    ap.add_argument("--pso", type=int, default=0, metavar="ITERS",
                    help="also time ITERS iterations of the device PSO (row f1) on this plan: swarms of 128 particles")
    ap.add_argument("--bands", type=int, default=None, metavar="N_SEG",
                    help="also time fstat_eval_batch_bands (row f2: per-template bands, N_SEG partitions) on this plan; default: "
                         "1024 on the default workload unless --no-sweep, else off")
    ap.add_argument("--bands-lattice", type=int, default=1,
                    help="edge lattice of --bands in bins (1: edges at any bin; >= 32: the lattice cells are the work units)")
    ap.add_argument("--channels", type=int, default=None, metavar="N",
                    help="also time fstat_eval_batch_channels (row f4: the first N of the TDI channels A, E, T, common amplitudes); "
                         "default: 3 on the default workload unless --no-sweep, else off")
    ap.add_argument("--graph", action="store_true",
                    help="also time fstat_eval_batch_noalloc captured once in a CUDA graph and replayed (small problems are launch-bound)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweep", action="store_true",
                    help="skip what the default workload adds to the line: the N_p sweep rows and the rows f2 / f4 legs (bands, channels)")
    ap.add_argument("--cpu-sample", type=int, default=None, help="particles in the cpu_baseline sample")
    args = ap.parse_args()
    default_wl = args.config == "first_stage" and args.n_part is None and args.particles is None and args.impl == "ours"
    extras = default_wl and not args.no_sweep
    if args.bands is None:
        args.bands = 1024 if extras else 0
    if args.channels is None:
        args.channels = 3 if extras else 0
    return args


def dataset_for(cfg, template_fn):
    t0 = time.time()
    ds = syn.make_dataset(cfg, template_fn)
    return ds, time.time() - t0


def gpu_template_fn(fs, cfg):
    """Injection template from the library itself (fstat_eval_template): the CUDA arm needs no oracle."""
    def fn(params6, freq):
        n = freq.shape[0]
        with fs.fstat_plan_create(freq, np.zeros(n, dtype=np.complex128), np.ones(n), np.array([0, n])) as plan:
            up, uc = fs.fstat_eval_template(plan, params6)
            return up.cpu().numpy(), uc.cpu().numpy()
    return fn


def rank_particles(cfg, P, rank, world):
    """Weak scaling: every rank evaluates its own batch of P particles (one swarm set per GPU)."""
    allp = syn.draw_particles(cfg, P * world)
    return np.ascontiguousarray(allp[rank * P:(rank + 1) * P])


def cpu_baseline(cfg, ds, n_part, sample=None):
    """The oracle as it stands, on the host cores, on a bounded sample of the same workload."""
    from oracle import oracle as orc
    orc.build()
    cores = orc.max_threads()
    edges = ds.edges(n_part)
    one = syn.draw_particles(cfg, 1)
    t0 = time.time()
    orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, one, n_threads=1)
    t1 = max(time.time() - t0, 1e-4)                      # one particle on one core
    if sample is None:                                     # aim at ~20 s of CPU work, at least one per core
        sample = int(min(max(cores, round(20.0 / t1)), 8 * cores, 4096))
    par = syn.draw_particles(cfg, sample)
    t0 = time.time()
    orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
    dt = time.time() - t0
    return {"value": sample * ds.n_bins / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d particles x %d bins (all partitions, N_p=%d) of the workload, %.2f s wall, "
                      "OpenMP over particles; 1 particle on 1 core: %.2f s" % (sample, ds.n_bins, n_part, dt, t1),
            "particles_per_s": sample / dt}


def run_reference(args):
    """--impl reference: the CPU oracle, unmodified, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from oracle import oracle as orc
    orc.build()
    cfg = syn.config_by_name(args.config)
    n_part = args.n_part or cfg.n_part[0]
    ds, _ = dataset_for(cfg, orc.template)
    cores = orc.max_threads()
    edges = ds.edges(n_part)
    t0 = time.time()
    orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, syn.draw_particles(cfg, 1), n_threads=1)
    t1 = max(time.time() - t0, 1e-4)
    total = max(args.steps + args.warmup, 1)
    # bounded sample per step: the whole run stays within ~2 minutes of wall time
    sample = int(min(max(1, round(120.0 / total / t1 * cores)), 4 * cores, args.particles or cfg.P[0]))
    par = syn.draw_particles(cfg, sample)
    for _ in range(args.warmup):
        orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
    t0 = time.time()
    for _ in range(args.steps):
        orc.fstat_batch(ds.freq, ds.dw, ds.inv_sn, edges, par)
    dt = time.time() - t0
    value = args.steps * sample * ds.n_bins / dt
    desc = "%d particles x %d bins per step, N_p=%d" % (sample, ds.n_bins, n_part)
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": cfg.name, "n_bins": ds.n_bins, "n_part": n_part, "particles_per_step": sample,
                      "note": "CPU oracle (oracle/fstat_oracle.c, gcc -O2, OpenMP over particles), bounded sample"},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))
    return 0


def fp64_model(fs, plan, P, n_bins, mix):
    """Executed FP64-pipe thread-instructions of the main kernels for the most recent evaluation on `plan` (P particles):
    per-bin x bins at each stride + per-interval x node intervals + per-item x CTA runs + direct bins, summed over the
    particle groups (fstat_plan_level_bins), x 128 particles per group."""
    lvl_bins, lvl_sub = fs.fstat_plan_level_bins(plan)
    n_items = fs.fstat_plan_n_ctas(plan, P)
    per_bin = mix["per_bin"] if mix else FAST_FP64_PER_BIN
    fast_share = float(lvl_bins[1:].sum()) / max(float(lvl_bins.sum()), 1.0)
    inst = 128.0 * (per_bin * float(lvl_bins[1:].sum()) + FAST_FP64_PER_INTERVAL * float(lvl_sub.sum())
                    + FAST_FP64_PER_ITEM * n_items * fast_share + DIRECT_FP64_PER_BIN * float(lvl_bins[0]))
    # flops with DFMA = 2, DADD = DMUL = 1, DSETP = 0: the per-bin mix from the SASS for the per-bin part; the rest of
    # the kernel (node evaluations, coefficients, Gram products) is FMA chains almost throughout: counted as the
    # per-bin mix too (an under-estimate of its flops)
    flop_per_inst = ((2.0 * mix["dfma"] + mix["dadd"] + mix["dmul"]) / mix["per_bin"]) if mix else 27.5 / 19.0
    share = {str(S): float(b) / max(float(lvl_bins.sum()), 1.0) for S, b in zip(STRIDES, lvl_bins)}
    return inst, inst * flop_per_inst, share, float(lvl_sub.sum()), n_items


def timed_steps(fs, torch, plan, par, F, Fk, stream, scratch, steps, warmup):
    """W warm-up evaluations, then `steps` evaluations each bracketed by its own CUDA event pair on the launch stream,
    L2 flushed (256 MiB write, not timed) before each.  Returns (mean ms per step, mean ms of the main kernels)."""
    for _ in range(warmup):
        fs.fstat_eval_batch(plan, par, F, Fk, stream)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in ev:
        scratch.fill_(5)
        e0.record(stream)
        fs.fstat_eval_batch(plan, par, F, Fk, stream)
        e1.record(stream)
    torch.cuda.synchronize()
    ms = float(np.mean([e0.elapsed_time(e1) for e0, e1 in ev]))
    main_ms = fs.fstat_plan_main_kernel_ms(plan, min(steps, 128))
    return ms, (float(np.mean(main_ms)) if len(main_ms) else float("nan"))


def run_sweep(fs, torch, plan1, ds1, args, mix, fp64_rate, stream, scratch):
    """north_star's "2.5-year N_p sweep" in the driver-run line: configs 2 (P = 8192; N_p = 256, 64, 16) and 3 (P = 4096,
    N_p = 1) on config 1's data through fstat_plan_set_partitions, and one wide-band point (config 4, P = 4096,
    N_p = 16).  Same timing rules as the headline step, fewer steps."""
    rows = []
    steps, warm = max(min(args.steps, 8), 3), 3

    def point(cfg, ds, plan, n_part, P):
        par = torch.as_tensor(np.ascontiguousarray(syn.draw_particles(cfg, P)), device="cuda")
        F = torch.empty(P, dtype=torch.float64, device="cuda")
        Fk = torch.empty((P, n_part), dtype=torch.float64, device="cuda")
        ms, main_ms = timed_steps(fs, torch, plan, par, F, Fk, stream, scratch, steps, warm)
        inst, _, share, _, _ = fp64_model(fs, plan, P, ds.n_bins, mix)
        rows.append({"workload": cfg.name, "n_bins": ds.n_bins, "n_part": n_part, "particles": P, "steps": steps,
                     "ms_per_step": ms, "value": float(P) * ds.n_bins / (ms * 1e-3), "unit": UNIT,
                     "particles_per_s": float(P) / (ms * 1e-3), "main_kernel_ms": main_ms,
                     "fp64_inst_per_template_bin": inst / (float(P) * ds.n_bins),
                     "frac": inst / (main_ms * 1e-3) / fp64_rate if fp64_rate > 0 else None,
                     "frac_of_nominal": inst / (main_ms * 1e-3) / NOMINAL_FP64_INST_PER_S,
                     "direct_kernel_share_of_bins": share["0"], "plan_table_bytes": fs.fstat_plan_table_bytes(plan)})

    cfg2, cfg3, cfg4 = syn.CONFIGS[2], syn.CONFIGS[3], syn.CONFIGS[4]
    for n_part in cfg2.n_part:
        fs.fstat_plan_set_partitions(plan1, ds1.edges(n_part))
        point(cfg2, ds1, plan1, n_part, cfg2.P[0])
    fs.fstat_plan_set_partitions(plan1, ds1.edges(1))
    point(cfg3, ds1, plan1, 1, cfg3.P[0])
    ds4 = syn.make_dataset(cfg4, gpu_template_fn(fs, cfg4))
    with fs.fstat_plan_create(ds4.freq, ds4.dw, ds4.inv_sn, ds4.edges(16)) as plan4:
        point(cfg4, ds4, plan4, 16, 4096)
    return rows


def run_ours(args):
    import torch
    import paper_2407_10797_b200 as fs
    from paper_2407_10797_b200 import build as cuda_build

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        cuda_build.build()
    if dist is not None:
        dist.barrier()
    fs.load_library()

    cfg = syn.config_by_name(args.config)
    n_part = args.n_part or cfg.n_part[0]
    P = args.particles or cfg.P[0]
    ds, t_data = dataset_for(cfg, gpu_template_fn(fs, cfg))
    edges = ds.edges(n_part)
    t0 = time.time()
    opts = fs.fstat_default_options(force_level=args.force_level, max_segment_bins=args.max_segment_bins,
                                    interp_tol=args.interp_tol)
    plan = fs.fstat_plan_create(ds.freq, ds.dw, ds.inv_sn, edges, opts)
    torch.cuda.synchronize()
    t_plan = time.time() - t0

    par_np = rank_particles(cfg, P, rank, world)
    par = torch.as_tensor(par_np, device="cuda")
    F = torch.empty(P, dtype=torch.float64, device="cuda")
    Fk = torch.empty((P, n_part), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident arm: W warm-up steps, then exactly K timed steps
    for _ in range(args.warmup):
        fs.fstat_eval_batch(plan, par, F, Fk, stream)
    barrier()
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    # exactly K timed steps; L2 (126 MB) is flushed before each one by a 256 MiB write that is NOT timed:
    # every step has its own event pair on the launch stream and the step times are summed
    scratch = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches_before = fs.fstat_plan_launch_count(plan)
    for e0, e1 in ev:
        scratch.fill_(1)
        e0.record(stream)
        fs.fstat_eval_batch(plan, par, F, Fk, stream)
        e1.record(stream)
    barrier()
    launches_timed = fs.fstat_plan_launch_count(plan) - launches_before      # our kernels inside the timed steps
    ms_total = float(sum(e0.elapsed_time(e1) for e0, e1 in ev))
    main_ms = fs.fstat_plan_main_kernel_ms(plan, min(args.steps, 128))
    clk = clocks.stop() if rank == 0 else None
    if dist is not None:
        t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / max(args.steps, 1)
    tb_per_step = float(P) * ds.n_bins * world
    value = tb_per_step / (ms_step * 1e-3)
    F_host = F.cpu().numpy()

    # ---- end-to-end arm: host (pinned) buffers through fstat_eval_batch_host, copies inside the timing
    par_pin = torch.as_tensor(par_np).pin_memory()
    F_pin = torch.empty(P, dtype=torch.float64).pin_memory()
    Fk_pin = torch.empty((P, n_part), dtype=torch.float64).pin_memory()
    for _ in range(min(args.warmup, 3)):
        fs.fstat_eval_batch_host(plan, par_pin, F_pin, Fk_pin, stream)
    barrier()
    hv = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for h0, h1 in hv:
        scratch.fill_(2)
        h0.record(stream)
        fs.fstat_eval_batch_host(plan, par_pin, F_pin, Fk_pin, stream)
        h1.record(stream)
    barrier()
    ms_e2e = float(sum(h0.elapsed_time(h1) for h0, h1 in hv))
    if dist is not None:
        t = torch.tensor([ms_e2e], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_e2e = float(t.item())
    e2e_value = tb_per_step / (ms_e2e / max(args.steps, 1) * 1e-3)
    assert np.array_equal(F_pin.numpy(), F_host), "host-buffer call disagrees with the device-resident call"

    if rank != 0:
        fs.fstat_plan_destroy(plan)
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant (main) kernels: FP64 pipe
    main_mean = float(np.mean(main_ms)) if len(main_ms) else float("nan")
    mix = sass_fp64_mix(fs.library_path())
    fp64_inst, fp64_flop, stride_share, n_intervals, n_items = fp64_model(fs, plan, P, ds.n_bins, mix)
    fp64_rate, n_sm = fs.fstat_probe_pipe_peak(0, 60.0, local)
    fp32_rate, _ = fs.fstat_probe_pipe_peak(1, 30.0, local)
    mufu_rate, _ = fs.fstat_probe_pipe_peak(2, 30.0, local)
    mixed_rate, _ = fs.fstat_probe_pipe_peak(3, 30.0, local)
    achieved = fp64_inst / (main_mean * 1e-3)                 # FP64-pipe thread-instructions per second
    # What the kernel's OTHER instructions cost it: an FP64 warp instruction occupies an SM sub-partition's FP64 pipe for
    # two cycles, and the 4 : 1 probe shows how many more cycles an instruction of another pipe takes there (about 0.2 on
    # B200: they issue in the gaps).  With n64 FP64 and n_other other instructions per template-bin the FP64 pipe can be
    # busy at most 2 n64 / (2 n64 + cost n_other) of the time: the bound this instruction mix allows.
    other_cost = 8.0 * (fp64_rate / mixed_rate - 1.0) if mixed_rate > 0 else None
    hbm_peak, hbm_src = peaks()
    n_groups = (P + 127) // 128
    # algorithmic HBM bytes of one launch: every particle group streams the folded data (16 B/bin) once, reads
    # one 192-B node row and one 192-B sub-block table per node interval, and writes one 80-B record of partial sums per
    # particle and segment (counted here per CTA run: a lower bound when a run holds several segments)
    hbm_bytes = 16.0 * ds.n_bins * n_groups + (192.0 + 192.0) * n_intervals + 80.0 * 128.0 * n_items
    default_wl = cfg.name == "first_stage" and n_part == 1024 and P == 2048
    roofline = {"bound": "alu", "kernel": "fstat_fast_kernel (+ fstat_main_kernel for the work items it leaves)",
                "pipe": "fp64",
                "achieved": achieved / 1e12, "peak": fp64_rate / 1e12, "unit": "T FP64-pipe inst/s",
                "frac": achieved / fp64_rate if fp64_rate > 0 else None,
                "frac_is": "executed FP64-pipe instructions (DFMA, DADD, DMUL, DSETP: one issue slot each) per second / the "
                           "builder-measured dependent-free DFMA stream of this run (fstat_probe_pipe_peak); a pipe-slot "
                           "utilisation, not a flop rate",
                "nominal_peak": NOMINAL_FP64_INST_PER_S / 1e12, "frac_of_nominal": achieved / NOMINAL_FP64_INST_PER_S,
                "flop_tflops": fp64_flop / (main_mean * 1e-3) / 1e12,
                "flop_frac": fp64_flop / (main_mean * 1e-3) / (2.0 * fp64_rate) if fp64_rate > 0 else None,
                "flop_frac_is": "flops with DFMA = 2, DADD = DMUL = 1 (mix of the per-bin loop from the SASS) / (2 x the DFMA rate)",
                "traffic": NCU_DRAM_BYTES_PER_LAUNCH if default_wl else None,
                "traffic_source": NCU_DRAM_CAPTURE if default_wl else None,
                "fp64_inst_per_launch": fp64_inst, "fp64_inst_per_template_bin": fp64_inst / (float(P) * ds.n_bins),
                "fp64_inst_model": {"fast_per_bin": mix["per_bin"] if mix else FAST_FP64_PER_BIN,
                                    "fast_per_bin_source": "SASS of the loaded library (cuobjdump) at run time" if mix
                                                           else "constant in bench.py (cuobjdump unavailable)",
                                    "fast_per_bin_mix": mix,
                                    "fast_per_node_interval": FAST_FP64_PER_INTERVAL,
                                    "fast_per_work_item": FAST_FP64_PER_ITEM, "direct_per_bin": DIRECT_FP64_PER_BIN,
                                    "source": FP64_COUNTS_BUILD},
                "stride_share_of_bins": stride_share,
                "main_kernel_ms": main_mean, "main_kernel_share_of_step": main_mean / ms_step,
                "measured_pipe_peaks_inst_per_s": {"fp64_fma": fp64_rate, "fp32_fma": fp32_rate, "mufu": mufu_rate,
                                                   "fp64_fma_with_one_fp32_per_four": mixed_rate},
                "hbm": {"algorithmic_bytes_per_launch": hbm_bytes,
                        "achieved_gbs": hbm_bytes / (main_mean * 1e-3) / 1e9,
                        "peak_gbs": hbm_peak, "peak_source": hbm_src}}

    if default_wl and other_cost is not None and roofline["frac"]:
        n64 = roofline["fp64_inst_per_template_bin"]
        bound = 2.0 * n64 / (2.0 * n64 + other_cost * NCU_OTHER_INST_PER_TEMPLATE_BIN)
        roofline["dispatch"] = {"other_inst_cost_cycles": other_cost,
                                "other_inst_per_template_bin": NCU_OTHER_INST_PER_TEMPLATE_BIN,
                                "other_inst_source": NCU_DRAM_CAPTURE,
                                "frac_bound_of_this_mix": bound, "frac_of_bound": roofline["frac"] / bound,
                                "is": "an FP64 warp instruction occupies the pipe for 2 cycles, another instruction costs "
                                      "other_inst_cost_cycles more (4 : 1 probe of this run): the share of time the FP64 pipe CAN be "
                                      "busy with this kernel's instruction mix; the rest of the gap is dependency and barrier stalls"}
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": cfg.name, "T_s": cfg.T, "n_bins": ds.n_bins, "n_part": n_part,
                      "particles_per_gpu": P, "parallelism": "particles sharded over %d GPU(s), plan replicated, "
                      "no collective on the data path" % world,
                      "l2": "L2 flushed before every timed step (256 MiB scratch write, outside the timed events)",
                      "n_ctas": fs.fstat_plan_n_ctas(plan, P), "n_sm": n_sm,
                      "plan_options": {"force_level": args.force_level, "max_segment_bins": args.max_segment_bins,
                                       "interp_tol": args.interp_tol},
                      "plan_create_s": t_plan, "dataset_s": t_data,
                      "plan_table_bytes": fs.fstat_plan_table_bytes(plan)},
           "particles_per_s": float(P) * world / (ms_step * 1e-3),
           "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(par_pin.numel() * 8),
                   "d2h_bytes_per_step": int(F_pin.numel() * 8 + Fk_pin.numel() * 8),
                   "ms_per_step": ms_e2e / max(args.steps, 1),
                   "call": "fstat_eval_batch_host (pinned host params in; F and F_k out)"},
           "gpu_launches": int(launches_timed),
           "clocks": clk, "roofline": roofline}
    if default_wl and world == 1 and not args.no_sweep:
        out["sweep"] = run_sweep(fs, torch, plan, ds, args, mix, fp64_rate, stream, scratch)
        fs.fstat_plan_set_partitions(plan, edges)
    if args.graph:
        # the same step as `value`, through the no-allocation entry point captured once into a CUDA graph: a replay costs one
        # launch on the host instead of seven.  Not timed with the L2 flush in between (a replay loop is the use case).
        fs.fstat_eval_batch_noalloc(plan, par, F, Fk, stream)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            fs.fstat_eval_batch_noalloc(plan, par, F, Fk)
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize()
        n_g = max(args.steps, 1) * 10
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record()
        for _ in range(n_g):
            g.replay()
        g1.record()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(n_g):
            fs.fstat_eval_batch(plan, par, F, Fk, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        out["graph"] = {"call": "fstat_eval_batch_noalloc captured in a CUDA graph", "replays": n_g,
                        "ms_per_replay": g0.elapsed_time(g1) / n_g,
                        "ms_per_step_back_to_back_without_graph": e0.elapsed_time(e1) / n_g,
                        "template_bins_per_s": float(P) * ds.n_bins / (g0.elapsed_time(g1) / n_g * 1e-3)}
        del g
    if args.pso > 0:
        # row f1: ITERS iterations of the device PSO (update -> fstat_eval_batch -> personal bests) enqueued back to
        # back on the stream, no host synchronisation in between; box = the particle ranges of the workload
        lo, hi = par_np.min(axis=0), par_np.max(axis=0)
        n_sw = max(P // 128, 1)
        pso = fs.fstat_pso_create(plan, n_sw, 128, args.pso, lo, hi, seed=1, stream=stream)
        fs.fstat_pso_iterate(pso, 3, stream)
        torch.cuda.synchronize()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record(stream)
        fs.fstat_pso_iterate(pso, args.pso, stream)
        p1.record(stream)
        torch.cuda.synchronize()
        ms_it = p0.elapsed_time(p1) / args.pso
        _, bf = fs.fstat_pso_best(pso, stream)
        out["pso"] = {"swarms": n_sw, "particles_per_swarm": 128, "iterations": args.pso, "ms_per_iteration": ms_it,
                      "template_bins_per_s": float(n_sw * 128) * ds.n_bins / (ms_it * 1e-3),
                      "overhead_vs_eval_step": ms_it / ms_step - 1.0, "best_F_max": float(bf.max())}
        fs.fstat_pso_destroy(pso)
        if args.bands > 0:
            # rows f1 x f2: the same swarms with fstat_eval_batch_bands as their fitness
            po = fs.fstat_pso_default_options(band_n_seg=args.bands, band_lattice=args.bands_lattice)
            pso = fs.fstat_pso_create(plan, n_sw, 128, args.pso, lo, hi, seed=1, opts=po, stream=stream)
            fs.fstat_pso_iterate(pso, 3, stream)
            torch.cuda.synchronize()
            p0.record(stream)
            fs.fstat_pso_iterate(pso, args.pso, stream)
            p1.record(stream)
            torch.cuda.synchronize()
            _, bf = fs.fstat_pso_best(pso, stream)
            out["pso"]["bands_fitness"] = {"n_seg": args.bands, "edge_lattice": args.bands_lattice,
                                           "ms_per_iteration": p0.elapsed_time(p1) / args.pso, "best_F_max": float(bf.max())}
            fs.fstat_pso_destroy(pso)
    if args.bands > 0:
        # row f2: the paper's own segment limits; unit = IN-BAND template-bins (bins with t_f in [0, T] per particle)
        for _ in range(2):
            _, _, band = fs.fstat_eval_batch_bands(plan, par, args.bands, args.bands_lattice, stream)
        torch.cuda.synchronize()
        n_b = max(min(args.steps, 10), 1)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_b)]
        for e0, e1 in evs:
            scratch.fill_(3)
            e0.record(stream)
            fs.fstat_eval_batch_bands(plan, par, args.bands, args.bands_lattice, stream)
            e1.record(stream)
        torch.cuda.synchronize()
        ms_b = float(np.mean([e0.elapsed_time(e1) for e0, e1 in evs]))
        kms = fs.fstat_plan_main_kernel_ms(plan, n_b)
        in_band = float((band[:, 1] - band[:, 0]).sum().item())
        # end to end through the host-buffer call: params in, F, F_k and the band limits out
        fs.fstat_eval_batch_bands_host(plan, par_pin, args.bands, args.bands_lattice, stream)      # pinned, as the headline e2e
        t0 = time.perf_counter()
        for _ in range(n_b):
            fs.fstat_eval_batch_bands_host(plan, par_pin, args.bands, args.bands_lattice, stream)
        ms_b_e2e = (time.perf_counter() - t0) * 1e3 / n_b
        st = fs.fstat_plan_band_stats(plan)               # warp-level bins, intervals, intervals with a cut, runs
        per_bin = mix["per_bin"] if mix else FAST_FP64_PER_BIN
        b_inst = 32.0 * (per_bin * st[0] + BAND_FP64_PER_INTERVAL * st[1] + BAND_FP64_PER_CUT_INTERVAL * st[2]
                         + BAND_FP64_PER_RUN * st[3])
        kms_mean = float(np.mean(kms)) if len(kms) else float("nan")
        band_roofline = {"bound": "alu", "pipe": "fp64", "kernel": "fstat_fastband_kernel",
                         "achieved": b_inst / (kms_mean * 1e-3) / 1e12, "peak": fp64_rate / 1e12, "unit": "T FP64-pipe inst/s",
                         "frac": b_inst / (kms_mean * 1e-3) / fp64_rate if fp64_rate > 0 else None,
                         "traffic": NCU_BAND_DRAM_BYTES if (default_wl and args.bands == 1024 and args.bands_lattice == 1) else None,
                         "fp64_inst_per_call": b_inst, "fp64_inst_per_in_band_template_bin": b_inst / max(in_band, 1.0),
                         "warp_bins": int(st[0]), "warp_node_intervals": int(st[1]), "warp_intervals_with_a_cut": int(st[2]),
                         "warp_runs": int(st[3]), "bins_walked_share_of_grid": 32.0 * st[0] / (float(P) * ds.n_bins),
                         "fp64_inst_model": {"per_bin": per_bin, "per_node_interval": BAND_FP64_PER_INTERVAL,
                                             "per_interval_with_a_cut": BAND_FP64_PER_CUT_INTERVAL,
                                             "per_run": BAND_FP64_PER_RUN}}
        assert st[4] == 0, "fstat_fastband_kernel raised its internal-invariant flag"
        out["bands"] = {"n_seg": args.bands, "edge_lattice": args.bands_lattice, "ms_per_step": ms_b, "roofline": band_roofline,
                        "main_kernel_ms": float(np.mean(kms)) if len(kms) else None,
                        "in_band_template_bins": in_band, "in_band_share_of_grid": in_band / (float(P) * ds.n_bins),
                        "in_band_template_bins_per_s": in_band * world / (ms_b * 1e-3),
                        "e2e_ms_per_step": ms_b_e2e, "e2e_in_band_template_bins_per_s": in_band * world / (ms_b_e2e * 1e-3),
                        "kernel": "fstat_fastband_kernel (interpolating kernel with per-thread partition edges)"}
    if args.channels > 1:
        # row f4: the channel sum of Eq. 3 over A, E, T (the combinations with independent noise): the same
        # grid, partitions and particles; channel data = seeded noise with that channel's PSD (timing does not depend on
        # the data); a1-a5 once per channel with the A / E / T response at the nodes, one joint epilogue
        import dataclasses
        names = "AET"[:min(args.channels, 3)]
        plans = []
        for c, name in enumerate(names):
            o = fs.fstat_default_options(force_level=args.force_level, max_segment_bins=args.max_segment_bins,
                                         interp_tol=args.interp_tol, tdi_channel=fs.TDI_CHANNELS[name])
            ds_c = syn.make_dataset(dataclasses.replace(cfg, noise_seed=cfg.noise_seed + 1 + c), None, channel=name)
            plans.append(fs.fstat_plan_create(ds_c.freq, ds_c.dw, ds_c.inv_sn, edges, o))
        # the same set once more with options.no_channel_fusion on plans[0]: one pass per channel instead of the fused pass
        o = fs.fstat_default_options(force_level=args.force_level, max_segment_bins=args.max_segment_bins,
                                     interp_tol=args.interp_tol, tdi_channel=fs.TDI_CHANNELS[names[0]], no_channel_fusion=1)
        ds_c = syn.make_dataset(dataclasses.replace(cfg, noise_seed=cfg.noise_seed + 1), None, channel=names[0])
        plans.append(fs.fstat_plan_create(ds_c.freq, ds_c.dw, ds_c.inv_sn, edges, o))
        del ds_c
        n_c = max(min(args.steps, 10), 1)

        def time_set(pset):
            for _ in range(2):
                fs.fstat_eval_batch_channels(pset, par, stream)
            torch.cuda.synchronize()
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_c)]
            for e0, e1 in evs:
                scratch.fill_(4)
                e0.record(stream)
                fs.fstat_eval_batch_channels(pset, par, stream)
                e1.record(stream)
            torch.cuda.synchronize()
            return float(np.mean([e0.elapsed_time(e1) for e0, e1 in evs]))

        n_ch = len(names)
        ms_c = time_set(plans[:n_ch])
        ms_sep = time_set([plans[n_ch]] + plans[1:n_ch])
        out["channels"] = {"channels": list(names), "ms_per_step": ms_c, "ms_per_step_one_pass_per_channel": ms_sep,
                           "ms_per_step_one_channel_X": ms_step,
                           "channel_template_bins_per_s": float(P) * ds.n_bins * n_ch * world / (ms_c * 1e-3),
                           "kernel": "fstat_fastmulti_kernel (one pass: node model and carrier shared by the channels)",
                           "data": "seeded noise with each channel's own PSD; timing does not depend on the data"}
        for pl in plans:
            fs.fstat_plan_destroy(pl)
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(cfg, ds, n_part, args.cpu_sample)
    fs.fstat_plan_destroy(plan)
    if dist is not None:
        dist.destroy_process_group()
    print(json.dumps(out))
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
