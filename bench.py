#!/usr/bin/env python
"""bench.py -- electron moves/s of the crowd move on B200 (BASELINE.json metric).

A "step" is one full sweep of the whole hot path (propose, spline VGL, ratio/grad, accept,
delayed append, DMMA flush) over one crowd: W x N proposed electron moves (reading A18).
Workload at N=1: BASELINE.json configs[4] (768 electrons, 80^3 fp32 table, delayed rank 32), the
largest configuration; it fits one GPU.  Crowd size via --walkers (default 4096, the largest crowd of the config).

  python bench.py [--gpus N] [--steps K] [--warmup W]        CUDA path, one JSON line
  python bench.py --impl reference ...                        the oracle on the host cores
  python bench.py --crowd-sweep                               extra lines: moves/s vs crowd size / rank
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import numpy as np  # noqa: E402

import qmc_inputs as qi  # noqa: E402

METRIC = "electron_moves_per_sec"
UNIT = "moves/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--cfg", type=int, default=5, help="BASELINE.json config index 1..5")
    ap.add_argument("--walkers", type=int, default=4096, help="crowd size W per GPU (cfg 5: 64..4096)")
    ap.add_argument("--delay-rank", type=int, default=None)
    ap.add_argument("--crowd-sweep", action="store_true", help="also print moves/s vs crowd size and delay rank")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--sub-crowds", type=int, default=None, help="sub-crowds qmc_sweep runs on separate streams (1..4)")
    ap.add_argument("--multi-crowd", action="store_true",
                    help="also time C crowds of W/C walkers, one stream and one host thread each (PAPER.md Alg. 4)")
    ap.add_argument("--drift", action="store_true",
                    help="also print the drift of the carried inverses against a recompute after 1..100 sweeps")
    ap.add_argument("--no-probes", action="store_true", help="skip the step-call / rank-1 kernel probes")
    ap.add_argument("--ref-walkers", type=int, default=None, help="walkers of the oracle sample (default = cores)")
    ap.add_argument("--no-sweep-points", action="store_true",
                    help="skip the compact crowd-size / delay-rank sweep carried inside the JSON line")
    ap.add_argument("--plan-only", action="store_true",
                    help="no GPU work: every rank reports its walker range (gloo), rank 0 prints the plan as JSON")
    return ap.parse_args()


# FP64 DMMA issue ceiling of one B200: 148 SMs x 64 FMA/clk/SM x 2 flop x 1.965 GHz (guide unit counts and max SM clock;
# a bare DMMA.8x8x4 loop measured exactly this in round 1, update.cuh).  The flush runs at the full SM clock (the
# bf16 "sustained" figure of MEASURED_PEAKS.json is power-capped at ~1.3 GHz and does not describe it).
FP64_DMMA_CEILING_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written) or the profiling guide's fallback.
    FP64 tensor: MEASURED_PEAKS.json has no entry.  The denominator of the flush is the larger of the cuBLAS DGEMM
    probe of the same run and the DMMA issue ceiling (filled in by run_cuda); the guide-derived figure (measured
    sustained bf16 GEMM x nominal 45/2250) is kept beside it for reference only -- it is lower than what cuBLAS
    reaches on the same box."""
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        bf16 = float(d.get("bf16_tflops_sustained", d.get("bf16_tflops", 1400.0)))
        return {"hbm_gbs": float(d["hbm_gbs"]), "fp64_bf16_derived_tflops": bf16 * 45.0 / 2250.0,
                "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "fp64_bf16_derived_tflops": 1400.0 * 45.0 / 2250.0,
            "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            self.thread.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        busy = sorted(sm)[len(sm) // 2:]           # upper half = samples under load
        return {"sm_mhz": float(np.median(busy)), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


# ----------------------------------------------------------------------------------------------
# the oracle arm: cpu_baseline and --impl reference (the only places bench.py runs oracle/)
# ----------------------------------------------------------------------------------------------
def oracle_sample(wl, kd, n_walkers, n_sweeps, coefs=None):
    """Times oracle_crowd_sweep (as it stands, OpenMP over walkers) on a bounded sample of the
    workload: the first n_walkers walkers, n_sweeps sweeps.  Returns (moves/s, cores, seconds, accept)."""
    import oracle
    coefs = qi.make_coefs(wl) if coefs is None else coefs
    pos = qi.make_positions(wl, n_walkers)
    osys = oracle.OracleSystem(wl.n_elec, (wl.grid,) * 3, (wl.box,) * 3, coefs, j2_a=wl.j2_a, j2_b=wl.j2_b,
                               tau=wl.tau, seed=wl.seed, delay_rank=kd)
    oc = oracle.OracleCrowd(osys, pos)
    t0 = time.perf_counter()
    acc = oc.sweep(n_sweeps)
    dt = time.perf_counter() - t0
    moves = n_walkers * wl.n_elec * n_sweeps
    oc.close()
    return moves / dt, oracle.num_threads(), dt, acc / moves


def run_reference(args):
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return 0
    wl = qi.WORKLOADS[args.cfg]
    kd = args.delay_rank or wl.delay_rank
    cores = len(os.sched_getaffinity(0))
    nw = args.ref_walkers or cores
    coefs = qi.make_coefs(wl)
    for _ in range(min(args.warmup, 1)):                     # one warm-up sample is enough for a CPU loop
        oracle_sample(wl, kd, nw, 1, coefs)
    t_tot, moves, acc = 0.0, 0, 0.0
    for _ in range(args.steps):
        v, threads, dt, a = oracle_sample(wl, kd, nw, 1, coefs)
        t_tot += dt
        moves += nw * wl.n_elec
        acc = a
    value = moves / t_tot
    sample = f"{nw} walkers x 1 sweep per step of cfg{args.cfg} (N={wl.n_elec}, k={kd}), oracle as it stands"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"cfg{args.cfg}_{wl.n_elec}e_k{kd}", "walkers": nw, "sweeps_per_step": 1},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "accept_fraction": acc, "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------------------------
# algorithmic work per launch
# ----------------------------------------------------------------------------------------------
def algorithmic(wl, W, kd, alpha, el, m_move=None):
    """Bytes / flops ONE launch of each kernel class moves for a crowd of W walkers, with
    acceptance fraction alpha (mean window fill at a flush = alpha*kd, mean fill at a move
    = alpha*(kd-1)/2)."""
    n = M = wl.n
    N = wl.n_elec
    if m_move is None:
        m_move = alpha * (kd - 1) / 2 if kd > 1 else 0.0
    m_flush = alpha * kd
    ratio_b = W * (8 * n + 4 * M * el + 24 * N)
    accept_b = alpha * W * (8 * M * el + (8 * n * m_move + 3 * 8 * n + M * el if kd > 1 else 0))
    row_b = W * (8 * n + 2 * 8 * n * m_move + 3 * M * el + 8 * n + 24 * N)
    out = {
        "spline_vgl": {"bytes": W * (64 * M * el + 5 * M * el), "flops": W * 600 * M},
        "row_propose": {"bytes": row_b},
        "ratio_grad": {"bytes": ratio_b},
        "accept": {"bytes": accept_b},
        "ratio_accept": {"bytes": ratio_b + accept_b},
        # one launch = all kd moves of a delay window in the eager-block form (window.cuh): per move the
        # spline gather, one inverse row and one gradient-cache row; per accepted move the cache / V / Cp
        # rows written and the still-to-be-proposed rows of the block read and rewritten ((kd-1)/2 on average);
        # positions once per window.  Orbitals at r' never leave the SM.
        # "bytes" = the COMPULSORY HBM bytes of that launch: the gather (table >> L2), the first touch of the block's
        # kd rows and the write-back of their final values, the gradient-cache rows read and (accepted) written, the
        # V / Cp rows written for the flush, positions.  The block rows a walker re-reads and re-writes inside its own
        # window (16 n (kd-1)/2 per accepted move) are L2-resident by construction (98 KB per walker x 592 resident
        # walkers) and are counted only in "l2_plus_hbm_bytes".
        "window": {"bytes": W * (kd * (64 * M * el + 3 * M * el + 16 * n) + alpha * kd * (4 * M * el + 16 * n) + 24 * N),
                   "l2_plus_hbm_bytes": W * (kd * (64 * M * el + 8 * n + 3 * M * el)
                                             + alpha * kd * (4 * M * el + 16 * n + 16 * n * (kd - 1) / 2) + 24 * N),
                   "flops": kd * W * 600 * M},
        # kinetic energy: both inverses, the four cache rows of every electron, positions; ~30 fp64 flop per pair term
        # (min image, rsqrt, reciprocal, u', u'') and 8 per (electron, orbital) of the four dots
        "kinetic": {"bytes": W * (16 * n * n + 4 * N * M * el + 24 * N), "flops": W * (30.0 * N * (N - 1) + 8.0 * N * M)},
        # branching probe: every tenth walker replaced by its neighbour; state read once and written once
        "branch": {"bytes": 2 * (W // 10) * (16 * n * n + 4 * N * M * el + 24 * N)},
        "rank1": {"bytes": alpha * W * 16 * n * n, "flops": alpha * W * 4 * n * n},
        "flush": {"bytes": W * 16 * n * n, "flops": W * (4 * n * n * m_flush + 2 * n * m_flush ** 2)},
    }
    return out


# ----------------------------------------------------------------------------------------------
# the CUDA arm
# ----------------------------------------------------------------------------------------------
def make_crowd(wl, W, kd, id0, coefs_dev, dev, inverse_fp32=False):
    import torch
    import paper_2209_14487_b200 as q
    pos = qi.make_positions(wl, id0 + W)[id0:]
    return q.Crowd(coefs_dev, wl.box, torch.from_numpy(np.ascontiguousarray(pos)).to(dev), tau=wl.tau, delay_rank=kd,
                   j2_a=wl.j2_a, j2_b=wl.j2_b, seed=wl.seed, walker_id0=id0, inverse_fp32=inverse_fp32), pos


def time_sweeps(crowd, steps, warmup, sync_all):
    """Device time (CUDA events on the crowd's stream) of `steps` sweeps after `warmup` sweeps."""
    import torch
    for _ in range(warmup):
        crowd.qmc_sweep(1)
    s0 = crowd.stats()
    l0 = crowd.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sync_all()
    e0.record(crowd.stream)
    for _ in range(steps):
        crowd.qmc_sweep(1)
    e1.record(crowd.stream)
    sync_all()
    s1 = crowd.stats()
    return e0.elapsed_time(e1), s1["proposed"] - s0["proposed"], s1["accepted"] - s0["accepted"], crowd.launch_count() - l0


def time_multi_crowd(wl, W, C, kd, coefs_dev, dev, steps=2, warmup=1):
    """C crowds of W/C walkers (global walker ids), each on its own stream, each driven by its own host thread
    (Alg. 4).  Device time: a start event on the current stream that every crowd's stream
    waits for, an end event that waits for every crowd's last launch.  Returns (ms, proposed, accepted)."""
    import threading
    import torch
    wc = W // C
    streams = [torch.cuda.Stream(device=dev) for _ in range(C)]
    crowds = []
    for c in range(C):
        pos = qi.make_positions(wl, (c + 1) * wc)[c * wc:]
        import paper_2209_14487_b200 as q
        crowds.append(q.Crowd(coefs_dev, wl.box, torch.from_numpy(np.ascontiguousarray(pos)).to(dev), tau=wl.tau,
                              delay_rank=kd, j2_a=wl.j2_a, j2_b=wl.j2_b, seed=wl.seed, walker_id0=c * wc,
                              stream=streams[c]))

    def drive(n):
        def one(cr):
            torch.cuda.set_device(dev)
            for _ in range(n):
                cr.qmc_sweep(1)
        th = [threading.Thread(target=one, args=(cr,)) for cr in crowds]
        for t in th:
            t.start()
        for t in th:
            t.join()

    drive(warmup)
    torch.cuda.synchronize()
    s0 = [cr.stats() for cr in crowds]
    main = torch.cuda.current_stream(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(main)
    for st in streams:
        st.wait_event(e0)
    drive(steps)
    for st in streams:
        main.wait_stream(st)
    e1.record(main)
    torch.cuda.synchronize()
    s1 = [cr.stats() for cr in crowds]
    prop = sum(b["proposed"] - a["proposed"] for a, b in zip(s0, s1))
    acc = sum(b["accepted"] - a["accepted"] for a, b in zip(s0, s1))
    for cr in crowds:
        cr.close()
    del crowds
    torch.cuda.empty_cache()
    return e0.elapsed_time(e1), prop, acc


def drift_study(wl, coefs_dev, dev, W=128, ranks=(1, 32, 64), marks=(1, 5, 10, 20, 50, 100), fp32_round=False):
    """Round-off drift of the carried inverses: after S free-running sweeps, the largest and
    median norm-wise difference between a walker's carried inverse and the one recomputed at the same positions."""
    import torch
    import paper_2209_14487_b200 as q
    pos = torch.from_numpy(np.ascontiguousarray(qi.make_positions(wl, W))).to(dev)
    for kd in ranks:
        mk = lambda: q.Crowd(coefs_dev, wl.box, pos, tau=wl.tau, delay_rank=kd, j2_a=wl.j2_a, j2_b=wl.j2_b, seed=wl.seed)
        c, f = mk(), mk()
        done = 0
        for S in marks:
            if fp32_round:   # a lower bound on what an fp32-stored inverse would do: round after every sweep
                for _ in range(S - done):
                    c.qmc_sweep(1)
                    for spin in (0, 1):
                        c.set_inverse(spin, c.inverse(spin).float().double())
            else:
                c.qmc_sweep(S - done)
            done = S
            f.set_positions(c.positions())
            worst, med = 0.0, 0.0
            for spin in (0, 1):
                B, F = c.inverse(spin), f.inverse(spin)
                rel = (B - F).abs().amax(dim=(1, 2)) / F.abs().amax(dim=(1, 2))
                worst, med = max(worst, float(rel.max())), max(med, float(rel.median()))
            print(json.dumps({"drift": True, "fp32_rounded_every_sweep": fp32_round, "walkers": W, "delay_rank": kd,
                              "sweeps": S, "rel_diff_max": worst, "rel_diff_median": med}), flush=True)
        c.close()
        f.close()


def csrc_digest():
    """sha256 (first 16 hex digits) over the CUDA sources and the C header: names the kernels a capture was made with
    (the GPU box has no .git, so a commit id cannot be read there)."""
    import hashlib
    h = hashlib.sha256()
    for f in sorted((ROOT / "paper_2209_14487_b200" / "csrc").glob("*.cu*")) + [ROOT / "include" / "qmc_crowd.h"]:
        h.update(f.name.encode())
        h.update(f.read_bytes())
    return h.hexdigest()[:16]


def ncu_traffic(cfg, W, kd):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture
    (profiles/dram_traffic.csv: cfg,walkers,delay_rank,kernel,bytes,csrc_digest), for the configuration timed here.
    Returns ({kernel: bytes}, source): an entry is used only if it was captured with the kernel sources that are being
    timed now (same csrc_digest); otherwise the field is null -- a stale capture is not a measurement of this run."""
    out, src = {}, None
    f = ROOT / "profiles" / "dram_traffic.csv"
    if f.exists():
        now = csrc_digest()
        for ln in f.read_text().splitlines():
            c = [x.strip() for x in ln.split(",")]
            if len(c) == 6 and c[0].isdigit() and (int(c[0]), int(c[1]), int(c[2])) == (cfg, W, kd):
                if c[5] == now:
                    out[c[3]] = float(c[4])
                    src = f"profiles/dram_traffic.csv @ csrc {now}"
                elif src is None:
                    src = f"stale: profiles/dram_traffic.csv was captured at csrc {c[5]}, timed sources are {now}"
    return out, src


def fp64_probe():
    """cuBLAS DGEMM 8192^3 on this GPU: context for the flush roofline (a probe, not product code)."""
    import torch
    a = torch.randn(8192, 8192, dtype=torch.float64, device="cuda")
    b = torch.randn(8192, 8192, dtype=torch.float64, device="cuda")
    torch.matmul(a, b)
    best = 1e9
    for _ in range(3):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); torch.matmul(a, b); e1.record(); torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    return 2 * 8192 ** 3 / (best * 1e-3) / 1e12


def run_cuda(args):
    import torch
    import paper_2209_14487_b200 as q
    from paper_2209_14487_b200 import dist as qd

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    rank, local_rank, world = qd.env_world()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    qd.init("nccl")
    wl = qi.WORKLOADS[args.cfg]
    kd = args.delay_rank or wl.delay_rank
    W = args.walkers
    el = 4 if wl.coef_dtype == "f32" else 8
    id0, _ = qd.walker_slice(rank, world, W)
    coefs_np = qi.make_coefs(wl)
    coefs_dev = torch.from_numpy(coefs_np).to(dev)

    def sync_all():
        torch.cuda.synchronize()
        qd.barrier()
        torch.cuda.synchronize()

    t0 = time.perf_counter()
    crowd, pos = make_crowd(wl, W, kd, id0, coefs_dev, dev)
    torch.cuda.synchronize()
    create_s = time.perf_counter() - t0
    if args.sub_crowds:
        crowd.set_option(q.QMC_OPT_SUBCROWDS, args.sub_crowds)

    with ClockSampler(local_rank) as clk:
        ms, proposed, accepted, launches = time_sweeps(crowd, args.steps, max(args.warmup, 0), sync_all)
    ms, (proposed, accepted, launches) = qd.reduce_job(ms, [proposed, accepted, launches], device=dev)
    value = proposed / (ms * 1e-3)
    alpha = accepted / max(proposed, 1)

    # per-kernel device time: one more sweep with an event pair around every launch
    crowd.set_option(q.QMC_OPT_PROFILE, 1)
    crowd.qmc_sweep(1)
    prof = crowd.profile()
    step_prof = {}
    if not args.no_probes and rank == 0:
        # the same kernels one call at a time (C-ABI step calls), 8 moves: stand-alone spline / row / ratio / accept
        for k in range(min(8, kd, wl.n)):
            crowd.qmc_spo_vgl(k)
            crowd.qmc_ratio_grad(k)
            crowd.qmc_accept_reject(k)
        crowd.qmc_flush_delayed()
        crowd.qmc_kinetic_energy()
        crowd.qmc_kinetic_energy()
        src = torch.arange(W, dtype=torch.int32, device=dev)
        src[9::10] -= 1
        crowd.qmc_crowd_branch(src)
        crowd.qmc_crowd_branch(src)
        step_prof = {k2: v for k2, v in crowd.profile().items() if v[1] and k2 != "flush"}
    crowd.set_option(q.QMC_OPT_PROFILE, 0)
    tot_ms = sum(v[0] for v in prof.values()) or 1.0
    alg = algorithmic(wl, W, kd, alpha, el)
    pk = peaks()
    kernels = {}
    for name, (kms, cnt) in prof.items():
        if cnt == 0:
            continue
        avg = kms / cnt
        ent = {"launches_per_sweep": cnt, "avg_us": 1e3 * avg, "share": kms / tot_ms,
               "gbs": alg[name]["bytes"] / (avg * 1e-3) / 1e9}
        ent["hbm_frac"] = ent["gbs"] / pk["hbm_gbs"]
        if "flops" in alg[name]:
            ent["tflops"] = alg[name]["flops"] / (avg * 1e-3) / 1e12
        kernels[name] = ent
    for name, (kms, cnt) in step_prof.items():
        if name in kernels or name not in alg:
            continue
        avg = kms / cnt
        a_step = algorithmic(wl, W, kd, alpha, el, m_move=alpha * 3.5)[name]     # window fill 0..7 in the probe
        ent = {"launches": cnt, "avg_us": 1e3 * avg, "share": 0.0, "gbs": a_step["bytes"] / (avg * 1e-3) / 1e9,
               "probe": "step calls, 8 moves"}
        ent["hbm_frac"] = ent["gbs"] / pk["hbm_gbs"]
        kernels[name] = ent
    dom = max(kernels, key=lambda k: kernels[k]["share"])
    traffic, traffic_source = ncu_traffic(args.cfg, W, kd)

    def with_traffic(ent, name):
        """traffic = ncu dram bytes per launch (null unless captured with the sources timed now); dram_frac = that
        traffic over the event-timed duration of this run over the measured copy rate."""
        t = traffic.get(name)
        ent["traffic"] = t
        ent["traffic_source"] = traffic_source
        if t and ent.get("avg_us"):
            ent["dram_frac"] = t / (ent["avg_us"] * 1e-6) / 1e9 / pk["hbm_gbs"]
        return ent

    roofline = with_traffic({"kernel": dom, "bound": "hbm", "achieved": kernels[dom]["gbs"], "peak": pk["hbm_gbs"],
                             "unit": "GB/s", "frac": kernels[dom]["gbs"] / pk["hbm_gbs"],
                             "peak_source": pk["source"] + ", of measured", "share_of_step": kernels[dom]["share"],
                             "avg_us": kernels[dom]["avg_us"], "algorithmic_bytes_per_launch": alg[dom]["bytes"],
                             "bytes_counted": "compulsory HBM bytes (DESIGN.md section 6)"}, dom)
    if "l2_plus_hbm_bytes" in alg[dom]:
        # the round-1 figure: every byte the kernel requests beyond L1, including the block rows that stay in L2
        roofline["l2_plus_hbm_bytes"] = alg[dom]["l2_plus_hbm_bytes"]
        roofline["l2_plus_hbm_gbs"] = alg[dom]["l2_plus_hbm_bytes"] / (kernels[dom]["avg_us"] * 1e-6) / 1e9
    probe, probe_err = None, None
    if rank == 0:
        try:
            probe = fp64_probe()
        except Exception as e:  # probe only
            probe_err = str(e)[:80]
    extra_rooflines = {}
    if "flush" in kernels:
        n = wl.n
        useful = kernels["flush"]["tflops"]
        kdp = 8
        while kdp < kd:
            kdp *= 2
        # executed DMMA work: GEMM 1 pads the window to whole 8-move blocks (~ kdp); GEMM 2 of the 32-row strip kernel
        # (fp64 inverses, n % 32 == 0, kdp >= 16) skips the k-steps of padding in units of four moves (~ m + 1.5 on average)
        k2 = kdp
        if n % 32 == 0 and kdp >= 16:   # the timed crowd carries fp64 inverses
            acc_moves = (alg["flush"]["flops"] / W) / (4.0 * n * n)      # ~ accepted moves per flush (finalize term small)
            k2 = min(float(kdp), acc_moves + 1.5)
        executed = useful * (2 * n * n * kdp + 2 * n * n * k2 + 2 * n * kdp * kdp) / max(alg["flush"]["flops"] / W, 1.0)
        # denominator: whichever is larger of what cuBLAS DGEMM reaches in this run and the DMMA issue ceiling
        peak64 = max(probe or 0.0, FP64_DMMA_CEILING_TFLOPS)
        extra_rooflines["flush"] = with_traffic({
            "kernel": "flush (finalize + DMMA strip)", "bound": "tensor", "achieved": useful, "peak": peak64,
            "unit": "TFLOP/s", "frac": useful / peak64,
            "peak_source": "max(cuBLAS DGEMM 8192^3 probe of this run, DMMA issue ceiling 148 SM x 64 FMA/clk x 1.965 GHz)",
            "share_of_step": kernels["flush"]["share"], "avg_us": kernels["flush"]["avg_us"],
            "executed_tflops_with_padding": executed, "executed_frac": executed / peak64,
            "frac_of_dgemm_probe": (useful / probe) if probe else None,
            "frac_of_dmma_issue_ceiling": useful / FP64_DMMA_CEILING_TFLOPS,
            "frac_of_bf16_derived_peak": useful / pk["fp64_bf16_derived_tflops"],
            "bf16_derived_peak_tflops": pk["fp64_bf16_derived_tflops"],
            "hbm_frac": kernels["flush"]["hbm_frac"]}, "flush")
    if "kinetic" in kernels:
        # plain fp64 ALU work (J2 pair terms): peak = 148 SMs x 64 FMA/clk x 2 x max SM clock
        k_ = kernels["kinetic"]
        tf = alg["kinetic"]["flops"] / (k_["avg_us"] * 1e-6) / 1e12
        alu_peak = FP64_DMMA_CEILING_TFLOPS
        extra_rooflines["kinetic"] = {"kernel": "kinetic_kernel (qmc_kinetic_energy)", "bound": "alu", "achieved": tf,
                                      "peak": alu_peak, "unit": "TFLOP/s", "frac": tf / alu_peak, "traffic": None,
                                      "avg_us": k_["avg_us"], "hbm_frac": k_["hbm_frac"]}
    for name in ("spline_vgl", "rank1", "branch"):
        if name in kernels:
            extra_rooflines[name] = with_traffic({"kernel": name, "bound": "hbm", "achieved": kernels[name]["gbs"],
                                                  "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": kernels[name]["hbm_frac"],
                                                  "avg_us": kernels[name]["avg_us"],
                                                  "share_of_step": kernels[name]["share"]}, name)

    if dom == "flush" and "flush" in extra_rooflines:
        # the DMMA flush has the largest share of the step: it is the dominant kernel, bound by the FP64 tensor pipe;
        # the window kernel's HBM roofline moves to rooflines["window"]
        extra_rooflines["window"] = with_traffic({
            "kernel": "window", "bound": "hbm", "achieved": kernels["window"]["gbs"], "peak": pk["hbm_gbs"],
            "unit": "GB/s", "frac": kernels["window"]["gbs"] / pk["hbm_gbs"], "peak_source": pk["source"] + ", of measured",
            "share_of_step": kernels["window"]["share"], "avg_us": kernels["window"]["avg_us"],
            "algorithmic_bytes_per_launch": alg["window"]["bytes"], "bytes_counted": "compulsory HBM bytes (DESIGN.md section 6)",
            "l2_plus_hbm_bytes": alg["window"]["l2_plus_hbm_bytes"]}, "window") if "window" in kernels else None
        roofline = dict(extra_rooflines["flush"])

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / max(args.steps, 1), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"cfg{args.cfg}_{wl.n_elec}e_k{kd}", "walkers_per_gpu": W, "n_elec": wl.n_elec,
                   "grid": wl.grid, "table_dtype": wl.coef_dtype, "delay_rank": kd, "sweeps_per_step": 1,
                   "parallelism": f"walkers sharded over {world} GPU(s), no collective",
                   "l2": "working set (table + inverses + caches) is far larger than the 126 MB L2; no flush needed"},
        "accept_fraction": alpha, "gpu_launches": launches, "create_s": create_s,
        "clocks": clk.summary(), "roofline": roofline, "rooflines": extra_rooflines, "kernels": kernels,
    }
    line["fp64_dgemm_probe_tflops"] = probe
    line["fp64_dmma_issue_ceiling_tflops"] = FP64_DMMA_CEILING_TFLOPS
    if probe_err:
        line["fp64_probe_error"] = probe_err

    # end to end through the host-buffer call: H2D positions, rebuild, sweep, D2H positions
    if not args.no_e2e:
        host = torch.from_numpy(np.ascontiguousarray(pos)).pin_memory()
        crowd.qmc_sweep_host(host, 1)
        sync_all()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            crowd.qmc_sweep_host(host, 1)
        torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3
        e2e_ms, (moves,) = qd.reduce_job(e2e_ms, [W * wl.n_elec * args.steps], device=dev)
        nbytes = W * wl.n_elec * 24
        line["e2e"] = {"value": moves / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": nbytes,
                       "d2h_bytes_per_step": nbytes + 8,
                       "what": "qmc_sweep_host: pinned positions H2D, Slater rebuild + inversion, 1 sweep, positions D2H"}
    crowd.close()
    del crowd
    torch.cuda.empty_cache()

    if rank == 0 and world == 1 and not args.no_probes and kd > 1:
        # Sherman-Morrison path (delay_rank = 1) on the same crowd size: 16 step moves, rank-1 kernel roofline
        c1, _ = make_crowd(wl, W, 1, 0, coefs_dev, dev)
        c1.set_option(q.QMC_OPT_PROFILE, 1)
        a0 = c1.stats()["accepted"]
        for k in range(16):
            c1.qmc_spo_vgl(k)
            c1.qmc_ratio_grad(k)
            c1.qmc_accept_reject(k)
        p1 = c1.profile()
        a1 = (c1.stats()["accepted"] - a0) / (16.0 * W)
        kms, cnt = p1["rank1"]
        if cnt:
            avg = kms / cnt
            byts = a1 * W * 16 * wl.n * wl.n
            ent = {"kernel": "rank1", "bound": "hbm", "achieved": byts / (avg * 1e-3) / 1e9, "peak": pk["hbm_gbs"],
                   "unit": "GB/s", "avg_us": 1e3 * avg, "accept_fraction": a1,
                   "probe": "delay_rank 1 crowd, 16 step moves"}
            ent["frac"] = ent["achieved"] / pk["hbm_gbs"]
            line["rooflines"]["rank1"] = with_traffic(ent, "rank1")
        c1.close()
        del c1
        torch.cuda.empty_cache()

    if rank == 0 and world == 1 and args.cfg == 5 and not args.no_sweep_points:
        # The metric is "electron moves/sec per B200 VS CROWD SIZE" (BASELINE.json; the analogue of the paper's Fig. 5,
        # P:184 / P:190): a compact sweep inside the parsed line -- crowd sizes at the configured rank, ranks at the
        # largest crowd; fresh crowd each, 1 warm-up + 2 timed sweeps, acceptance alongside.
        pts = [(w2, kd) for w2 in (64, 256, 1024) if w2 != W] + [(W, k2) for k2 in (1, 16, 64) if k2 != kd]
        sweep_pts = [{"walkers": W, "delay_rank": kd, "value": value, "accept_fraction": alpha,
                      "ms_per_sweep": ms / max(args.steps, 1)}]
        for W2, k2 in pts:
            c2, _ = make_crowd(wl, W2, k2, 0, coefs_dev, dev)
            ms2, prop2, acc2, _ = time_sweeps(c2, 2, 1, torch.cuda.synchronize)
            sweep_pts.append({"walkers": W2, "delay_rank": k2, "value": prop2 / (ms2 * 1e-3),
                              "accept_fraction": acc2 / prop2, "ms_per_sweep": ms2 / 2})
            c2.close()
            del c2
            torch.cuda.empty_cache()
        line["crowd_sweep"] = sorted(sweep_pts, key=lambda r: (r["delay_rank"], r["walkers"]))

    if rank == 0 and world == 1 and not args.no_sweep_points and kd <= 32:
        # Mixed precision (R6): the same workload with the carried inverses STORED in
        # fp32 (all arithmetic fp64).  An extra number, never the headline: BASELINE.json's configs say fp64 inverses.
        c3, _ = make_crowd(wl, W, kd, 0, coefs_dev, dev, inverse_fp32=True)
        ms3, prop3, acc3, _ = time_sweeps(c3, 2, 1, torch.cuda.synchronize)
        c3.set_option(q.QMC_OPT_PROFILE, 1)
        c3.qmc_sweep(1)
        p3 = c3.profile()
        line["mixed_precision"] = {"dtype": "f32inv", "what": "inverses stored in fp32, fp64 arithmetic (DESIGN.md R6)",
                                   "value": prop3 / (ms3 * 1e-3), "unit": UNIT, "ms_per_sweep": ms3 / 2,
                                   "accept_fraction": acc3 / prop3,
                                   "kernels_avg_us": {k2: 1e3 * v[0] / v[1] for k2, v in p3.items() if v[1]}}
        c3.close()
        del c3
        torch.cuda.empty_cache()

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = len(os.sched_getaffinity(0))
        nw = (args.ref_walkers or cores) * 2
        # size the sample for roughly 15 s of CPU work: one timed sweep first, then as many as fit
        v1, threads, dt1, _ = oracle_sample(wl, kd, nw, 1, coefs_np)
        n_sw = int(min(max(round(15.0 / max(dt1, 1e-3)), 2), 40))
        v, threads, dt, a = oracle_sample(wl, kd, nw, n_sw, coefs_np)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                                "sample": f"{nw} walkers x {n_sw} sweeps of the same workload ({dt:.1f} s wall)",
                                "accept_fraction": a}
    if rank == 0:
        print(json.dumps(line), flush=True)

    if args.crowd_sweep and world == 1:
        sizes = qi.CFG5_CROWD_SIZES if args.cfg == 5 else (wl.n_walkers // 4, wl.n_walkers // 2, wl.n_walkers)
        ranks = qi.CFG5_DELAY_RANKS if args.cfg == 5 else (kd,)
        for k2 in ranks:
            for W2 in sizes:
                c2, _ = make_crowd(wl, W2, k2, 0, coefs_dev, dev)
                ms2, prop2, acc2, _ = time_sweeps(c2, 2, 1, torch.cuda.synchronize)
                print(json.dumps({"crowd_sweep": True, "walkers": W2, "delay_rank": k2, "value": prop2 / (ms2 * 1e-3),
                                  "unit": UNIT, "accept_fraction": acc2 / prop2, "ms_per_sweep": ms2 / 2}), flush=True)
                c2.close()
                del c2
                torch.cuda.empty_cache()
    if args.drift and world == 1:
        drift_study(wl, coefs_dev, dev)
        drift_study(wl, coefs_dev, dev, ranks=(32,), marks=(1, 2, 5, 10, 20), fp32_round=True)
    if args.multi_crowd and world == 1:
        # S:8(f) item 1: does splitting a crowd of W into C crowds on C streams / host threads pay at small W?
        for W2 in (256, 512, 1024, 4096):
            for C in (1, 2, 4, 8):
                ms2, prop2, acc2 = time_multi_crowd(wl, W2, C, kd, coefs_dev, dev)
                print(json.dumps({"multi_crowd": True, "walkers": W2, "crowds": C, "delay_rank": kd,
                                  "value": prop2 / (ms2 * 1e-3), "unit": UNIT, "accept_fraction": acc2 / prop2,
                                  "ms_per_sweep": ms2 / 2}), flush=True)
    return 0


def run_plan_only(args):
    """No GPU work: every rank derives its walker range exactly as run_cuda does and the ranks agree on the plan over
    gloo; rank 0 prints it.  Lets `--gpus N` (launch, rendezvous, sharding) be tested on a CPU box."""
    import torch
    from paper_2209_14487_b200 import dist as qd
    rank, local_rank, world = qd.env_world()
    d = qd.init("gloo")
    id0, cnt = qd.walker_slice(rank, world, args.walkers)
    mine = torch.tensor([rank, os.getpid(), id0, cnt], dtype=torch.int64)
    rows = [mine]
    if world > 1:
        rows = [torch.zeros(4, dtype=torch.int64) for _ in range(world)]
        d.all_gather(rows, mine)
    if rank == 0:
        print(json.dumps({"plan_only": True, "n_gpus": world, "scaling": "weak",
                          "ranks": [{"rank": int(r[0]), "pid": int(r[1]), "walker_id0": int(r[2]),
                                     "walkers": int(r[3])} for r in rows]}), flush=True)
    if world > 1:
        d.barrier()
        d.destroy_process_group()
    return 0


def relaunch_ranks(args):
    """`python bench.py --gpus N` outside torchrun: start the N ranks here (one process per GPU, rendezvous on
    127.0.0.1, a free port), exactly the command the driver uses for N > 1."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(Path(__file__).resolve())] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return relaunch_ranks(args)
    if args.plan_only:
        return run_plan_only(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
