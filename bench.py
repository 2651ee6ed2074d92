#!/usr/bin/env python
"""bench.py -- LSQR iterations/s of the AVU-GSR hot path on B200 (BASELINE.json metric).

A "step" is one LSQR iteration (aprod1 + aprod2 + norms + vector updates + stop tests, SURVEY 8(a)
rows a2-a11) over one synthetic Gaia-shaped system resident in HBM.  Default workload: BASELINE
configs[2] "medium" (1M stars x 200 obs = 200M rows, 46.4 GB), the config the metric's 70 %-of-HBM
target is quoted on.  Inputs are seeded and synthetic (paper_2308_00778_b200.synth); the paper's
Gaia datasets are proprietary.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload medium|small|tiny|skewed]
  python bench.py --impl reference ...     # the CPU oracle, as it stands, on a bounded sample

N > 1: the path does not shard in this build (north_star: one GPU, no collectives), so N ranks run
N independent replicas ("replicas only") and `value` is their aggregate.
Prints ONE JSON line on rank 0.
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

METRIC = "lsqr_iterations_per_s"
UNIT = "it/s"
ROW_BYTES_APROD1 = 248      # 192 values + 40 indices + 8 read y + 8 write y
ROW_BYTES_APROD2 = 240      # 192 values + 40 indices + 8 read y


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="medium")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel-reps", type=int, default=20)
    return ap.parse_args()


def workload_cfg(name):
    from paper_2308_00778_b200 import synth
    return {"tiny": synth.tiny, "small": synth.small, "medium": synth.medium, "skewed": synth.skewed,
            "large": synth.large}[name]()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.stop = index, [], threading.Event()
        self.t = threading.Thread(target=self.run, daemon=True)

    def run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        sm = sorted(int(r[0]) for r in self.rows if len(r) >= 6 and r[0].isdigit())
        mx = [int(r[1]) for r in self.rows if len(r) >= 6 and r[1].isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) >= 6 and r[2 + k] == "Active" for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def build_on_device(cfg, G, dev, torch, synth):
    """Generate the system chunk by chunk on the GPU and hand each chunk to gsr_upload_rows
    (device pointers).  b = A x_true + noise is formed by the library's own aprod1."""
    rp = synth.star_rowptr(cfg, dev)
    m = int(rp[-1])
    step = 20_000 if cfg.obs_per_star > 0 else 50_000
    noise = torch.zeros(m + cfg.n_con, dtype=torch.float64, device=dev)   # constraint rows: b_c = A_c x_true
    for s0 in range(0, cfg.n_stars, step):
        s1 = min(s0 + step, cfg.n_stars)
        part = synth.generate_rows(cfg, s0, s1, dev, rp)
        r0, nr = part["row0"], part["values"].shape[0]
        noise[r0:r0 + nr] = part["noise"]
        G.gsr_upload_rows(r0, nr, part["values"].contiguous(), part["matrixIndexAstro"].contiguous(),
                          part["matrixIndexAtt"].contiguous(), part["instrCol"].contiguous(),
                          part["noise"].contiguous())
        del part
    G.gsr_upload_finish(noise[m:].contiguous() if cfg.n_con else None)
    if cfg.n_con:
        G.gsr_upload_constraints(*synth.constraints(cfg, dev))
    xt = synth.x_true(cfg, dev)
    G.gsr_aprod1(xt, noise)             # noise <- noise + A x_true
    G.gsr_set_b(noise)
    del noise, xt
    torch.cuda.empty_cache()
    return m


def oracle_sample_run(cfg, steps, warmup):
    """The CPU oracle, as it stands (single thread, plain C), on a bounded sample of the workload:
    the first `ns` stars with the full attitude / instrument column ranges.  Returns it/s scaled
    linearly in rows to the full workload, plus a description of the sample."""
    import dataclasses
    import numpy as np
    import oracle
    from paper_2308_00778_b200 import synth
    full_rows = int(synth.star_rowptr(cfg)[-1])
    target_rows = 3_000_000
    ns = max(1, min(cfg.n_stars, int(cfg.n_stars * target_rows / max(full_rows, 1))))
    sub = dataclasses.replace(cfg, name=cfg.name + "_sample", n_stars=ns, n_con=0, con_nnz=0)
    d = {k: v.numpy() for k, v in synth.generate(sub).items()}
    S = oracle.OracleSystem(sub.n_stars, sub.n_dof_att, sub.n_instr, d["values"], d["matrixIndexAstro"],
                            d["matrixIndexAtt"], d["instrCol"])
    b = S.aprod1(d["x_true"], d["noise"])
    S.precondition()
    if warmup > 0:
        S.lsqr(b, warmup, 0.0, 0.0)
    t0 = time.perf_counter()
    r = S.lsqr(b, steps, 0.0, 0.0)
    dt = time.perf_counter() - t0
    assert r.itn == steps
    its_sample = steps / dt
    scaled = its_sample * S.m / full_rows
    sample = (f"oracle LSQR (gcc -O2, 1 thread), {steps} iterations on the first {ns} stars = {S.m} rows of "
              f"'{cfg.name}' ({full_rows} rows); it/s scaled by rows {S.m}/{full_rows}")
    return scaled, dt / steps, sample, 1


def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = workload_cfg(args.workload)
    steps = max(1, min(args.steps, 10))
    val, s_per_step, sample, cores = oracle_sample_run(cfg, steps, min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": 1e3 / val,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": args.workload, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def aggregate_replicas(loop_ms_rank, steps, world, dev, torch, dist):
    """Replicas only: every rank runs the same workload on its own GPU.  The job's time is the
    MAX of the ranks' device times (one all-reduce of a scalar, outside the timed region); the job's
    throughput is all ranks' iterations over that time."""
    t = torch.tensor([loop_ms_rank], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    return ms, world * steps / (ms * 1e-3)


def main_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2308_00778_b200 import gsr, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = workload_cfg(args.workload)
    rp = synth.star_rowptr(cfg)
    m = int(rp[-1])
    G = gsr.Gsr(m, cfg.n_stars, cfg.n_dof_att, cfg.n_instr, cfg.n_con, cfg.n_con * cfg.con_nnz, device=local)
    t_gen = time.perf_counter()
    build_on_device(cfg, G, dev, torch, synth)
    G.gsr_precondition()
    t_gen = time.perf_counter() - t_gen

    # ---- device-resident timing: W warm-up iterations, then exactly K timed iterations
    G.gsr_lsqr(max(args.warmup, 3), 0.0, 0.0, want_se=False)
    barrier()
    with ClockSampler(local) as clk:
        barrier()
        r = G.gsr_lsqr(args.steps, 0.0, 0.0)
        barrier()
    assert r.itn == args.steps and r.istop == 7, (r.itn, r.istop)
    loop_ms, value = aggregate_replicas(r.loop_ms, args.steps, world, dev, torch, dist)
    xt = synth.x_true(cfg, dev)
    x_err = float(torch.linalg.norm(r.x - xt) / torch.linalg.norm(xt))
    del xt

    # ---- per-kernel roofline: the two products timed alone (CUDA events on the library's stream)
    peak, peak_src = peaks()
    ms1 = G.gsr_time_aprod(11, args.kernel_reps)
    ms2 = G.gsr_time_aprod(12, args.kernel_reps)
    try:
        ms2a = G.gsr_time_aprod(13, args.kernel_reps)      # time-ordered attitude kernel, if in use
    except gsr.GsrError:
        ms2a = None
    try:
        msf = G.gsr_time_aprod(21, args.kernel_reps)       # fused pass of gsr_lsqr (aprod1 + main scatter of aprod2)
    except gsr.GsrError:
        msf = None
    ms1g = G.gsr_time_aprod(1, args.kernel_reps)
    ms2g = G.gsr_time_aprod(2, args.kernel_reps)
    gb1 = ROW_BYTES_APROD1 * m / 1e9
    gb2 = (ROW_BYTES_APROD2 * m + 8 * G.n) / 1e9
    # per-kernel algorithmic bytes: with the attitude section on its own
    # time-ordered copy the main aprod2 kernel needs 96 B of non-attitude values + 32 B indices + 8 B y
    # per row, the attitude kernel 96 B values + 4 B start + 4 B permutation + 8 B y
    gb2_main = (136 * m + 8 * G.n) / 1e9 if ms2a is not None else gb2
    k = {"k_aprod1": {"ms": ms1, "alg_gb": gb1, "gbs": gb1 / (ms1 * 1e-3)},
         "k_aprod2": {"ms": ms2, "alg_gb": gb2_main, "gbs": gb2_main / (ms2 * 1e-3)},
         "aprod1_group_ms": ms1g, "aprod2_group_ms": ms2g}
    if ms2a is not None:
        gb2a = 112 * m / 1e9
        k["k_aprod2_att"] = {"ms": ms2a, "alg_gb": gb2a, "gbs": gb2a / (ms2a * 1e-3)}
    in_step = ["k_aprod1", "k_aprod2"] + (["k_aprod2_att"] if ms2a is not None else [])
    if msf is not None:
        # the timed step runs the fused pass: the work of aprod1 (248 B/row) and of aprod2's main kernel (136 B/row)
        # on one read of A, then k_aprod2_att; the standalone products above are what gsr_aprod1/2 expose
        gbf = gb1 + gb2_main
        k["k_aprod2_fused"] = {"ms": msf, "alg_gb": gbf, "gbs": gbf / (msf * 1e-3)}
        in_step = ["k_aprod2_fused", "k_aprod2_att"]
    dom = max(in_step, key=lambda n: k[n]["ms"])
    traffic = None      # ncu-measured DRAM bytes per launch of the dominant kernel (profiles/r01_traffic.csv)
    tpath = os.path.join(ROOT, "profiles", "r01_traffic.csv")
    if os.path.exists(tpath):
        for ln in open(tpath).read().splitlines()[1:]:
            w, kn, bts = ln.split(",")
            if w == args.workload and kn == dom:
                traffic = float(bts) / 1e9
    roofline = {"bound": "hbm", "kernel": dom, "achieved": k[dom]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": k[dom]["gbs"] / peak, "traffic": traffic, "traffic_unit": "GB per launch (ncu dram read+write)",
                "peak_source": peak_src,
                "aprod1_plus_aprod2_gbs": (gb1 + gb2) / ((ms1g + ms2g) * 1e-3),
                "aprod1_plus_aprod2_frac": (gb1 + gb2) / ((ms1g + ms2g) * 1e-3) / peak,
                "iteration_alg_gb": (gb1 + gb2), "iteration_gbs": (gb1 + gb2) / (loop_ms / args.steps * 1e-3),
                "iteration_frac": (gb1 + gb2) / (loop_ms / args.steps * 1e-3) / peak,
                "iteration_form": "fused (A's row layout streamed once)" if msf is not None else "two products",
                "kernels": k}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": loop_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "rows": m, "cols": G.n, "nnz_per_row": 24,
                       "matrix_gb": 232 * m / 1e9, "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": "inputs larger than L2" if 232 * m > 2.5e8 else "L2-resident (launch-bound config)",
                       "x_rel_err_vs_planted": x_err, "setup_s": t_gen},
            "clocks": clk.summary(), "gpu_launches": int(r.kernel_launches), "roofline": roofline}

    # ---- end to end through the C ABI with HOST buffers: upload + precondition + K iterations + results
    if not args.no_e2e and rank == 0:
        line["e2e"] = e2e_run(args, cfg, G, dev, torch, synth, gsr)
    if not args.no_cpu_baseline and rank == 0 and world == 1:
        val, _, sample, cores = oracle_sample_run(cfg, 10, 1)
        line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    G.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def e2e_run(args, cfg, G, dev, torch, synth, gsr):
    """Same metric through the public calls with host buffers: gsr_upload from pinned host memory,
    gsr_precondition, gsr_lsqr(K) writing x and se to host memory, all inside the timed region."""
    import psutil
    m = G.n_obs
    need = 232 * m + 8 * m
    avail = psutil.virtual_memory().available
    if need * 1.15 > avail:
        return {"value": None, "unit": UNIT, "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                "note": f"host RAM {avail / 1e9:.0f} GB cannot hold the {need / 1e9:.0f} GB workload"}
    # current (preconditioned) device state is not what a user uploads: regenerate the raw arrays on
    # the host side by pulling a fresh device generation chunk by chunk into pinned buffers
    hv = torch.empty((m, 24), dtype=torch.float64, pin_memory=True)
    hia = torch.empty(m, dtype=torch.int64, pin_memory=True)
    hit = torch.empty(m, dtype=torch.int64, pin_memory=True)
    hic = torch.empty((m, 6), dtype=torch.int32, pin_memory=True)
    hb = torch.empty(m, dtype=torch.float64, pin_memory=True)
    rp = synth.star_rowptr(cfg, dev)
    step = 20_000 if cfg.obs_per_star > 0 else 50_000
    G2 = G  # reuse the handle: gsr_upload replaces the system
    for s0 in range(0, cfg.n_stars, step):
        part = synth.generate_rows(cfg, s0, min(s0 + step, cfg.n_stars), dev, rp)
        r0, nr = part["row0"], part["values"].shape[0]
        hv[r0:r0 + nr].copy_(part["values"])
        hia[r0:r0 + nr].copy_(part["matrixIndexAstro"])
        hit[r0:r0 + nr].copy_(part["matrixIndexAtt"])
        hic[r0:r0 + nr].copy_(part["instrCol"])
        hb[r0:r0 + nr].copy_(part["noise"])
        del part
    torch.cuda.synchronize()
    # b = A x_true + noise with the library (upload raw system once, untimed, to form b)
    G2.gsr_upload(hv, hia, hit, hic, hb)
    bt = hb.to(dev)
    G2.gsr_aprod1(synth.x_true(cfg, dev), bt)
    hb.copy_(bt)
    del bt
    torch.cuda.synchronize()
    K = args.steps
    t0 = time.perf_counter()
    G2.gsr_upload(hv, hia, hit, hic, hb)
    G2.gsr_precondition()
    r = G2.gsr_lsqr(K, 0.0, 0.0, host_out=True)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    assert r.itn == K
    h2d = (hv.numel() * 8 + hia.numel() * 8 + hit.numel() * 8 + hic.numel() * 4 + hb.numel() * 8) / K
    d2h = 2 * G.n * 8 / K
    return {"value": K / dt, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
            "seconds": dt, "steps": K,
            "note": "timed: gsr_upload (pinned host -> HBM) + gsr_precondition + gsr_lsqr(K) with x, se to host"}


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        main_reference(a)
    else:
        main_ours(a)
