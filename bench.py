#!/usr/bin/env python
"""bench.py -- LSQR iterations/s of the AVU-GSR hot path on B200 (BASELINE.json metric).

A "step" is one LSQR iteration (aprod1 + aprod2 + norms + vector updates + stop tests, SURVEY 8(a)
rows a2-a11) over one synthetic Gaia-shaped system resident in HBM.  Default workload: BASELINE
configs[2] "medium" (1M stars x 200 obs = 200M rows, 46.4 GB), the config the metric's 70 %-of-HBM
target is quoted on.  Inputs are seeded and synthetic (paper_2308_00778_b200.synth); the paper's
Gaia datasets are proprietary.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload medium|small|tiny|skewed|large]
                  [--skew-alpha 1.47] [--rerun 2] [--layout NA,NT,NI,NG]
  python bench.py --impl reference ...     # the CPU oracle, as it stands, on a bounded sample

K iterations are timed as solves of at most 20 iterations of the same system (the synthetic systems reach the rounding
floor, istop 5, after ~31 iterations at Medium); the timed quantity is the device time of the iteration loops.

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
# The METHOD's algorithmic bytes per row (upload-format widths): what one aprod must move however it is
# implemented.  Used only for the two north-star figures `iteration_frac` and `aprod1_plus_aprod2_frac`.
ROW_BYTES_APROD1 = 248      # 192 values + 40 indices + 8 read y + 8 write y
ROW_BYTES_APROD2 = 240      # 192 values + 40 indices + 8 read y
SOLVE_LEN = 20             # iterations per timed solve (see main_ours)
NOMINAL_HBM_GBS = 8000.0    # north_star's "~8 TB/s", printed beside the measured copy peak


def kernel_row_bytes(cfg, path_info, gsr):
    """Bytes per row each kernel has to stream with the DEVICE layout -- its own algorithmic bytes; a
    kernel is never credited with bytes it does not move.  values 8 B each; instrument columns 2 or 4 B; attitude
    start 4 B; star: 8 B per 32-row tile; u 8 B read (+ 8 B written).  For any section widths (cfg); `method_*` are the
    METHOD's bytes with the upload-format index widths (8 B per M_i entry, 4 B per instrument column)."""
    ic = (2 if path_info & gsr.GSR_PATH_IC16 else 4) * cfg.n_instr_par
    star = 8 / 32 if cfg.n_astro_par else 0
    att = 4 if cfg.n_att_par else 0
    full = 8 * cfg.n_par + ic + att + star
    idx = 8 * bool(cfg.n_astro_par) + 8 * bool(cfg.n_att_par) + 4 * cfg.n_instr_par
    return {
        "k_aprod1": full + 8 + 8,                                # whole row, y read + written
        "k_aprod2_redatt": full + 8,                             # all sections in one kernel (no attitude copy)
        "k_aprod2": full - 8 * cfg.n_att_par - att + 8,          # astro / instr / global sections only
        "k_aprod2_att": 96 + 4 + 4 + 8,                          # attT + start + permutation + gathered y
        "k_aprod2_att_linear": 96 + 4 + 8,                       # attT + start + uT
        "k_u_to_time": 4 + 8 + 8,                                # permutation + gathered u + uT written
        "k_aprod2_fused": full + 8 + 8,                          # whole row ONCE, u read + written
        "k_aprod2_noins": 8 * (cfg.n_astro_par + cfg.n_glob) + star + 8,   # astro + global coefficients only (instr by k_ins_scatter)
        "k_ins_scatter": 6 * (8 + 4) + 8,                        # column-ordered copy: value + (column, row) word; u staged once
        "method_aprod1": 8 * cfg.n_par + idx + 16, "method_aprod2": 8 * cfg.n_par + idx + 8,
    }


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
    ap.add_argument("--skew-alpha", type=float, default=2.0,
                    help="exponent of the skewed workload's obs-count law (2.0: literal, ~53 M rows; 1.47: ~150 M rows, DESIGN.md R18)")
    ap.add_argument("--layout", default="5,12,6,1",
                    help="section widths N_Astro,N_Att,N_Instr,N_Glob of the workload (PAPER.md:78; 5,12,6,1 = production; "
                         "0,12,6,0 and 5,0,0,0 are the section subsets of the paper's 40/300 GB and 100 GB datasets)")
    ap.add_argument("--rerun", type=int, default=0,
                    help="extra solves of the same system after the timed one; reports run-to-run max|dx| (atomics)")
    return ap.parse_args()


def workload_cfg(name, skew_alpha=2.0, layout="5,12,6,1"):
    import dataclasses
    from paper_2308_00778_b200 import synth
    if layout != "5,12,6,1":
        na, nt, ni, ng = (int(t) for t in layout.split(","))
        return dataclasses.replace(workload_cfg(name, skew_alpha), n_astro_par=na, n_att_par=nt, n_instr_par=ni, n_glob=ng)
    if name == "skewed":
        return synth.skewed(alpha=skew_alpha)
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


def host_facts():
    import psutil
    model = "?"
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "physical_cores": psutil.cpu_count(logical=False), "cpu_model": model,
            "ram_gb": round(psutil.virtual_memory().total / 1e9, 1)}


def oracle_sample_run(cfg, steps, warmup, target_rows=3_000_000, omp=True):
    """The CPU oracle, as it stands, on a bounded sample of the workload: the first `ns` stars with the full
    attitude / instrument column ranges.  (a) oracle/gsr_oracle.c, one thread (the parity oracle itself);
    (b) oracle/gsr_oracle_omp.c, the same loops threaded the way the paper's CPU solver is, on all
    cores.  it/s are scaled linearly in rows to the full workload and labelled as such."""
    import dataclasses
    import oracle
    from paper_2308_00778_b200 import synth
    full_rows = int(synth.star_rowptr(cfg)[-1])
    ns = max(1, min(cfg.n_stars, int(cfg.n_stars * target_rows / max(full_rows, 1))))
    sub = dataclasses.replace(cfg, name=cfg.name + "_sample", n_stars=ns, n_con=0, con_nnz=0)
    d = {k: v.numpy() for k, v in synth.generate(sub).items()}
    S = oracle.OracleSystem(sub.n_stars, sub.n_dof_att, sub.n_instr, d["values"], d["matrixIndexAstro"],
                            d["matrixIndexAtt"], d["instrCol"], n_glob=sub.n_glob, n_astro_par=sub.n_astro_par,
                            n_att_par=sub.n_att_par, n_instr_par=sub.n_instr_par)
    b = S.aprod1(d["x_true"], d["noise"])
    S.precondition()
    out = {"rows_sample": S.m, "rows_full": full_rows, "stars_sample": ns, "steps": steps, "host": host_facts()}

    def timed(solver):
        if warmup > 0:
            solver(b, warmup, 0.0, 0.0)
        t0 = time.perf_counter()
        r = solver(b, steps, 0.0, 0.0)
        dt = time.perf_counter() - t0
        assert r.itn == steps
        return dt / steps

    s1 = timed(S.lsqr)
    out["one_thread"] = {"s_per_it_sample": s1, "its_scaled": (1.0 / s1) * S.m / full_rows, "cores": 1}
    if omp:
        R = oracle.OmpRunner(S, 0)
        sN = timed(R.lsqr)
        out["all_cores"] = {"s_per_it_sample": sN, "its_scaled": (1.0 / sN) * S.m / full_rows, "cores": R.threads}
    out["sample"] = (f"oracle LSQR (gcc -O2), {steps} iterations on the first {ns} stars = {S.m} rows of "
                     f"'{cfg.name}' ({full_rows} rows); it/s scaled by rows {S.m}/{full_rows}")
    return out


def cpu_baseline_block(o):
    """`cpu_baseline` object of the JSON line: the all-core figure is the headline value, the one-thread figure
    (the parity oracle itself) sits beside it."""
    best = o.get("all_cores", o["one_thread"])
    blk = {"value": best["its_scaled"], "unit": UNIT, "cores": best["cores"], "kind": "oracle", "sample": o["sample"],
           "one_thread_its": o["one_thread"]["its_scaled"], "host": o["host"]}
    if "all_cores" in o:
        blk["all_cores_its"] = o["all_cores"]["its_scaled"]
        blk["threading"] = "oracle/gsr_oracle_omp.c: omp for over rows (aprod1), star-aligned row ranges with private att/instr/gamma accumulators (aprod2), PAPER.md:150"
    return blk


def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = workload_cfg(args.workload, args.skew_alpha, args.layout)
    # exactly --steps timed and --warmup untimed iterations per solver (one thread, then all cores), each step on a
    # bounded sample of the workload: 3 M rows, fewer when many steps are asked for, so that the run stays within minutes
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    o = oracle_sample_run(cfg, steps, warmup, target_rows=int(3_000_000 * min(1.0, 40.0 / (steps + warmup))))
    blk = cpu_baseline_block(o)
    val = blk["value"]
    best = o.get("all_cores", o["one_thread"])
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": 1e3 * best["s_per_it_sample"],
            "row_scale": o["rows_sample"] / o["rows_full"],
            "value_is": "1 / (ms_per_step of the sample) x row_scale: it/s extrapolated linearly in rows to the full workload",
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": args.workload, "sample": o["sample"]},
            "cpu_baseline": blk,
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

    cfg = workload_cfg(args.workload, args.skew_alpha, args.layout)
    rp = synth.star_rowptr(cfg)
    m = int(rp[-1])
    prod = (cfg.n_astro_par, cfg.n_att_par, cfg.n_instr_par, cfg.n_glob) == (5, 12, 6, 1)
    G = gsr.Gsr(m, cfg.n_stars, cfg.n_dof_att, cfg.n_instr, cfg.n_con, cfg.n_con * cfg.con_nnz, device=local,
                n_glob=cfg.n_glob, n_astro_par=cfg.n_astro_par, n_att_par=cfg.n_att_par, n_instr_par=cfg.n_instr_par)
    t_gen = time.perf_counter()
    build_on_device(cfg, G, dev, torch, synth)
    G.gsr_precondition()
    t_gen = time.perf_counter() - t_gen

    # ---- device-resident timing: W warm-up iterations, then exactly K timed iterations.
    # The synthetic systems are well conditioned after column scaling: LSQR reaches the rounding floor (istop 5) after
    # ~31 iterations at Medium, so K iterations are timed as ceil(K / SOLVE_LEN) solves of at most SOLVE_LEN iterations
    # of the same system; the timed quantity is the device time of the iteration loops (CUDA events on the library's
    # stream, gsr_last_timing), each solve bracketed by barrier + synchronize.
    G.gsr_lsqr(max(args.warmup, 3), 0.0, 0.0, want_se=False)
    barrier()
    lens = [SOLVE_LEN] * (args.steps // SOLVE_LEN) + ([args.steps % SOLVE_LEN] if args.steps % SOLVE_LEN else [])
    loop_ms_rank, launches, r = 0.0, 0, None
    with ClockSampler(local) as clk:
        for k in lens:
            barrier()
            r = G.gsr_lsqr(k, 0.0, 0.0)
            barrier()
            assert r.itn == k and r.istop == 7, (r.itn, r.istop, k)
            loop_ms_rank += r.loop_ms
            launches += int(r.kernel_launches)
    loop_ms, value = aggregate_replicas(loop_ms_rank, args.steps, world, dev, torch, dist)
    xt = synth.x_true(cfg, dev)
    x_err = float(torch.linalg.norm(r.x - xt) / torch.linalg.norm(xt))
    del xt
    rerun = None
    if args.rerun > 0:      # att / instr sums use floating-point atomics: how far do repeated solves of one system differ?
        dmax, drel = 0.0, 0.0
        for _ in range(args.rerun):
            r2 = G.gsr_lsqr(lens[-1], 0.0, 0.0)
            dmax = max(dmax, float((r2.x - r.x).abs().max()))
            drel = max(drel, float(torch.linalg.norm(r2.x - r.x) / torch.linalg.norm(r.x)))
            del r2
        rerun = {"solves": args.rerun + 1, "iterations": lens[-1], "max_abs_dx": dmax, "max_abs_x": float(r.x.abs().max()),
                 "rel_l2_dx": drel,
                 "what": "largest |x_run_k - x_run_0| over all unknowns (and the largest relative L2 difference) after "
                         "the same number of iterations"}

    # ---- per-kernel roofline: every kernel timed alone (CUDA events on the library's stream) against ITS OWN bytes
    peak, peak_src = peaks()
    info = G.gsr_path_info()
    fused = bool(info & gsr.GSR_PATH_FUSED)
    att_copy = bool(info & gsr.GSR_PATH_ATT_COPY)
    rb = kernel_row_bytes(cfg, info, gsr)
    reps = args.kernel_reps

    def timed_kernel(which):
        try:
            return G.gsr_time_aprod(which, reps)
        except gsr.GsrError:
            return None

    def entry(ms, bytes_per_row, extra_bytes=0.0):
        gb = (bytes_per_row * m + extra_bytes) / 1e9
        return {"ms": ms, "alg_gb": gb, "bytes_per_row": bytes_per_row, "gbs": gb / (ms * 1e-3),
                "frac_of_measured_peak": gb / (ms * 1e-3) / peak}

    k = {}
    ms1 = timed_kernel(gsr.GSR_TIME_K_APROD1)
    k["k_aprod1"] = entry(ms1, rb["k_aprod1"])
    ms2 = timed_kernel(gsr.GSR_TIME_K_APROD2_MAIN)
    ins_copy = bool(info & gsr.GSR_PATH_INS_COPY)
    k["k_aprod2"] = entry(ms2, (rb["k_aprod2_noins"] if ins_copy else rb["k_aprod2"]) if att_copy else rb["k_aprod2_redatt"], 8 * G.n)
    if ins_copy:
        k["k_aprod2"]["form"] = "astro + gamma only; the instrumental section runs in k_ins_scatter"
        k["k_ins_scatter"] = entry(timed_kernel(gsr.GSR_TIME_K_INS_SCATTER), rb["k_ins_scatter"])
    msut = timed_kernel(gsr.GSR_TIME_K_U_TO_TIME) if (info & gsr.GSR_PATH_UT) else None
    if msut is not None:
        k["k_u_to_time"] = entry(msut, rb["k_u_to_time"])
    ms2a = timed_kernel(gsr.GSR_TIME_K_APROD2_ATT) if att_copy else None
    att_linear = bool(info & gsr.GSR_PATH_UT)
    if ms2a is not None:
        k["k_aprod2_att"] = entry(ms2a, rb["k_aprod2_att_linear"] if att_linear else rb["k_aprod2_att"])
        k["k_aprod2_att"]["form"] = "linear (u in block-time order)" if att_linear else "gathers u through permT"
    msf = timed_kernel(gsr.GSR_TIME_K_FUSED) if fused else None
    if msf is not None:
        k["k_aprod2_fused"] = entry(msf, rb["k_aprod2_fused"])
    ms1g = G.gsr_time_aprod(gsr.GSR_TIME_APROD1_GROUP, reps)
    ms2g = G.gsr_time_aprod(gsr.GSR_TIME_APROD2_GROUP, reps)
    in_step = ["k_aprod2_fused", "k_aprod2_att"] + (["k_ins_scatter"] if ins_copy else []) + (["k_u_to_time"] if msut is not None else []) \
        if msf is not None else ["k_aprod1", "k_aprod2"] + (["k_aprod2_att"] if ms2a is not None else []) + (["k_ins_scatter"] if ins_copy else [])
    dom = max(in_step, key=lambda n: k[n]["ms"])
    # north-star figures on the METHOD's bytes (two products of 248 + 240 B/row)
    gb1 = rb["method_aprod1"] * m / 1e9      # 248 B/row in the production layout (ROW_BYTES_APROD1)
    gb2 = (rb["method_aprod2"] * m + 8 * G.n) / 1e9      # 240 B/row
    ms_step = loop_ms / args.steps
    # bytes the timed step actually has to stream with the device layout
    if msf is not None:
        moved = rb["k_aprod2_fused"] + (rb["k_aprod2_att_linear"] + rb["k_u_to_time"] if att_linear else rb["k_aprod2_att"])
        moved += rb["k_ins_scatter"] if ins_copy else 0
    else:
        moved = rb["k_aprod1"] + ((rb["k_aprod2_noins"] + rb["k_ins_scatter"] if ins_copy else rb["k_aprod2"]) + rb["k_aprod2_att"]
                                  if att_copy else rb["k_aprod2_redatt"])
    moved_gb = (moved * m + 12 * 8 * G.n) / 1e9
    traffic, traffic_src = None, None      # ncu-measured DRAM bytes per launch of the dominant kernel
    tpath = os.path.join(ROOT, "profiles", "r03_traffic.csv")
    if os.path.exists(tpath) and prod:
        for ln in open(tpath).read().splitlines()[1:]:
            w, kn, bts = ln.split(",")[:3]
            if w == args.workload and kn == dom and (w != "skewed" or abs(args.skew_alpha - 1.47) < 1e-9):
                traffic, traffic_src = float(bts) / 1e9, "profiles/r03_traffic.csv (one ncu --set full capture, see r03_ncu_full_summary.md)"
    roofline = {"bound": "hbm", "kernel": dom, "achieved": k[dom]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": k[dom]["gbs"] / peak, "traffic": traffic, "traffic_unit": "GB per launch (ncu dram read+write)",
                "traffic_source": traffic_src, "peak_source": peak_src, "nominal_peak": NOMINAL_HBM_GBS,
                "frac_of_nominal": k[dom]["gbs"] / NOMINAL_HBM_GBS,
                "note": "achieved = the dominant kernel's own device-layout bytes / its CUDA-event time; the two "
                        "north-star figures below use the METHOD's 248 + 240 B/row",
                "aprod1_plus_aprod2": {"alg_gb": gb1 + gb2, "ms": ms1g + ms2g, "gbs": (gb1 + gb2) / ((ms1g + ms2g) * 1e-3),
                                       "frac": (gb1 + gb2) / ((ms1g + ms2g) * 1e-3) / peak,
                                       "frac_of_nominal": (gb1 + gb2) / ((ms1g + ms2g) * 1e-3) / NOMINAL_HBM_GBS,
                                       "what": "gsr_aprod1 + gsr_aprod2 kernel groups timed alone, method bytes"},
                "iteration": {"alg_gb": gb1 + gb2, "ms": ms_step, "gbs": (gb1 + gb2) / (ms_step * 1e-3),
                              "frac": (gb1 + gb2) / (ms_step * 1e-3) / peak,
                              "frac_of_nominal": (gb1 + gb2) / (ms_step * 1e-3) / NOMINAL_HBM_GBS,
                              "moved_gb": moved_gb, "moved_gbs": moved_gb / (ms_step * 1e-3),
                              "moved_frac": moved_gb / (ms_step * 1e-3) / peak,
                              "form": "fused (A's row layout streamed once)" if msf is not None else "two products",
                              "what": "one LSQR iteration of the timed loop: method bytes (alg_gb) and bytes the device "
                                      "layout streams (moved_gb)"},
                "target": "north_star: aprod1+aprod2 >= 0.70 of HBM bandwidth at Medium",
                "kernels": k, "aprod1_group_ms": ms1g, "aprod2_group_ms": ms2g}

    # the same figures once more as flat scalars (a reader that keeps only the scalar keys of `roofline` loses nothing)
    a12, itn = roofline["aprod1_plus_aprod2"], roofline["iteration"]
    roofline.update({"aprod12_ms": a12["ms"], "aprod12_frac": a12["frac"], "aprod12_frac_nominal": a12["frac_of_nominal"],
                     "iteration_frac": itn["frac"], "iteration_moved_frac": itn["moved_frac"],
                     "iteration_moved_gb": itn["moved_gb"], "kernels_timed": "alone, back to back (gsr_time_aprod): "
                     "5-8 % slower than the same kernels inside the captured iteration, so their sum can exceed ms_per_step"})
    for name, e in k.items():
        roofline[name + "_ms"] = e["ms"]
        roofline[name + "_frac"] = e["frac_of_measured_peak"]

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": loop_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "layout": args.layout, "rows": m, "cols": G.n, "nnz_per_row": cfg.n_par,
                       "matrix_gb": (rb["method_aprod1"] - 16) * m / 1e9, "device_matrix_gb": (rb["k_aprod1"] - 16) * m / 1e9, "path_info": info, "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": "inputs larger than L2" if 232 * m > 2.5e8 else "L2-resident (launch-bound config)",
                       "x_rel_err_vs_planted": x_err, "setup_s": t_gen,
                       "timed_as": f"{len(lens)} solve(s) of <= {SOLVE_LEN} iterations; device time of the iteration loops",
                       **({"skew_alpha": args.skew_alpha} if args.workload == "skewed" else {}),
                       **({"run_to_run": rerun} if rerun else {})},
            "clocks": clk.summary(), "gpu_launches": launches, "roofline": roofline}

    # ---- end to end through the C ABI with HOST buffers: upload + precondition + K iterations + results
    if not args.no_e2e and rank == 0 and prod:
        line["e2e"] = e2e_run(args, cfg, G, dev, torch, synth, gsr)
    if not args.no_cpu_baseline and rank == 0 and world == 1:
        line["cpu_baseline"] = cpu_baseline_block(oracle_sample_run(cfg, 5, 1, omp=prod))
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
    need = 232 * m + 8 * (m + cfg.n_con)
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
    hb = torch.zeros(m + cfg.n_con, dtype=torch.float64, pin_memory=True)   # constraint rows: b_c = A_c x_true (noise 0)
    con = tuple(t.cpu().pin_memory() for t in synth.constraints(cfg, dev)) if cfg.n_con else None
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
    if con:
        G2.gsr_upload_constraints(*con)
    bt = hb.to(dev)
    G2.gsr_aprod1(synth.x_true(cfg, dev), bt)
    hb.copy_(bt)
    del bt
    torch.cuda.synchronize()
    K = min(args.steps, 25)      # one solve; the system reaches the rounding floor (istop 5) near iteration 31
    t0 = time.perf_counter()
    G2.gsr_upload(hv, hia, hit, hic, hb)
    if con:                                  # an upload discards the constraint rows (they are scaled in place)
        G2.gsr_upload_constraints(*con)
    t1 = time.perf_counter()                 # (every library call synchronises before it returns)
    G2.gsr_precondition()
    t2 = time.perf_counter()
    r = G2.gsr_lsqr(K, 0.0, 0.0, host_out=True)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    t_lsqr = time.perf_counter() - t2
    K = int(r.itn)               # iterations actually done (K unless the stop test fired earlier)
    h2d = (hv.numel() * 8 + hia.numel() * 8 + hit.numel() * 8 + hic.numel() * 4 + hb.numel() * 8) / K
    if con:
        h2d += sum(t.numel() * t.element_size() for t in con) / K
    d2h = 2 * G.n * 8 / K
    return {"value": K / dt, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
            "seconds": dt, "steps": K,
            # the parts of `seconds`: the first two do not depend on K, so `value` moves with K; the last one is per iteration
            "upload_s": t1 - t0, "precondition_s": t2 - t1, "lsqr_s": t_lsqr, "s_per_iteration": t_lsqr / K,
            "note": "timed: gsr_upload (pinned host -> HBM) + gsr_precondition + gsr_lsqr(K) with x, se to host"}


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        main_reference(a)
    else:
        main_ours(a)
