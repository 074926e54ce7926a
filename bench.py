#!/usr/bin/env python
"""bench.py - H_eff*psi sustained FP64 TFLOPS on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cyp] [--impl ours|reference]
                    [--davidson | --site-update | --stream FRAC] [--share-adjoint] [--D D]

A *step* is one pass of the whole hot path (hpsi_apply: prep, first GEMM, second GEMM, reduce) over one seeded
synthetic psi of the named config (default ``cyp`` = BASELINE.json configs[2], the D=4096 config the metric is
quoted on).  ``value`` = useful flops (A18: sum over tasks of min(f1, f2)) x steps / device time, inputs
resident in HBM; ``e2e`` = the same through hpsi_apply_host with pinned HOST psi/out buffers (H2D + D2H inside the
timed region).  N > 1: one rank per GPU (started by torchrun, or by this script itself when WORLD_SIZE is not set);
the term list is sharded over the ranks by hpsi_shard_terms (balanced by useful flops; operators are the big object),
every rank plans its shard with hpsi_plan_ex, psi is replicated, and the exchange step inside the timed region is one
NCCL all-gather of the partial psi' plus hpsi_sum_shards (rank-ordered sum: same bits on every rank); total work is
fixed -> "strong".  ``--impl reference`` times the CPU oracle (oracle/, as it stands) on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "H_eff*psi sustained FP64 TFLOPS on 1 B200 (% of measured FP64 TC peak)"
CONFIG_DESC = {
    "toy": "configs[0] toy", "small": "configs[1] small QC-like D=1024", "cyp": "configs[2] CYP-shaped D=4096",
    "femoco": "configs[3] FeMoco-shaped D=8192", "stress": "configs[4] load-imbalance stress D=4096",
}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# --------------------------------------------------------------------------------------------- clocks sampling
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *exc):
        if self.proc is not None:
            time.sleep(0.25)
            self.proc.terminate()
            self.thread.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------------ calibration
def dgemm_calibration(torch, secs=2.0, sizes=(4096, 8192, 16384), device_index=0):
    """Same-run FP64 tensor-core peak: cuBLAS DGEMM (torch.matmul on float64), sustained 2N^3/t over >= ``secs`` of
    back-to-back launches per N between two CUDA events (no host synchronisation inside the window), SM clocks sampled
    meanwhile.  Returns (best TFLOP/s, {per-N figures, clocks})."""
    best, detail = 0.0, {}
    stream = torch.cuda.current_stream()
    with ClockSampler(device_index) as clk:
        for N in sizes:
            a = torch.randn(N, N, dtype=torch.float64, device="cuda")
            b = torch.randn(N, N, dtype=torch.float64, device="cuda")
            c = torch.empty_like(a)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for _ in range(2):
                torch.matmul(a, b, out=c)
            e0.record(stream)
            torch.matmul(a, b, out=c)
            e1.record(stream)
            torch.cuda.synchronize()
            reps = max(3, int(np.ceil(secs * 1e3 / max(e0.elapsed_time(e1), 1e-3))))
            e0.record(stream)
            for _ in range(reps):
                torch.matmul(a, b, out=c)
            e1.record(stream)
            torch.cuda.synchronize()
            sec = e0.elapsed_time(e1) * 1e-3
            tf = 2.0 * N ** 3 * reps / sec / 1e12
            detail[f"dgemm_{N}"] = round(tf, 3)
            detail[f"dgemm_{N}_seconds"] = round(sec, 2)
            best = max(best, tf)
            del a, b, c
    detail["clocks"] = clk.summary()
    return best, detail


def pipe_probes(H, calib):
    """Register-resident DMMA / DFMA issue-rate probes (libhpsi_bench.so) next to the DGEMM figure."""
    for kind, name in ((0, "dmma_pipe_probe"), (1, "dfma_pipe_probe")):
        ms_pipe, fl_pipe = H.hpsi_bench_fp64_pipe(kind, 20000)
        calib[name] = round(fl_pipe / ms_pipe / 1e9, 3)


def git_head():
    try:
        return subprocess.check_output(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], stderr=subprocess.DEVNULL,
                                       text=True).strip()
    except (OSError, subprocess.CalledProcessError):
        return None


KERNEL_SOURCES = ("kernels.cu", "kernels.cuh", "kernels_common.cuh", "kernels_paired.cu", "kernels_fused.cu", "plan.h")


def kernel_sources_digest():
    """sha1 over the sources of the GEMM kernels: what tells whether a committed ncu capture still describes the kernels
    being timed (there is no .git on the GPU box, so the commit id alone cannot)."""
    import hashlib
    h = hashlib.sha1()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2407_07411_b200", "csrc", name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(key, kernel):
    """DRAM bytes per launch of ``kernel`` from the committed ncu --set full capture (profiles/ncu_traffic.json.txt).
    The file records the digest of the kernel sources the capture was taken with; if today's sources differ the figure is
    withheld (None) - a stale capture says nothing about the kernels being timed."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json.txt")) as fh:
            tab = json.load(fh)
    except (OSError, ValueError):
        return None, None
    now = kernel_sources_digest()
    src = {"file": "profiles/ncu_traffic.json.txt", "capture": tab.get("_capture"), "capture_commit": tab.get("_commit"),
           "capture_kernels_digest": tab.get("_kernels_digest"), "kernels_digest": now, "bench_commit": git_head()}
    val = tab.get(key, {}).get(kernel)
    if tab.get("_kernels_digest") != now:
        val = None
    return val, src


def host_cores():
    """What the CPU baseline ran on: logical CPUs the process may use, and physical cores if /proc/cpuinfo tells."""
    try:
        usable = len(os.sched_getaffinity(0))
    except AttributeError:
        usable = os.cpu_count()
    phys = None
    try:
        pairs = set()
        pid = cid = None
        for line in open("/proc/cpuinfo"):
            if line.startswith("physical id"):
                pid = line.split(":")[1].strip()
            elif line.startswith("core id"):
                cid = line.split(":")[1].strip()
            elif not line.strip():
                if pid is not None and cid is not None:
                    pairs.add((pid, cid))
                pid = cid = None
        phys = len(pairs) or None
    except OSError:
        pass
    return {"logical_cpus_usable": usable, "physical_cores_on_box": phys}


def sample_points(p, n, seed=1):
    rng = np.random.default_rng(seed)
    blocks = p.psi_blocks()
    bi = rng.integers(0, len(blocks), n)
    sl = np.array([blocks[b][0] for b in bi], np.int32)
    sx = np.array([rng.integers(0, blocks[b][2]) for b in bi], np.int32)
    sy = np.array([rng.integers(0, blocks[b][3]) for b in bi], np.int32)
    idx = np.array([blocks[b][4] + x * blocks[b][3] + y for b, x, y in zip(bi, sx, sy)], np.int64)
    return sl, sx, sy, idx


def cpu_baseline(cfg, budget_s=15.0):
    """The oracle as it stands, timed on this box's host cores on a bounded sample: the first n base terms (and their
    adjoints) of the config, n sized from a 1-term probe so that one apply takes about ``budget_s`` seconds."""
    import oracle
    half = workloads.config_params(cfg)["n_terms"] // 2

    def run(n):
        sp = workloads.make_problem(cfg, base_terms=np.arange(min(n, half)))
        psi = workloads.make_psi(sp)
        t0 = time.time()
        oracle.apply(sp, psi)
        dt = time.time() - t0
        return oracle.useful_flops(sp)[0], dt, sp.n_terms

    n = 1
    fl, dt, _ = run(n)
    for _ in range(3):                          # grow the sample until one apply takes a sizeable part of the budget
        if dt >= budget_s / 3 or n >= half:
            break
        n = int(max(n + 1, min(half, n * budget_s / max(dt, 1e-3))))
        fl, dt, _ = run(n)
    return {"value": fl / dt / 1e12, "unit": "TFLOPS", "cores": oracle.num_threads(), "kind": "oracle",
            "cores_detail": {"openmp_threads": oracle.num_threads(), **host_cores()},
            "sample": f"one oracle.apply on the first {n} of {half} base terms + adjoints of {cfg} "
                      f"({fl / 1e9:.2f} useful GF in {dt:.2f} s)"}, fl, dt


# ------------------------------------------------------------------------------------------- reference arm
def run_reference(args, rank):
    """bench.py --impl reference: the CPU oracle on host cores, bounded sample per step (rank 0 only)."""
    if rank != 0:
        return
    import oracle
    half = workloads.config_params(args.config)["n_terms"] // 2
    total_budget = 150.0
    per_step = total_budget / (args.steps + args.warmup)
    probe = workloads.make_problem(args.config, base_terms=np.arange(1))
    psi = workloads.make_psi(probe)
    t0 = time.time()
    oracle.apply(probe, psi)
    dt1 = max(time.time() - t0, 1e-4)
    n = int(max(1, min(half, per_step / dt1)))
    sp = workloads.make_problem(args.config, base_terms=np.arange(n))
    psi = workloads.make_psi(sp)
    flops = oracle.useful_flops(sp)[0]
    for _ in range(args.warmup):
        oracle.apply(sp, psi)
    t0 = time.time()
    for _ in range(args.steps):
        oracle.apply(sp, psi)
    dt = time.time() - t0
    val = flops * args.steps / dt / 1e12
    sample = f"each step = one oracle.apply on the first {n} of {half} base terms + adjoints ({flops / 1e9:.2f} useful GF)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "TFLOPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
        "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": CONFIG_DESC[args.config], "sample": sample},
        "cpu_baseline": {"value": val, "unit": "TFLOPS", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "TFLOPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


# ------------------------------------------------------------------------------ streamed operators (8(f)-3)
def run_streamed(args):
    """bench.py --stream FRAC: operators in pinned HOST memory, streamed through two device windows of FRAC of the
    arenas each (hpsi_stream_apply).  The step is host->device-bandwidth bound; reported beside the
    resident-operator line, it is not the headline."""
    import torch
    import paper_2407_07411_b200 as H
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(0)
    cfg = args.config
    p = workloads.make_problem(cfg, share_adjoint=args.share_adjoint)
    a_host = torch.from_numpy(p.a_data).pin_memory()
    b_host = torch.from_numpy(p.b_data).pin_memory()
    sp = H.hpsi_stream_create(p, a_host, b_host, int((p.a_len + p.b_len) * args.stream))
    psi = torch.from_numpy(workloads.make_psi(p)).cuda()
    out = torch.empty_like(psi)
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        H.hpsi_stream_apply(sp, psi, out, stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(0) as clk:
        e0.record(stream)
        for _ in range(args.steps):
            H.hpsi_stream_apply(sp, psi, out, stream)
        e1.record(stream)
        torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    flops = H.hpsi_stream_query(sp, H.HPSI_Q_USEFUL_FLOPS)
    copied = H.hpsi_stream_query(sp, H.HPSI_Q_OPERATOR_BYTES)
    sl, sx, sy, idx = sample_points(p, 32)
    ref = oracle_samples(cfg, workloads.make_psi(p), sl, sx, sy)          # the oracle on the fully materialised config
    got = out.cpu().numpy()[idx]
    print(json.dumps({
        "metric": METRIC, "value": flops / (ms * 1e-3) / 1e12, "unit": "TFLOPS", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": CONFIG_DESC[cfg], "operator_storage": "pinned host memory, streamed (hpsi_stream_apply)" +
                   (", adjoint terms share their partner's blocks (every byte crosses the link once)" if args.share_adjoint else ""),
                   "windows": H.hpsi_stream_query(sp, H.HPSI_SQ_N_WINDOWS),
                   "staging_bytes": H.hpsi_stream_query(sp, H.HPSI_SQ_STAGING_BYTES),
                   "h2d_operator_bytes_per_step": copied},
        "roofline": {"bound": "pcie", "achieved": copied / (ms * 1e-3) / 1e9, "unit": "GB/s", "peak": None, "frac": None,
                     "traffic": copied, "note": "host->device copy of the operator windows; compute overlaps it"},
        "clocks": clk.summary(), "parity_sample_rel_err": float(np.linalg.norm(got - ref) / np.linalg.norm(ref)),
        "gpu_launches": 4 * H.hpsi_stream_query(sp, H.HPSI_SQ_N_WINDOWS) * args.steps,
    }), flush=True)


# -------------------------------------------------------------------------- site update
def run_site_update(args):
    """bench.py --site-update: the two steps after the eigen-solve on the named config - hpsi_truncate (block Jacobi
    SVD of psi, chi_max = D/4: the enlarged basis carries the site dimension 4) and hpsi_rotate_apply
    (A' = O^T A O for every left operator block).  A step = one truncation + one operator update.  The update's
    roofline is the FP64 tensor pipe when its flops per operator byte exceed the ridge (same-run DGEMM / HBM copy
    bandwidth), HBM otherwise; reported beside the H_eff*psi line, not the headline."""
    import torch
    import paper_2407_07411_b200 as H
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(0)
    cfg = args.config
    p = workloads.make_problem(cfg)
    a = torch.from_numpy(p.a_data).cuda()
    b = torch.zeros(8, dtype=torch.float64, device="cuda")       # the right operators play no part here
    p_plan = workloads.make_problem(cfg, n_terms=2)               # psi block table only (sector table is the config's)
    pa, pb = torch.from_numpy(p_plan.a_data).cuda(), torch.from_numpy(p_plan.b_data).cuda()
    plan = H.plan_problem(p_plan, pa, pb)
    D = int(p.d_left.sum())
    chi_max = max(1, D // 4)
    psi_h = workloads.make_psi(p)
    psi = torch.from_numpy(psi_h).cuda()
    ot = torch.zeros(H.hpsi_query(plan, H.HPSI_Q_ISO_CAPACITY), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    chi, sigma, disc = H.hpsi_truncate(plan, psi, chi_max, ot, stream)
    rot = H.hpsi_rotate_plan(p.d_left, chi, p.a_desc, a, p.a_len)
    rq = lambda w: H.hpsi_rotate_query(rot, w)  # noqa: E731
    out = torch.empty(rq(H.HPSI_RQ_OUT_LENGTH), dtype=torch.float64, device="cuda")
    log(f"{cfg}: D {D} -> chi {int(chi.sum())} (discarded weight {disc:.3e}), {len(p.a_desc)} A blocks, "
        f"{rq(H.HPSI_RQ_ALGO_BYTES) / 1e9:.2f} GB read+written, {rq(H.HPSI_RQ_USEFUL_FLOPS) / 1e9:.1f} GF, "
        f"T^T {rq(H.HPSI_RQ_INTERMEDIATE_BYTES) / 1e9:.2f} GB, units {rq(H.HPSI_RQ_N_UNITS_1)} + {rq(H.HPSI_RQ_N_UNITS_2)}")

    def step():
        H.hpsi_truncate(plan, psi, chi_max, ot, stream)
        H.hpsi_rotate_apply(rot, ot, out, stream)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(0) as clk:
        e0.record(stream)
        for _ in range(args.steps):
            step()
        e1.record(stream)
        torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    # the two parts separately
    e0.record(stream)
    for _ in range(args.steps):
        H.hpsi_truncate(plan, psi, chi_max, ot, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_trunc = e0.elapsed_time(e1) / args.steps
    e0.record(stream)
    for _ in range(args.steps):
        H.hpsi_rotate_apply(rot, ot, out, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms_rot = e0.elapsed_time(e1) / args.steps
    prof = np.zeros(3)
    for _ in range(3):
        prof += np.array(H.hpsi_rotate_apply_profiled(rot, ot, out, stream))
    prof /= 3
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            hbm_peak, peak_src = float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (burst copy)"
    except (OSError, ValueError, KeyError):
        hbm_peak, peak_src = 6550.0, "fallback of B200_PROFILING.md"
    algo = rq(H.HPSI_RQ_ALGO_BYTES)
    dgemm_peak, calib = dgemm_calibration(torch)
    rot_tf = rq(H.HPSI_RQ_USEFUL_FLOPS) / (ms_rot * 1e-3) / 1e12
    rot_gbs = algo / (ms_rot * 1e-3) / 1e9
    ridge = dgemm_peak * 1e12 / (hbm_peak * 1e9)
    tensor_bound = rq(H.HPSI_RQ_USEFUL_FLOPS) / max(algo, 1) > ridge
    traffic, traffic_src = ncu_traffic(cfg + "_site_update", "p1_kernel_rot")   # DRAM bytes of the two launches (ncu --set full)
    # parity on a sample of blocks the oracle rotates one by one, with the device's own isometries
    from oracle import site_update as su
    oth = ot.cpu().numpy()
    ots, o = [], 0
    for l in range(len(chi)):
        n = int(chi[l]) * int(p.d_left[l])
        ots.append(oth[o:o + n].reshape(int(chi[l]), int(p.d_left[l])))
        o += n
    rng = np.random.default_rng(7)
    pick = np.sort(rng.choice(len(p.a_desc), size=min(64, len(p.a_desc)), replace=False))
    desc = H.hpsi_rotate_query(rot, H.HPSI_RQ_OUT_BLOCKS)[pick]
    t0 = time.time()
    ref = su.rotate(p.d_left, chi, p.a_desc[pick], p.a_data, ots)
    outh = out.cpu().numpy()
    num = den = 0.0
    for e, x in zip(desc, ref):
        if e["offset"] < 0:
            continue
        g = np.lib.stride_tricks.as_strided(outh[int(e["offset"]):], shape=x.shape, strides=(int(e["ld"]) * 8, 8))
        num += float(np.sum((g - x) ** 2)); den += float(np.sum(x ** 2))
    # CPU baseline: the oracle (numpy SVD per block + BLAS rotation) on a bounded sample of blocks
    t0 = time.time()
    su.truncate(p, psi_h, chi_max)
    t_trunc_cpu = time.time() - t0
    nb = min(len(p.a_desc), 4000)
    t0 = time.time()
    su.rotate(p.d_left, chi, p.a_desc[:nb], p.a_data, ots)
    t_rot_cpu = (time.time() - t0) * len(p.a_desc) / nb
    print(json.dumps({
        "metric": "site update (SVD truncation + operator update O^T A O) per second, FP64", "value": 1e3 / ms,
        "unit": "updates/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": CONFIG_DESC[cfg] + " - site update", "D": D, "chi_max": chi_max, "kept": int(chi.sum()),
                   "a_blocks": int(len(p.a_desc)), "algorithmic_bytes": algo, "useful_flops": rq(H.HPSI_RQ_USEFUL_FLOPS),
                   "intermediate_bytes": rq(H.HPSI_RQ_INTERMEDIATE_BYTES), "l2": "inputs larger than L2 (operators read once)"},
        "parts_ms": {"hpsi_truncate": ms_trunc, "hpsi_rotate_apply": ms_rot, "rot_prep": float(prof[0]),
                     "rotate launch 1 (A O)": float(prof[1]), "rotate launch 2 (O^T T)": float(prof[2]),
                     "svd_sweeps": H.hpsi_query(plan, H.HPSI_Q_SVD_SWEEPS), "svd_launches": H.hpsi_query(plan, H.HPSI_Q_SVD_LAUNCHES)},
        "roofline": {"bound": "tensor" if tensor_bound else "hbm", "kernel": "p1_kernel<TMA, ROT> x2 (hpsi_rotate_apply)",
                     "achieved": rot_tf if tensor_bound else rot_gbs, "peak": dgemm_peak if tensor_bound else hbm_peak,
                     "unit": "TFLOP/s" if tensor_bound else "GB/s",
                     "frac": rot_tf / dgemm_peak if tensor_bound else rot_gbs / hbm_peak, "traffic": traffic,
                     "traffic_source": traffic_src, "peak_source": "same-run cuBLAS DGEMM calibration" if tensor_bound else peak_src,
                     "flops_per_algorithmic_byte": rq(H.HPSI_RQ_USEFUL_FLOPS) / max(algo, 1), "ridge": ridge,
                     "tflops": rot_tf, "algorithmic_gbs": rot_gbs},
        "calibration": {"fp64_tc_peak_tflops": dgemm_peak, **calib},
        "clocks": clk.summary(), "parity_sample_rel_err": float(np.sqrt(num / max(den, 1e-300))),
        "gpu_launches": (H.hpsi_query(plan, H.HPSI_Q_SVD_LAUNCHES) + 3) * args.steps,
        "cpu_baseline": {"value": 1.0 / (t_trunc_cpu + t_rot_cpu), "unit": "updates/s", "cores": os.cpu_count(), "kind": "oracle",
                         "sample": f"oracle truncate in full ({t_trunc_cpu:.2f} s) + oracle rotate on the first {nb} of "
                                   f"{len(p.a_desc)} blocks, scaled ({t_rot_cpu:.2f} s)"},
    }), flush=True)


# ------------------------------------------------------------------------------------------------- our arm
def shard_for_rank(cfg, rank, world, share_adjoint=False, D=None):
    """What rank ``rank`` of ``world`` holds and plans: the library partitions the term list
    (hpsi_shard_terms, balanced by useful flops, adjoint pairs kept together), the generator fills the arenas of the
    rank's own terms only, and the returned keyword arguments make hpsi_plan_ex plan exactly that shard.
    Returns (problem, plan kwargs, useful flops per shard or None)."""
    if world == 1:
        return workloads.make_problem(cfg, share_adjoint=share_adjoint, D=D), {}, None
    import paper_2407_07411_b200 as H
    desc = workloads.make_problem(cfg, fill=False, share_adjoint=share_adjoint, D=D)
    half = desc.n_terms // 2
    shard_of, shard_flops = H.hpsi_shard_terms(desc, world, np.arange(desc.n_terms) % half)
    p = workloads.make_shard(cfg, shard_of, rank, share_adjoint=share_adjoint, D=D)
    return p, {"shard_of_term": shard_of, "shard_index": rank}, shard_flops


def oracle_samples(cfg, psi, sl, sx, sy, D=None, chunk_terms=64):
    """Sampled outputs of the UNSHARDED, fully materialised config, the oracle computing them one by one; the terms are
    streamed through it in chunks so that the host never holds more than ``chunk_terms`` base terms of operators."""
    import oracle
    half = workloads.config_params(cfg)["n_terms"] // 2
    vals = np.zeros(len(sl))
    for lo in range(0, half, chunk_terms):
        sp = workloads.make_problem(cfg, base_terms=np.arange(lo, min(half, lo + chunk_terms)), D=D)
        oracle.apply_samples(sp, psi, sl, sx, sy, vals=vals)
    return vals


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    import paper_2407_07411_b200 as H
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    H.lib()

    cfg = args.config
    t0 = time.time()
    p, plan_kw, shard_flops = shard_for_rank(cfg, rank, world, args.share_adjoint, args.D)
    gen_s = time.time() - t0
    a = torch.from_numpy(p.a_data).to(dev)
    b = torch.from_numpy(p.b_data).to(dev)
    arena_bytes = int(8 * (p.a_len + p.b_len))
    keep_host = world == 1 and not args.share_adjoint         # the parity leg's oracle reads the very same host arrays
    if not keep_host:
        p.a_data = p.b_data = None
    t0 = time.time()
    nv = max(1, args.n_vectors)                               # > 1: batched apply (hpsi_apply_multi), value counts all vectors
    if nv > 1:
        plan_kw = dict(plan_kw, n_vectors=nv)
    plan = H.plan_problem(p, a, b, **plan_kw)
    plan_s = time.time() - t0
    q = lambda w: H.hpsi_query(plan, w)  # noqa: E731
    n = q(H.HPSI_Q_PSI_LENGTH)
    sums = torch.tensor([q(H.HPSI_Q_USEFUL_FLOPS), q(H.HPSI_Q_OPERATOR_BYTES), q(H.HPSI_Q_N_TASKS), arena_bytes],
                        dtype=torch.int64, device=dev)
    if world > 1:
        dist.all_reduce(sums)
    useful_flops, operator_bytes, n_tasks, arena_total = (int(v) for v in sums.tolist())
    useful_flops *= nv                                        # one step = H psi_v for every vector of the batch
    log(f"[rank {rank}] {cfg}: gen {gen_s:.1f}s plan {plan_s:.2f}s tasks {q(H.HPSI_Q_N_TASKS)} "
        f"useful {q(H.HPSI_Q_USEFUL_FLOPS) / 1e9:.1f} GF issued {q(H.HPSI_Q_ISSUED_FLOPS) / 1e9:.1f} GF "
        f"operators {q(H.HPSI_Q_OPERATOR_BYTES) / 1e9:.2f} GB workspace {q(H.HPSI_Q_WORKSPACE_BYTES) / 1e9:.2f} GB")

    # DGEMM calibration before the timed region (and again after it: same process, interleaved - SURVEY.md 8(d), H6)
    dgemm_before, calib = dgemm_calibration(torch, device_index=local_rank)
    pipe_probes(H, calib)

    stream = torch.cuda.current_stream()
    n_psi = 10 if cfg == "femoco" else 1                      # A17: 10 different psi's for the FeMoco config
    if nv > 1:
        assert world == 1, "--n-vectors is a single-GPU measurement"
        psis = [torch.from_numpy(np.stack([workloads.make_psi(p, k * nv + v) for v in range(nv)])).to(dev) for k in range(n_psi)]
        out = torch.empty(nv * n, dtype=torch.float64, device=dev)
    else:
        psis = [torch.from_numpy(workloads.make_psi(p, k)).to(dev) for k in range(n_psi)]
        out = torch.empty(n, dtype=torch.float64, device=dev)
    parts = torch.empty(world * n, dtype=torch.float64, device=dev) if world > 1 else None
    mine = parts[rank * n:(rank + 1) * n] if world > 1 else out

    def step(i):
        if nv > 1:
            H.hpsi_apply_multi(plan, psis[i % n_psi], out, nv, stream)
            return
        H.hpsi_apply(plan, psis[i % n_psi], mine, stream)
        if world > 1:                                         # exchange step: all-gather + rank-ordered sum
            dist.all_gather_into_tensor(parts, mine)
            H.hpsi_sum_shards(parts, world, out, stream)

    def sync_all():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, sampler=None):
        """device milliseconds of ``steps`` calls: barrier + synchronize on both sides, events on the launching stream,
        max over ranks (plus every rank's own figure)"""
        sync_all()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(steps):
            fn(i)
        e1.record(stream)
        sync_all()
        ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
        allms = [ms.clone() for _ in range(world)]
        if world > 1:
            dist.all_gather(allms, ms)
        per_rank = [float(x.item()) for x in allms]
        return max(per_rank), per_rank

    for i in range(args.warmup):
        step(i)
    with ClockSampler(local_rank) as clk:
        ms_total, per_rank_ms = timed(step, args.steps)
    value = useful_flops * args.steps / (ms_total * 1e-3) / 1e12

    # ---- roofline of the dominant kernel (live CUDA events between the kernels of an apply), taken right after the timed
    # region, i.e. in the same clock / power state as `value` (the >= 2 s legs below pull the SM clock down under the 1 kW cap)
    prof = np.zeros(4)
    for i in range(3):                                        # (one vector's worth of work, also for a batched plan)
        prof += np.array(H.hpsi_apply_profiled(plan, psis[0][:n] if nv > 1 else psis[0], mine[:n], stream))
    prof /= 3
    names = ["prep_kernel", "p1_kernel (first GEMM)", "p2_kernel (second GEMM)", "reduce_kernel"]
    fl_p1 = q(H.HPSI_Q_USEFUL_FLOPS_P1)
    fl = [0, fl_p1, q(H.HPSI_Q_USEFUL_FLOPS) - fl_p1, 0]
    dom = int(np.argmax(prof))
    achieved = fl[dom] / (prof[dom] * 1e-3) / 1e12 if prof[dom] > 0 else 0.0


    # ---- the same, sustained: >= 2 s of back-to-back steps (SURVEY.md 8(d) protocol; the K-step figure above is a burst
    # when K steps last a fraction of a second)
    n_sus = max(args.steps, int(np.ceil(2000.0 / max(ms_total / args.steps, 1e-3))))
    with ClockSampler(local_rank) as clk_sus:
        ms_sus, _ = timed(step, n_sus)
    sustained = {"value": useful_flops * n_sus / (ms_sus * 1e-3) / 1e12, "unit": "TFLOPS", "steps": n_sus,
                 "seconds": ms_sus * 1e-3, "clocks": clk_sus.summary()}

    # ---- compute only (no exchange step): shows the imbalance of the term shards
    apply_ms = None
    if world > 1:
        _, per_rank_apply = timed(lambda i: H.hpsi_apply(plan, psis[i % n_psi], mine, stream), args.steps)
        apply_ms = [x / args.steps for x in per_rank_apply]

    # ---- end to end: pinned HOST psi / out, H2D + D2H inside the timed region
    hpsi_in = [(psis[k].cpu() if nv > 1 else torch.from_numpy(workloads.make_psi(p, k))).pin_memory() for k in range(n_psi)]
    hout = torch.empty(nv * n, dtype=torch.float64).pin_memory()
    xdev = torch.empty(nv * n, dtype=torch.float64, device=dev)

    def e2e_step(i):
        if nv > 1:                                            # no host-buffer entry point for a batch: copies + hpsi_apply_multi
            xdev.copy_(hpsi_in[i % n_psi].reshape(-1), non_blocking=True)
            H.hpsi_apply_multi(plan, xdev, out, nv, stream)
            hout.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        elif world == 1:
            H.hpsi_apply_host(plan, hpsi_in[i % n_psi], hout, stream)       # the C-ABI call with HOST buffers
        else:
            xdev.copy_(hpsi_in[i % n_psi], non_blocking=True)
            H.hpsi_apply(plan, xdev, mine, stream)
            dist.all_gather_into_tensor(parts, mine)
            H.hpsi_sum_shards(parts, world, out, stream)
            hout.copy_(out, non_blocking=True)
            torch.cuda.synchronize()

    for i in range(min(args.warmup, 3)):
        e2e_step(i)
    ms2, _ = timed(e2e_step, args.steps)
    e2e_value = useful_flops * args.steps / (ms2 * 1e-3) / 1e12

    dgemm_after, calib_after = dgemm_calibration(torch, device_index=local_rank)
    calib["after_timed_region"] = calib_after
    dgemm_peak = max(dgemm_before, dgemm_after)               # the larger denominator (the smaller fraction)
    traffic, traffic_src = (None, None)
    if world == 1 and args.D is None:
        traffic, traffic_src = ncu_traffic(cfg + ("_share_adjoint" if args.share_adjoint else ""), names[dom].split()[0])
    roofline = {"bound": "tensor", "kernel": names[dom], "achieved": achieved, "peak": dgemm_peak, "unit": "TFLOP/s",
                "frac": achieved / dgemm_peak, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "same-run cuBLAS DGEMM calibration (north_star), best of N = 4096 / 8192 / 16384 sustained "
                               f">= 2 s each, before and after the timed region; DMMA.8x8x4 pipe probe {calib['dmma_pipe_probe']} TFLOP/s",
                "kernel_ms": {k: round(float(v), 4) for k, v in zip(names, prof)},
                "useful_flops_per_launch": int(fl[dom])}

    res = {
        "metric": METRIC, "value": value, "unit": "TFLOPS", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "pct_of_fp64_tc_peak": 100.0 * value / (dgemm_peak * world),
        "sustained": sustained,
        "operator_gbs": operator_bytes * args.steps / (ms_total * 1e-3) / 1e9,   # operator bytes streamed once per apply
        "config": {"workload": CONFIG_DESC[cfg], "sectors_per_side": int(p.q_left.shape[0]),
                   "D": int(p.d_left.sum()), "terms": int(workloads.config_params(cfg)["n_terms"]), "tasks": n_tasks,
                   "useful_flops_per_step": useful_flops, "operator_bytes": operator_bytes, "psi_length": n,
                   "parallelism": "1 GPU" if world == 1 else
                   f"terms sharded x{world} (hpsi_shard_terms + hpsi_plan_ex), psi replicated, NCCL all-gather of psi' + "
                   "hpsi_sum_shards (rank-ordered sum)",
                   "l2": "inputs larger than L2 (operators streamed once per step)",
                   "operator_storage": "adjoint terms share their partner's blocks (read transposed)" if args.share_adjoint
                   else "every block materialised", "operator_arena_bytes": arena_total,
                   "schedule": dict(zip(("p1_stages_per_unit", "p2_waves", "p2_min_unit_dmma"), q(H.HPSI_Q_TUNING))),
                   "vectors_per_step": nv},
        "calibration": {"fp64_tc_peak_tflops": dgemm_peak, **calib},
        "clocks": clk.summary(),
        "e2e": {"value": e2e_value, "unit": "TFLOPS", "h2d_bytes_per_step": 8 * n * world * nv, "d2h_bytes_per_step": 8 * n * world * nv},
        "gpu_launches": (int(q(H.HPSI_Q_LAUNCHES_PER_APPLY)) + (1 if world > 1 else 0)) * args.steps * world,
        "roofline": roofline,
    }
    if world > 1:
        res["ranks"] = {"step_ms": [x / args.steps for x in per_rank_ms], "apply_only_ms": apply_ms,
                        "apply_only_ms_min_max": [min(apply_ms), max(apply_ms)],
                        "shard_useful_flops": [int(x) for x in shard_flops],
                        "exchange_bytes_per_rank_per_step": 8 * n * (world - 1)}
    # ---- parity spot check on sampled outputs the oracle computes one by one, on the UNSHARDED problem (all ranks ran the
    # step; rank 0 checks the summed result)
    step(0)
    torch.cuda.synchronize()
    if rank == 0:
        sl, sx, sy, idx = sample_points(p, 32)
        psi0 = workloads.make_psi(p, 0)
        got = out.cpu().numpy()[idx]                    # (batched: the first vector of the batch)
        if nv > 1:
            psi0 = psis[0][0].cpu().numpy()
        del a, b
        if keep_host:
            import oracle
            ref = oracle.apply_samples(p, psi0, sl, sx, sy)
        else:                                   # the oracle only knows fully materialised, unsharded operators
            ref = oracle_samples(cfg, psi0, sl, sx, sy, D=args.D)
        res["parity_sample_rel_err"] = float(np.linalg.norm(got - ref) / np.linalg.norm(ref))
        if args.D is None and world == 1:           # the timed oracle: rank 0 at N = 1 only
            res["cpu_baseline"], _, _ = cpu_baseline(cfg)
        elif args.D is not None:
            res["config"]["workload"] += f" with D overridden to {args.D} (bond-dimension sweep, not a BASELINE config)"
        print(json.dumps(res), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# ----------------------------------------------------------------- eigensolver drivers (reading A17)
def run_davidson(args):
    """bench.py --davidson: the on-device drivers themselves ("total wall time spent in the Davidson
    diagonalization").  hpsi_davidson / hpsi_lanczos run a fixed number of mat-vecs (tol = 0 never stops them); reported:
    time per iteration, time of a bare hpsi_apply, and the driver's overhead = iteration time / apply time - 1."""
    import torch
    import paper_2407_07411_b200 as H
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(0)
    cfg = args.config
    p = workloads.make_problem(cfg, D=args.D)
    a, b = torch.from_numpy(p.a_data).cuda(), torch.from_numpy(p.b_data).cuda()
    p.a_data = p.b_data = None
    plan = H.plan_problem(p, a, b)
    n = H.hpsi_query(plan, H.HPSI_Q_PSI_LENGTH)
    flops = H.hpsi_query(plan, H.HPSI_Q_USEFUL_FLOPS)
    stream = torch.cuda.current_stream()
    psi0 = torch.from_numpy(workloads.make_psi(p)).cuda()
    out = torch.empty_like(psi0)
    iters = max(args.steps, 8)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def time_apply(k):
        for _ in range(3):
            H.hpsi_apply(plan, psi0, out, stream)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(k):
            H.hpsi_apply(plan, psi0, out, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / k

    res_solvers = {}
    with ClockSampler(0) as clk:
        apply_ms = time_apply(iters)
        for name, fn in (("davidson", H.hpsi_davidson), ("davidson_unpreconditioned", H.hpsi_davidson), ("lanczos", H.hpsi_lanczos)):
            kw = dict(tol=0.0, max_iter=iters, m_max=16)
            if name == "davidson_unpreconditioned":
                kw["precondition"] = False
            x = psi0.clone()
            fn(plan, x, stream=stream, **dict(kw, max_iter=4))                  # warm-up (allocates the subspace buffers)
            best = None
            for _ in range(3):
                x.copy_(psi0)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                e0.record(stream)
                theta, info = fn(plan, x, stream=stream, **kw)
                e1.record(stream)
                torch.cuda.synchronize()
                wall = (time.perf_counter() - t0) * 1e3
                ms = e0.elapsed_time(e1)
                if best is None or ms < best[0]:
                    best = (ms, wall, theta, info)
            ms, wall, theta, info = best
            per_it = ms / info["n_matvec"]
            res_solvers[name] = {"total_ms": ms, "host_wall_ms": wall, "n_matvec": info["n_matvec"], "ms_per_matvec": per_it,
                                 "theta": theta, "residual": info["residual"],
                                 "tflops": flops * info["n_matvec"] / (ms * 1e-3) / 1e12}
        # multi-root: the 4 lowest pairs, the new vectors of an iteration multiplied in one batched apply (a plan laid out
        # for 4 vectors over the same arenas); fixed mat-vec budget, so ms per mat-vec is comparable with the lines above
        if cfg in ("toy", "small") or args.D is not None:
            k = 4
            plan_k = H.plan_problem(p, a, b, n_vectors=k)
            X0 = torch.from_numpy(np.stack([workloads.make_psi(p, v) for v in range(k)])).cuda()
            X = X0.clone()
            H.hpsi_davidson_multi(plan_k, X, k, tol=0.0, max_iter=2 * k, m_max=16, stream=stream)
            best = None
            for _ in range(3):
                X.copy_(X0)
                torch.cuda.synchronize()
                e0.record(stream)
                thetas, info = H.hpsi_davidson_multi(plan_k, X, k, tol=0.0, max_iter=4 * iters, m_max=16, stream=stream)
                e1.record(stream)
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1)
                if best is None or ms < best[0]:
                    best = (ms, thetas, info)
            ms, thetas, info = best
            res_solvers["davidson_multi_4_roots"] = {
                "total_ms": ms, "host_wall_ms": ms, "n_matvec": info["n_matvec"], "ms_per_matvec": ms / info["n_matvec"],
                "theta": [float(t) for t in thetas], "residual": info["residual"],
                "tflops": flops * info["n_matvec"] / (ms * 1e-3) / 1e12}
            del plan_k
        apply_ms_after = time_apply(iters)
    # the drivers run after the first bare-apply loop, i.e. in the power state the second loop sees (at cyp size the SM
    # clock sags under the 1 kW cap after ~1 s): the overhead is quoted against both
    for v in res_solvers.values():
        v["overhead_vs_bare_apply_before"] = v["ms_per_matvec"] / apply_ms - 1.0
        v["overhead_vs_bare_apply_after"] = v["ms_per_matvec"] / apply_ms_after - 1.0
    d = res_solvers["davidson"]
    print(json.dumps({
        "metric": "hpsi_davidson sustained FP64 TFLOPS (useful flops of its mat-vecs / total solver time)", "value": d["tflops"],
        "unit": "TFLOPS", "n_gpus": 1, "steps": d["n_matvec"], "warmup": 4, "ms_per_step": d["ms_per_matvec"],
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": CONFIG_DESC[cfg] + " - eigensolver drivers, fixed mat-vec count (tol = 0)", "psi_length": n,
                   "m_max": 16, "useful_flops_per_matvec": flops, "D": int(p.d_left.sum()),
                   "l2": "inputs larger than L2 (operators streamed once per mat-vec)" if cfg not in ("toy", "small") else
                   "operators fit L2 at this size; the regime is latency-bound (PAPER.md:82 pre-plateau)"},
        "bare_apply_ms": apply_ms, "bare_apply_ms_after": apply_ms_after, "solvers": res_solvers, "clocks": clk.summary(),
        "gpu_launches": int(d["n_matvec"] * (H.hpsi_query(plan, H.HPSI_Q_LAUNCHES_PER_APPLY) + 8)),
    }), flush=True)


def run_davidson_sharded(args, rank, world, local_rank):
    """bench.py --davidson --gpus N (or --exchange at N = 1): the term-sharded eigensolver, the paper's headline object
    ("eight GPU accelerated diagonalization procedure").  Every rank plans its shard (shard_for_rank), runs the
    same hpsi_davidson call on the replicated start vector, and the library hands every product to the exchange hook
    (hpsi_set_exchange): NCCL all-gather of the partial H v, then hpsi_sum_shards in rank order, so that all ranks hold
    the same bits and stay in lockstep.  Fixed mat-vec count (tol = 0); time on the device, max over ranks."""
    import torch
    import torch.distributed as dist
    import paper_2407_07411_b200 as H
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if not dist.is_initialized():
        if "MASTER_ADDR" not in os.environ:                   # --exchange at N = 1, started as plain python
            os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(free_port()), RANK="0", WORLD_SIZE="1")
        dist.init_process_group("nccl", device_id=dev)
    cfg = args.config
    p, plan_kw, shard_flops = shard_for_rank(cfg, rank, world, args.share_adjoint, args.D)
    a, b = torch.from_numpy(p.a_data).to(dev), torch.from_numpy(p.b_data).to(dev)
    p.a_data = p.b_data = None
    plan = H.plan_problem(p, a, b, **plan_kw)
    n = H.hpsi_query(plan, H.HPSI_Q_PSI_LENGTH)
    fl = torch.tensor([H.hpsi_query(plan, H.HPSI_Q_USEFUL_FLOPS)], dtype=torch.int64, device=dev)
    dist.all_reduce(fl)
    flops = int(fl.item())
    stream = torch.cuda.current_stream()
    parts = torch.empty((world, n), dtype=torch.float64, device=dev)
    n_exchanges = [0]

    def exchange(v, w, n_, nvec, ld, _stream):
        wt = H.device_tensor(w, (nvec, ld), torch)
        for k in range(nvec):
            dist.all_gather_into_tensor(parts, wt[k, :n_])
            H.hpsi_sum_shards(parts, world, wt[k, :n_], stream)
            n_exchanges[0] += 1
    H.hpsi_set_exchange(plan, exchange)
    psi0 = torch.from_numpy(workloads.make_psi(p)).to(dev)
    iters = max(args.steps, 8)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    x = psi0.clone()
    H.hpsi_davidson(plan, x, tol=0.0, max_iter=4, m_max=16, stream=stream)          # warm-up: buffers, NCCL channels
    best = None
    with ClockSampler(local_rank) as clk:
        for _ in range(3):
            x.copy_(psi0)
            n_exchanges[0] = 0
            torch.cuda.synchronize()
            dist.barrier()
            e0.record(stream)
            theta, info = H.hpsi_davidson(plan, x, tol=0.0, max_iter=iters, m_max=16, stream=stream)
            e1.record(stream)
            torch.cuda.synchronize()
            ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
            dist.all_reduce(ms, op=dist.ReduceOp.MAX)
            if best is None or ms.item() < best[0]:
                best = (ms.item(), theta, info, n_exchanges[0])
    ms, theta, info, nex = best
    # every rank must hold the same Ritz value and vector, bit for bit (rank-ordered sums)
    chk = torch.stack([x.sum(), x.abs().max(), torch.tensor(theta, dtype=torch.float64, device=dev)])
    allchk = [torch.empty_like(chk) for _ in range(world)]
    dist.all_gather(allchk, chk)
    same = all(torch.equal(allchk[0], c) for c in allchk)
    if rank == 0:
        print(json.dumps({
            "metric": "term-sharded hpsi_davidson sustained FP64 TFLOPS (useful flops of its mat-vecs over all ranks / solver time)",
            "value": flops * info["n_matvec"] / (ms * 1e-3) / 1e12, "unit": "TFLOPS", "n_gpus": world, "steps": info["n_matvec"],
            "warmup": 4, "ms_per_step": ms / info["n_matvec"], "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": CONFIG_DESC[cfg] + " - term-sharded Davidson, exchange = NCCL all-gather + hpsi_sum_shards",
                       "psi_length": n, "m_max": 16, "useful_flops_per_matvec": flops,
                       "shard_useful_flops": None if shard_flops is None else [int(v) for v in shard_flops]},
            "theta": theta, "residual": info["residual"], "exchanges": nex, "ranks_bitwise_equal": bool(same),
            "clocks": clk.summary(),
            "gpu_launches": int(info["n_matvec"] * (H.hpsi_query(plan, H.HPSI_Q_LAUNCHES_PER_APPLY) + 9)),
        }), flush=True)
    dist.barrier()
    dist.destroy_process_group()


def free_port():
    import socket
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    return port


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cyp", choices=list(CONFIG_DESC))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--stream", type=float, default=0.0,
                    help="stream the operators from pinned host memory through two windows of this fraction of the arenas")
    ap.add_argument("--share-adjoint", action="store_true",
                    help="adjoint terms read their partner's blocks transposed (half the operator bytes; hpsi_terms_t a_transposed)")
    ap.add_argument("--D", type=int, default=None,
                    help="override the config's bond dimension per side (sweep over D as in the paper's Fig. 1-2; 1 GPU)")
    ap.add_argument("--site-update", action="store_true",
                    help="time the steps after the eigen-solve instead: hpsi_truncate + hpsi_rotate_apply (SURVEY 8(f)-4)")
    ap.add_argument("--n-vectors", type=int, default=1,
                    help="batched apply: hpsi_apply_multi on this many vectors per step (plan built with n_vectors; 1 GPU)")
    ap.add_argument("--davidson", action="store_true",
                    help="time the eigensolver drivers (hpsi_davidson, hpsi_lanczos) and their overhead over a bare hpsi_apply")
    ap.add_argument("--exchange", action="store_true",
                    help="with --davidson at 1 GPU: run the term-sharded solver path (exchange hook, NCCL group of one rank)")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if "WORLD_SIZE" not in os.environ and args.gpus > 1 and args.impl == "ours":
        # started as plain `python bench.py --gpus N`: become N ranks, one per GPU (same launch the driver uses)
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but only {have} CUDA device(s) are visible")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
        os.execv(sys.executable, cmd)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and args.impl == "ours":
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE is {world}")
    if args.impl == "reference":
        run_reference(args, rank)
    elif args.stream > 0:
        if rank == 0:
            run_streamed(args)
    elif args.site_update:
        if rank == 0:
            run_site_update(args)
    elif args.davidson and (world > 1 or args.exchange):
        run_davidson_sharded(args, rank, world, local_rank)
    elif args.davidson:
        if rank == 0:
            run_davidson(args)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
