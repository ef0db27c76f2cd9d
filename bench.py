#!/usr/bin/env python
"""bench.py -- one CheFSI step (filter -> project -> rotate) on a synthetic workload, on N B200s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path: Chebyshev filter of degree m on the
N_d x N_s block, Hs = Psi^T H Psi, Ms = Psi^T Psi, and the in-place rotation Psi <- Psi Q, all through the
C ABI (include/sparc_gpu.h).  The headline `value` is BASELINE.json's metric: filter throughput in
grid-pt*orbital*degree/s (N_d*N_s*m / filter time); `hbm_gbs` (x24 B) and `subspace_tflops` are the other two
parts of that compound metric.  Default workload: BASELINE.json configs[4] (96x96x144, N_s = 7680, degree 24: the
largest one, 81.5 GB of Psi on one GPU); the default run then also times configs 0-3 and the sixth (finer-mesh, degree
33) workload for a few steps each and reports them under `per_config`.  `e2e` is the whole step through the host-buffer
entry point sparc_gpu_chefsi_step_host.

N > 1 (one rank per GPU under torchrun; `python bench.py --gpus N` starts the ranks itself): --parallelism shard (default)
partitions ONE workload as the paper does -- filter by columns without communication, all-to-all,
projection / rotation by rows with an all-reduce of Hs, Ms (paper_2302_09708_b200/dist.py) -- scaling = "strong";
--parallelism replicas runs N independent copies, scaling = "weak".

--impl reference times the CPU oracle (oracle/, acc_t = double build) on the host cores: a deliberately slow
program, reported as context.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "CheFSI filter grid-pt·orbital·degree/s + HBM GB/s; subspace FP64 TFLOP/s"
UNIT = "grid-pt*orbital*degree/s"
ALG_BYTES_PER_UNIT = 24.0       # read Psi_k, read Psi_{k-1}, write Psi_{k+1}

def load_ncu_traffic():
    """(config, kernel) -> dram__bytes_read.sum + dram__bytes_write.sum of ONE launch, from the committed `ncu --set full`
    captures (profiles/ncu_traffic.json names the capture and the kernel version of every entry)."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    try:
        with open(p) as f:
            doc = json.load(f)
        return {(int(e["config"]), e["kernel"]): float(e["bytes_per_launch"]) for e in doc["entries"]}
    except (OSError, ValueError, KeyError):
        return {}


NCU_TRAFFIC_BYTES_PER_LAUNCH = load_ncu_traffic()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms during the timed region."""

    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index: int):
        self.dev = device_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "50",
                 "-i", str(self.dev)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, pmax, reasons = [], None, None, set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax = float(f[2])
                pmax = max(pmax or 0.0, float(f[3]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_min_mhz": min(sm) if sm else None,
                "sm_max_mhz": smax, "power_w_max": pmax, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_filter_rate(wl, ncols, acc="f64"):
    """Time the CPU oracle's Chebyshev filter on `ncols` columns; returns (units/s, seconds, threads)."""
    from oracle import oracle as orc
    H = orc.Hamiltonian(wl, acc=acc)
    X = wl.psi_columns(range(ncols))
    t0 = time.perf_counter()
    H.chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    dt = time.perf_counter() - t0
    return wl.nd * ncols * wl.degree / dt, dt


def oracle_step_time(wl, ncols):
    """The oracle's whole step on `ncols` columns: filter, Hs / Ms, rotation by an ncols x ncols orthogonal Q.
    Returns (filter seconds, whole-step seconds)."""
    from oracle import oracle as orc
    H = orc.Hamiltonian(wl, acc="f64")
    X = wl.psi_columns(range(ncols))
    Q = np.linalg.qr(wl.q_matrix()[:ncols, :ncols])[0]
    t0 = time.perf_counter()
    F = H.chebyshev_filter(X, wl.degree, wl.a, wl.b, wl.a0)
    t1 = time.perf_counter()
    H.project(F)
    orc.rotate(F, Q)
    t2 = time.perf_counter()
    return t1 - t0, t2 - t0


def run_reference(args):
    """--impl reference: the CPU oracle as it stands on the host cores.  `value` = its filter rate (what our `value` measures),
    `e2e` = the same metric over its WHOLE step (filter + project + rotate) on the same sampled columns, which is what our
    `e2e` measures: the two ratios the driver forms are like for like."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2302_09708_b200 import workloads as wlmod
    from oracle import oracle as orc
    orc.build()
    cores = os.cpu_count() or 1
    wl = wlmod.make_workload(args.config)
    ncols = max(1, min(wl.ns, cores))
    tf, ts = [], []
    for i in range(args.warmup + args.steps):
        f, w = oracle_step_time(wl, ncols)
        if i >= args.warmup:
            tf.append(f)
            ts.append(w)
    dt, dt_step = sum(tf) / len(tf), sum(ts) / len(ts)
    units = float(wl.nd) * ncols * wl.degree
    value = units / dt
    sample = (f"{ncols} of the {wl.ns} columns of {wl.name} per step (degree {wl.degree}; columns are independent in the "
              f"filter; project / rotate on the {ncols} x {ncols} subspace), OpenMP over columns")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "nd": wl.nd, "ns": wl.ns, "degree": wl.degree, "sample_columns": ncols},
        "step_ms": {"filter": dt * 1e3, "project_rotate": (dt_step - dt) * 1e3},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": units / dt_step, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                "scope": "filter+project+rotate, solve excluded"},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def host_memory_available_bytes():
    """MemAvailable of the box, capped by the cgroup limit when there is one."""
    avail = None
    try:
        with open("/proc/meminfo") as f:
            for ln in f:
                if ln.startswith("MemAvailable:"):
                    avail = int(ln.split()[1]) * 1024
    except OSError:
        pass
    for pth in ("/sys/fs/cgroup/memory.max", "/sys/fs/cgroup/memory/memory.limit_in_bytes"):
        try:
            v = open(pth).read().strip()
            if v.isdigit():
                cur = 0
                try:
                    cur = int(open(pth.replace("memory.max", "memory.current")
                                   .replace("limit_in_bytes", "usage_in_bytes")).read().strip())
                except (OSError, ValueError):
                    pass
                lim = int(v) - cur
                avail = lim if avail is None else min(avail, lim)
        except OSError:
            pass
    return avail


KINDS = {0: "stencil_generic", 1: "stencil_tma", 2: "nl_project", 3: "nl_pull", 4: "gemm_tn", 5: "gemm_nn",
         6: "splitk_reduce", 7: "copy2d", 8: "nl_fused", 9: "nl_brick"}


def bench_config(env, config, steps, warmup, *, col_block=0, stencil_path=0, stencil_stages=0, do_e2e=True,
                 do_cpu=False, e2e_reps=2):
    """Time `steps` whole steps (filter -> project -> rotate) of workload `config` after `warmup` untimed ones; returns
    the numbers of one bench line (value, per-operator times, per-kernel rooflines, e2e, clocks, cpu_baseline)."""
    torch, dist, api, wlmod = env["torch"], env["dist"], env["api"], env["wlmod"]
    world, rank, local_rank, dev = env["world"], env["rank"], env["local_rank"], env["dev"]

    wl = wlmod.make_workload(config)
    g = api.SparcGpu(wl, device=local_rank)
    if stencil_path:
        g.set_option("stencil_path", stencil_path)
    if stencil_stages:
        g.set_option("stencil_stages", stencil_stages)
    nd, ns, m = wl.nd, wl.ns, wl.degree
    ld = nd
    psi = torch.empty((ns, ld), dtype=torch.float64, device=dev)

    def refill():
        # the filter is in place: regenerate Psi with the device restatement of the seeded generator (outside the
        # timers); this also sweeps L2 (the block is larger than the 126 MB L2 from config 1 on)
        api.fill_uniform(psi, wl.seed, wlmod.STREAM_PSI, 0, -1.0, 1.0)
    Qh = wl.q_matrix()
    Q = api.colmajor_from_numpy(Qh, device=dev)
    Hs = torch.empty((ns, ns), dtype=torch.float64, device=dev)
    Ms = torch.empty_like(Hs)
    col_block = col_block if col_block else wl.col_block
    l2_flush = None
    if ns * ld * 8 <= (256 << 20):              # config 0: the block fits L2 -- sweep it with a 256 MB write between steps
        l2_flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def ev():
        return torch.cuda.Event(enable_timing=True)

    def one_step(timers=None):
        refill()
        if l2_flush is not None:
            l2_flush.zero_()
        e = [ev() for _ in range(4)] if timers is not None else None
        if e: e[0].record()
        g.chebyshev_filter(psi, m, wl.a, wl.b, wl.a0, col_block=col_block)
        if e: e[1].record()
        g.project(psi, col_block=col_block, Hs=Hs, Ms=Ms)
        if e: e[2].record()
        g.rotate(psi, Q)
        if e: e[3].record()
        if timers is not None:
            timers.append(e)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        one_step()

    def timed_loop():
        barrier()
        sampler = ClockSampler(local_rank)
        if rank == 0:
            sampler.start()
        launches0 = g.get_info("kernel_launches")
        timers = []
        t_wall0 = time.perf_counter()
        for _ in range(steps):
            one_step(timers)
        barrier()
        t_wall = time.perf_counter() - t_wall0
        return timers, t_wall, g.get_info("kernel_launches") - launches0, (sampler.stop() if rank == 0 else None)

    def clocks_rejected(ck):
        # thermal / hardware slowdown, or SM clocks stuck well below max with no reason given (a leftover clock lock);
        # sw_power_cap is kept and noted
        if not ck or ck.get("sm_mhz") is None:
            return False
        bad = {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"} & set(ck["reasons"])
        stuck = ck["sm_max_mhz"] and ck["sm_mhz"] < 0.85 * ck["sm_max_mhz"] and not ck["reasons"]
        return bool(bad or stuck)

    timers, t_wall, launches, clocks = timed_loop()
    flag = torch.tensor([1.0 if clocks_rejected(clocks) else 0.0], dtype=torch.float64, device=dev)
    if world > 1:
        dist.broadcast(flag, 0)
    if float(flag.cpu()[0]) > 0:                 # rejected: measured again, once
        first = clocks
        timers, t_wall, launches, clocks = timed_loop()
        if clocks is not None:
            clocks["remeasured_after"] = first
            clocks["rejected"] = clocks_rejected(clocks)
    elif clocks is not None:
        clocks["rejected"] = False

    filt = sum(e[0].elapsed_time(e[1]) for e in timers) / steps
    proj = sum(e[1].elapsed_time(e[2]) for e in timers) / steps
    rot = sum(e[2].elapsed_time(e[3]) for e in timers) / steps
    t = torch.tensor([filt, proj, rot], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    filt, proj, rot = (float(x) for x in t.cpu())
    step_ms = filt + proj + rot

    # ---- end to end: the whole step through sparc_gpu_chefsi_step_host with HOST buffers -----------------------------
    # pinned host Psi -> H2D (column chunks, overlapped with the filter) -> filter -> project -> Hs, Ms -> host;
    # Q host -> device -> rotate (row panels) -> Psi -> host.  Wall clock around the call (it synchronises).
    e2e = None
    if do_e2e:
        need = ns * ld * 8
        avail = host_memory_available_bytes()
        ns_e = ns
        if avail is not None:
            avail = avail // world                     # every rank pins its own block
        if avail is not None and need > 0.55 * avail:
            ns_e = max(64, int(0.55 * avail // (ld * 8)) // 64 * 64)
        ns_e = min(ns, ns_e)
        refill()
        torch.cuda.synchronize()
        host_psi = torch.empty((ns_e, ld), dtype=torch.float64, pin_memory=True)
        host_src = psi[:ns_e]
        Qe = Qh if ns_e == ns else np.linalg.qr(Qh[:ns_e, :ns_e])[0]
        Q_host = torch.from_numpy(np.ascontiguousarray(Qe.T)).pin_memory()
        Hs_host = torch.empty((ns_e, ns_e), dtype=torch.float64, pin_memory=True)
        Ms_host = torch.empty_like(Hs_host).pin_memory()
        mats = torch.empty(3 * ns_e * ns_e, dtype=torch.float64, device=dev)
        e2e_times = []
        for i in range(1 + e2e_reps):
            refill()
            host_psi.copy_(host_src)                  # fresh input in host memory (outside the timer)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            g.chefsi_step_host(host_psi, Q_host, Hs_host, Ms_host, m, wl.a, wl.b, wl.a0, psi_dev=psi[:ns_e], mats_dev=mats,
                               col_block=col_block)
            if i > 0:
                e2e_times.append(time.perf_counter() - t0)
        te = torch.tensor([sum(e2e_times) / len(e2e_times)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e_s = float(te.cpu()[0])
        e2e = {"value": float(nd) * ns_e * m * world / e2e_s, "unit": UNIT,
               "h2d_bytes_per_step": ns_e * ld * 8 + ns_e * ns_e * 8, "d2h_bytes_per_step": ns_e * ld * 8 + 2 * ns_e * ns_e * 8,
               "columns": ns_e, "step_s": e2e_s, "scope": "filter+project+rotate, solve excluded",
               "what": "whole step filter+project+rotate through sparc_gpu_chefsi_step_host (C ABI, pinned host buffers, copies "
                       "overlapped, wall clock incl. final sync); subspace solve excluded (Q given); value = Nd*Ns*degree / step_s"
                       + ("" if ns_e == ns else f"; host memory bounds the sample to the first {ns_e} of {ns} columns")}
        # the same step with the subspace eigenproblem inside it (Algorithm 1 whole: sparc_gpu_chefsi_step_host_solve), where the
        # device eigensolver is in its range (one-sided Jacobi is HBM-bound past N_s ~ 2048: DESIGN.md section 6.4)
        if ns_e == ns and ns <= 2048:
            mats_s = torch.empty(3 * ns * ns + ns + 1, dtype=torch.float64, device=dev)
            ts, info = [], None
            for i in range(1 + e2e_reps):
                refill()
                host_psi.copy_(host_src)
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                _, _, info = g.chefsi_step_host_solve(host_psi, Hs_host, Ms_host, m, wl.a, wl.b, wl.a0, psi_dev=psi, mats_dev=mats_s,
                                                      col_block=col_block)
                if i > 0:
                    ts.append(time.perf_counter() - t0)
            tsv = torch.tensor([sum(ts) / len(ts)], dtype=torch.float64, device=dev)
            if world > 1:
                dist.all_reduce(tsv, op=dist.ReduceOp.MAX)
            s_s = float(tsv.cpu()[0])
            e2e["with_solve"] = {"value": float(nd) * ns * m * world / s_s, "step_s": s_s, "status": int(info[0]), "sweeps": int(info[1]),
                                 "scope": "filter+project+device eigensolve+rotate (sparc_gpu_chefsi_step_host_solve)"}
            del mats_s
        del host_psi, Q_host, Hs_host, Ms_host, mats
        if hasattr(torch._C, "_host_emptyCache"):
            torch._C._host_emptyCache()           # hand the pinned block back to the OS (the next workload sizes its own)

    # ---- rooflines: per-launch CUDA events inside the library (option "profile"), same launch configuration ----
    roofline = None
    rooflines = {}
    filter_roofs = None
    if rank == 0:
        reps = 2 if step_ms < 4000 else 1
        g.set_option("profile_reset", 1)
        g.set_option("profile", 1)
        for _ in range(reps):
            refill()
            g.chebyshev_filter(psi, m, wl.a, wl.b, wl.a0, col_block=col_block)
        torch.cuda.synchronize()
        prof_f = {k: (g.get_info(f"prof_ns:{k}"), g.get_info(f"prof_count:{k}")) for k in KINDS}
        g.set_option("profile_reset", 1)
        for _ in range(reps):
            g.project(psi, col_block=col_block, Hs=Hs, Ms=Ms)
            g.rotate(psi, Q)
        torch.cuda.synchronize()
        g.set_option("profile", 0)
        prof_s = {k: (g.get_info(f"prof_ns:{k}"), g.get_info(f"prof_count:{k}")) for k in KINDS}
        tot_f = sum(v[0] for v in prof_f.values()) or 1
        share = {KINDS[k]: round(v[0] / tot_f, 4) for k, v in prof_f.items() if v[1]}
        tot_step = tot_f + (sum(v[0] for v in prof_s.values()) or 0)
        hbm_peak, hbm_src = measured_peaks()
        if "peaks" not in env:
            env["peaks"] = (api.probe_peak(0, local_rank), api.probe_peak(1, local_rank))
        dfma_peak, dmma_peak = env["peaks"]       # TFLOP/s, register-resident DFMA / DMMA.8x8x4 chains, measured in this run
        supp_rows = float(wl.supp_idx.shape[0])
        pbar = float(wl.chi.shape[0]) / max(supp_rows, 1.0)          # mean projectors per support row

        def entry(name, bound, ns_total, n_launch, work_total, peak, unit, src, traffic=None, note=None):
            if not n_launch or not ns_total:
                return None
            ach = work_total / (ns_total * 1e-9) / (1e9 if unit == "GB/s" else 1e12)
            e = {"bound": bound, "kernel": name, "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak,
                 "traffic": traffic, "peak_source": src, "launches_timed": n_launch,
                 "avg_launch_us": ns_total / n_launch / 1e3, "alg_work_per_launch": work_total / n_launch,
                 "share_of_step": round(ns_total / tot_step, 4)}
            if note:
                e["note"] = note
            return e

        sk = 1 if prof_f[1][1] else 0
        # stencil: each column block launches 1 kernel without Prev (16 B/pt) and m-1 with Prev (24 B/pt) per call
        rooflines["stencil"] = entry(KINDS[sk], "hbm", prof_f[sk][0], prof_f[sk][1],
                                     reps * nd * ns * (16.0 + 24.0 * (m - 1)), hbm_peak, "GB/s", hbm_src,
                                     traffic=NCU_TRAFFIC_BYTES_PER_LAUNCH.get((config, "stencil")))
        # nonlocal: 2 flop x P x (pull + project) per (support row, column) and degree step; the first pass projects
        # only, the last pulls only: 2m half-passes per filter call
        nlk = 9 if prof_f[9][1] else (8 if prof_f[8][1] else None)
        if nlk is not None:
            rooflines["nonlocal"] = entry(KINDS[nlk], "tensor" if nlk == 9 else "alu", prof_f[nlk][0], prof_f[nlk][1],
                                          reps * 2.0 * m * 2.0 * supp_rows * pbar * ns,
                                          dmma_peak if nlk == 9 else dfma_peak, "TFLOP/s",
                                          "measured now (sparc_gpu_probe_peak, FP64 %s)" % ("DMMA" if nlk == 9 else "DFMA"),
                                          traffic=NCU_TRAFFIC_BYTES_PER_LAUNCH.get((config, "nonlocal")),
                                          note="algorithmic flop 4*c*P per pt*orb*deg; padding flop of partial octets not counted")
        # GEMMs: flop ISSUED, counted by the library (Hs and Ms are computed as upper-triangle tiles + mirror, reading R12,
        # so the TN kernels issue about half of the nominal 2 x 2*Nd*Ns^2; no credit for skipped work)
        rooflines["gemm_tn"] = entry("gemm_tn", "tensor", prof_s[4][0], prof_s[4][1], g.get_info("gemm_tn_mflop") * 1e6,
                                     dmma_peak, "TFLOP/s", "measured now (sparc_gpu_probe_peak, FP64 DMMA)",
                                     traffic=NCU_TRAFFIC_BYTES_PER_LAUNCH.get((config, "gemm_tn")),
                                     note="flop issued (upper-triangle tiles incl. tile padding); nominal full products: %.3e"
                                          % (reps * 2 * 2.0 * nd * ns * ns))
        rooflines["gemm_nn"] = entry("gemm_nn", "tensor", prof_s[5][0], prof_s[5][1], g.get_info("gemm_nn_mflop") * 1e6,
                                     dmma_peak, "TFLOP/s", "measured now (sparc_gpu_probe_peak, FP64 DMMA)",
                                     traffic=NCU_TRAFFIC_BYTES_PER_LAUNCH.get((config, "gemm_nn")))
        rooflines = {k: v for k, v in rooflines.items() if v}
        # the filter as a whole: 24 B and 2*(37+3) + 4*c*P flop per unit; the lower roof binds
        flop_unit = 80.0 + 4.0 * supp_rows * pbar / nd
        roof_hbm = hbm_peak * 1e9 / ALG_BYTES_PER_UNIT
        roof_fp64 = dmma_peak * 1e12 / flop_unit
        value1 = float(nd) * ns * m / (filt * 1e-3)          # one GPU's filter rate
        filter_roofs = {"flop_per_unit": flop_unit, "hbm_roof_units_per_s": roof_hbm, "fp64_roof_units_per_s": roof_fp64,
                        "binding": "hbm" if roof_hbm <= roof_fp64 else "fp64",
                        "frac_of_binding": value1 / min(roof_hbm, roof_fp64),
                        "frac_of_hbm": value1 / roof_hbm, "frac_of_fp64": value1 / roof_fp64}
        # `roofline`: the dominant kernel of the step.  The filter's two kernels (stencil + nonlocal) run as one fused
        # sequence per degree step; when together they are the largest share, the entry is the filter as a whole against
        # its binding roof.
        groups = {"filter": sum(rooflines[k]["share_of_step"] for k in ("stencil", "nonlocal") if k in rooflines)}
        for k in ("gemm_tn", "gemm_nn"):
            if k in rooflines:
                groups[k] = rooflines[k]["share_of_step"]
        top = max(groups, key=groups.get)
        if top == "filter":
            if filter_roofs["binding"] == "hbm":
                roofline = {"bound": "hbm", "kernel": "filter (stencil + nonlocal kernels)", "achieved": value1 * ALG_BYTES_PER_UNIT / 1e9,
                            "peak": hbm_peak, "unit": "GB/s", "frac": value1 / roof_hbm,
                            "traffic": None, "peak_source": hbm_src, "share_of_step": round(groups["filter"], 4)}
            else:
                roofline = {"bound": "tensor", "kernel": "filter (stencil + nonlocal kernels)", "achieved": value1 * flop_unit / 1e12,
                            "peak": dmma_peak, "unit": "TFLOP/s", "frac": value1 / roof_fp64, "traffic": None,
                            "peak_source": "measured now (sparc_gpu_probe_peak, FP64 DMMA; DFMA and DMMA share the pipe)",
                            "share_of_step": round(groups["filter"], 4)}
        else:
            roofline = dict(rooflines[top])
        roofline["step_share_by_group"] = {k: round(v, 4) for k, v in groups.items()}
        roofline["filter_time_share_by_kernel"] = share
        roofline["fp64_peaks_tflops"] = {"dfma": dfma_peak, "dmma": dmma_peak}

    # ---- CPU oracle beside it (rank 0, N = 1 only) --------------------------------------------------------
    cpu_baseline = None
    if rank == 0 and world == 1 and do_cpu:
        from oracle import oracle as orc
        orc.build()
        cores = os.cpu_count() or 1
        ncols = max(1, min(ns, cores))
        rate, dt = oracle_filter_rate(wl, ncols)
        while dt < 8.0 and ncols * 2 <= ns:
            ncols *= 2
            rate, dt = oracle_filter_rate(wl, ncols)
        cpu_baseline = {"value": rate, "unit": UNIT, "cores": cores,
                        "kind": "oracle", "detail": "oracle/chefsi_oracle.c, acc_t = double build, OpenMP over columns",
                        "sample": f"Chebyshev filter degree {m} on {ncols} of {ns} columns of {wl.name}: {dt:.1f} s"
                                  + ("" if ncols == ns else " (same per-column work as the full block: columns are independent)")}

    units = float(nd) * ns * m * world
    value = units / (filt * 1e-3)
    sub_flops = 3 * 2.0 * nd * ns * ns * world
    res = {
        "value": value, "ms_per_step": step_ms,
        "config": {"workload": wl.name, "grid": list(wl.n), "nd": nd, "ns": ns, "degree": m,
                   "atoms": wl.n_atoms, "col_block": col_block, "stencil_path": g.get_info("stencil_path_last"),
                   "parallelism": f"replicas x{world}",
                   "l2": (f"Psi block {ns * ld * 8 / 1e6:.0f} MB > 126 MB L2, regenerated between steps"
                          if l2_flush is None else "Psi block fits L2: 256 MB written between steps (flush)")},
        "hbm_gbs": value * ALG_BYTES_PER_UNIT / 1e9,
        "subspace_tflops": sub_flops / ((proj + rot) * 1e-3) / 1e12,
        "step_ms": {"filter": filt, "project": proj, "rotate": rot, "wall_per_step": t_wall / steps * 1e3},
        "steps": steps, "warmup": warmup,
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roofline, "roofline_by_kernel": rooflines, "filter_roofs": filter_roofs,
        "cpu_baseline": cpu_baseline,
    }
    g.close()
    del psi, Q, Hs, Ms, g, l2_flush
    torch.cuda.empty_cache()
    return res


def bench_shard(env, config, steps, warmup, col_block=0):
    """N > 1: ONE workload partitioned over the ranks as the paper does (dist.py): columns for the
    filter, rows for projection / rotation, an all-to-all each way and an all-reduce of Hs / Ms.  Strong scaling."""
    torch, dist, api, wlmod = env["torch"], env["dist"], env["api"], env["wlmod"]
    world, rank, local_rank, dev = env["world"], env["rank"], env["local_rank"], env["dev"]
    from paper_2302_09708_b200 import dist as pdist

    wl = wlmod.make_workload(config)
    g = api.SparcGpu(wl, device=local_rank)
    local = pdist.SparcGpuLocal(g)
    nd, ns, m = wl.nd, wl.ns, wl.degree
    cb, ce = pdist.partition(ns, world, rank)
    Xc = torch.empty((ce - cb, nd), dtype=torch.float64, device=dev)

    def refill():       # this rank's columns of the same global seeded block
        if ce > cb:
            api.fill_uniform(Xc, wl.seed, wlmod.STREAM_PSI, cb * nd, -1.0, 1.0)
    Q = api.colmajor_from_numpy(wl.q_matrix(), device=dev)
    col_block = col_block if col_block else (wl.col_block or 1024)
    names = ["start", "filter", "to_rows", "project", "solve", "rotate", "to_columns"]

    def one_step(record=None):
        refill()
        evs = {}

        def mark(name):
            if record is not None:
                e = torch.cuda.Event(enable_timing=True)
                e.record()
                evs[name] = e
        pdist.chefsi_step(local, Xc, nd, ns, m, wl.a, wl.b, wl.a0, Q=Q, col_block=col_block, timers={"mark": mark})
        if record is not None:
            record.append(evs)

    for _ in range(warmup):
        one_step()
    pdist.barrier(dev)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    launches0 = g.get_info("kernel_launches")
    rec = []
    t0 = time.perf_counter()
    for _ in range(steps):
        one_step(rec)
    pdist.barrier(dev)
    t_wall = time.perf_counter() - t0
    launches = g.get_info("kernel_launches") - launches0
    clocks = sampler.stop() if rank == 0 else None
    phase = [sum(e[names[i]].elapsed_time(e[names[i + 1]]) for e in rec) / steps for i in range(len(names) - 1)]
    phase = pdist.max_over_ranks(phase, dev)                     # slowest rank per phase
    filt = phase[0]
    step_ms = sum(phase)
    # end to end: this rank's columns from pinned host memory and back around the same step
    host = torch.empty((ce - cb, nd), dtype=torch.float64, pin_memory=True)
    refill()
    host.copy_(Xc)
    pdist.barrier(dev)
    t0 = time.perf_counter()
    Xc.copy_(host, non_blocking=True)
    pdist.chefsi_step(local, Xc, nd, ns, m, wl.a, wl.b, wl.a0, Q=Q, col_block=col_block)
    host.copy_(Xc, non_blocking=True)
    pdist.barrier(dev)
    e2e_s = pdist.max_over_ranks([time.perf_counter() - t0], dev)[0]
    units = float(nd) * ns * m
    res = {
        "value": units / (filt * 1e-3), "ms_per_step": step_ms, "scaling": "strong",
        "config": {"workload": wl.name, "grid": list(wl.n), "nd": nd, "ns": ns, "degree": m, "atoms": wl.n_atoms,
                   "col_block": col_block, "stencil_path": g.get_info("stencil_path_last"),
                   "parallelism": f"shard x{world}: filter by columns with the all-to-all of each finished block overlapped, "
                                  "project / rotate by rows, all-reduce of Hs, Ms (NCCL)",
                   "l2": "each rank's slice is larger than the 126 MB L2 and is regenerated between steps"},
        "hbm_gbs": units / (filt * 1e-3) * ALG_BYTES_PER_UNIT / 1e9,
        "subspace_tflops": 3 * 2.0 * nd * ns * ns / ((phase[2] + phase[4]) * 1e-3) / 1e12,
        "step_ms": dict(zip(["filter", "to_rows", "project", "solve", "rotate", "to_columns"], phase),
                        wall_per_step=t_wall / steps * 1e3),
        "steps": steps, "warmup": warmup, "clocks": clocks,
        "e2e": {"value": units / e2e_s, "unit": UNIT, "h2d_bytes_per_step": ns * nd * 8, "d2h_bytes_per_step": ns * nd * 8,
                "step_s": e2e_s, "scope": "filter+project+rotate, solve excluded", "what": "every rank: its columns pinned host -> device, the distributed step, device -> host"},
        "gpu_launches": int(launches), "roofline": None, "roofline_by_kernel": {}, "filter_roofs": None, "cpu_baseline": None,
    }
    g.close()
    return res


def bench_next_rows(env, config=2):
    """The SURVEY.md section 8(f) rows measured on one workload's grid and atoms (device-resident inputs, CUDA events, best of
    3 after a warm-up): gradient stencil, chi^T X, nonlocal force (NEXT-3); device eigensolve (NEXT-1); complex k-point
    filter / project / rotate (NEXT-4).  NEXT-2 is what `--gpus N` times."""
    torch, api, wlmod, dev, local_rank = env["torch"], env["api"], env["wlmod"], env["dev"], env["local_rank"]
    wl = wlmod.make_workload(config)
    g = api.SparcGpu(wl, device=local_rank)
    nd, ns = wl.nd, min(wl.ns, 1024)
    hbm_peak, hbm_src = measured_peaks()
    dmma_peak = env["peaks"][1] if "peaks" in env else api.probe_peak(1, local_rank)
    out = {"workload": wl.name, "columns": ns, "peaks": {"hbm_gbs": hbm_peak, "hbm_source": hbm_src, "dmma_tflops": dmma_peak}}

    def timed(fn, reps=3):
        fn()
        torch.cuda.synchronize()
        best = None
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            torch.cuda.synchronize()
            ms = a.elapsed_time(b)
            best = ms if best is None else min(best, ms)
        return best

    psi = torch.empty((ns, nd), dtype=torch.float64, device=dev)
    api.fill_uniform(psi, wl.seed, wlmod.STREAM_PSI, 0, -1.0, 1.0)
    Y = torch.empty_like(psi)
    supp_rows = float(wl.supp_idx.shape[0])
    pbar = float(wl.chi.shape[0]) / max(supp_rows, 1.0)
    grad = {}
    for axis in range(3):
        ms = timed(lambda: g.gradient(psi, axis, Y))
        gbs = 16.0 * nd * ns / (ms * 1e-3) / 1e9
        grad["xyz"[axis]] = {"ms": ms, "achieved": gbs, "unit": "GB/s", "peak": hbm_peak, "frac": gbs / hbm_peak, "bound": "hbm",
                             "alg_bytes_per_point": 16}
    out["gradient"] = grad
    ms = timed(lambda: g.nl_project(psi))
    out["nl_project"] = {"ms": ms, "achieved": 2.0 * supp_rows * pbar * ns / (ms * 1e-3) / 1e12, "unit": "TFLOP/s",
                         "note": "chi^T X, 2 flop per (support row, projector, column); per-atom FMA kernel"}
    occ = torch.from_numpy(wl.occupations()[:ns].copy()).to(dev)
    ms = timed(lambda: g.nonlocal_force(psi, occ))
    out["nonlocal_force"] = {"ms": ms, "orbitals_per_s": ns / (ms * 1e-3),
                             "what": "3 gradient passes + 4 projector contractions + the force contraction per column block"}
    del Y
    # NEXT-1: device eigensolve on a well-conditioned synthetic pencil of the subspace sizes of configs 1-2 (and 2048)
    eig = {}
    for n in (256, 1024, 2048):
        A = torch.empty((n, n), dtype=torch.float64, device=dev)
        api.fill_uniform(A, 77, 1, 0, -1.0, 1.0)
        Hs = (A + A.T).contiguous()
        Ms = (A @ A.T / n + torch.eye(n, dtype=torch.float64, device=dev)).contiguous()     # SPD input for the timing (torch: input generation only)
        info = []
        ms = timed(lambda: info.append(g.eigensolve(Hs, Ms)[2]), reps=2)
        st = info[-1].cpu().numpy()
        eig[str(n)] = {"ms": ms, "sweeps": int(st[1]), "status": int(st[0])}
        del A, Hs, Ms
    out["eigensolve"] = eig
    # NEXT-4: complex k-point operators, 256 complex orbitals
    nk = min(256, ns)
    g.set_kpoint((0.5 * np.pi, 0.5 * np.pi, 0.0 if wl.bc[2] else 0.5 * np.pi), wl.supp_shift)
    pk = torch.empty((nk, nd), dtype=torch.complex128, device=dev)
    api.fill_uniform(torch.view_as_real(pk), wl.seed, wlmod.STREAM_PSI, 0, -1.0, 1.0)
    m = wl.degree
    ms = timed(lambda: g.chebyshev_filter_k(pk, m, wl.a, wl.b, wl.a0), reps=2)
    units = float(nd) * nk * m
    out["kpoint_filter"] = {"ms": ms, "value": units / (ms * 1e-3), "unit": UNIT + " (complex orbitals)",
                            "achieved": 48.0 * units / (ms * 1e-3) / 1e9, "peak": hbm_peak, "frac": 48.0 * units / (ms * 1e-3) / 1e9 / hbm_peak,
                            "bound": "hbm", "alg_bytes_per_unit": 48,
                            "note": "generic one-thread-per-point complex stencil + per-atom phased projectors (first version)"}
    api.fill_uniform(torch.view_as_real(pk), wl.seed, wlmod.STREAM_PSI, 0, -1.0, 1.0)
    ms = timed(lambda: g.project_k(pk), reps=2)
    out["kpoint_project"] = {"ms": ms, "gemm_tflops_nominal": 2 * 8.0 * nd * nk * nk / (ms * 1e-3) / 1e12, "peak": dmma_peak,
                             "note": "Hs, Ms = 2 Hermitian products = 4 real TN GEMMs over 2 N_d rows (8 N_d N_s^2 flop each product) "
                                     "+ H(k) Psi; time includes the H(k) apply"}
    Qk = torch.linalg.qr(torch.randn(nk, nk, dtype=torch.complex128, device=dev))[0].contiguous()
    ms = timed(lambda: g.rotate_k(pk, Qk), reps=2)
    out["kpoint_rotate"] = {"ms": ms, "achieved": 8.0 * nd * nk * nk / (ms * 1e-3) / 1e12, "unit": "TFLOP/s", "peak": dmma_peak,
                            "frac": 8.0 * nd * nk * nk / (ms * 1e-3) / 1e12 / dmma_peak, "bound": "tensor"}
    g.close()
    del psi, pk
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        # NCCL's init lines (communicator size, NVLS / ring choice) on stderr, so that a scaling run can be checked for the
        # rank count and the transport it really used; INIT only, to keep the log short
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=dev)

    from paper_2302_09708_b200 import api, workloads as wlmod
    env = {"torch": torch, "dist": dist, "api": api, "wlmod": wlmod, "world": world, "rank": rank,
           "local_rank": local_rank, "dev": dev}

    res = None
    if (world > 1 or args.force_shard) and args.parallelism == "shard":
        try:
            res = bench_shard(env, args.config, args.steps, args.warmup, col_block=args.col_block)
        except Exception as exc:        # e.g. a collective this NCCL build refuses: every rank sees the same error and the run
            if world == 1:              # falls back to N independent replicas, saying so in `config.parallelism`
                raise
            shard_error = f"{type(exc).__name__}: {exc}"[:200]
            torch.cuda.empty_cache()
    if res is None:
        res = bench_config(env, args.config, args.steps, args.warmup, col_block=args.col_block,
                           stencil_path=args.stencil_path, stencil_stages=args.stencil_stages,
                           do_e2e=not args.no_e2e, do_cpu=not args.no_cpu)
    if world > 1 and args.parallelism == "shard" and "scaling" not in res:
        res["config"]["parallelism"] += f" (shard path failed: {shard_error})"
    # The LAST stdout line is the short headline record the driver parses (round 2's single 27 KB line was cut off by the
    # driver's tail: VERDICT r02).  Everything long -- per-kernel rooflines, the other workloads, the 8(f) rows -- goes to
    # EARLIER stdout lines ({"detail": name, ...}) and to gpurun_out/bench_detail.json, and a failure there cannot lose
    # the headline.
    detail = {"roofline_by_kernel": res["roofline_by_kernel"], "filter_roofs": res["filter_roofs"],
              "roofline_extra": {k: (res["roofline"] or {}).get(k) for k in ("step_share_by_group", "filter_time_share_by_kernel",
                                                                              "fp64_peaks_tflops", "note")},
              "e2e_what": (res["e2e"] or {}).get("what"), "cpu_baseline_detail": (res["cpu_baseline"] or {}).get("detail"),
              "clocks_full": res["clocks"], "config_full": res["config"],
              "subspace_tflops_note": "nominal 3 x 2*Nd*Ns^2 flop over (project + rotate) time; Hs and Ms are computed as "
                                      "upper-triangle tiles + mirror, so this is time-to-result, not issued flop"}

    def emit_detail(name, obj):
        if rank == 0 and obj is not None:
            print(json.dumps({"detail": name, name: obj}), flush=True)

    for k in ("roofline_by_kernel", "filter_roofs"):
        emit_detail(k, detail[k])
    # the other workloads of BASELINE.json (and the sixth, finer-mesh one), a few steps each, same measurement
    keys = ("value", "hbm_gbs", "subspace_tflops", "ms_per_step", "step_ms", "steps", "warmup", "config", "filter_roofs",
            "roofline_by_kernel", "clocks", "e2e")
    if args.per_config and world == 1:
        per_config = {str(args.config): {k: res[k] for k in keys}}
        for c in (0, 1, 2, 3, 5):
            if c == args.config:
                continue
            try:
                r = bench_config(env, c, min(args.steps, 5), max(3, min(args.warmup, 3)), do_e2e=not args.no_e2e, do_cpu=False)
                per_config[str(c)] = {k: r[k] for k in keys}
            except Exception as exc:                    # never lose the headline to a side measurement
                per_config[str(c)] = {"error": f"{type(exc).__name__}: {exc}"[:300]}
                torch.cuda.empty_cache()
            emit_detail(f"per_config_{c}", per_config[str(c)])
        detail["per_config"] = per_config
    if args.next_rows and world == 1:
        try:
            detail["next_rows"] = bench_next_rows(env, 2)
        except Exception as exc:
            detail["next_rows"] = {"error": f"{type(exc).__name__}: {exc}"[:300]}
        emit_detail("next_rows", detail["next_rows"])
    if rank == 0:
        short = lambda d, ks: None if d is None else {k: d[k] for k in ks if k in d}
        roof = short(res["roofline"], ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic", "peak_source",
                                       "launches_timed", "avg_launch_us", "alg_work_per_launch", "share_of_step"))
        fr = res["filter_roofs"] or {}
        cfg = short(res["config"], ("workload", "grid", "nd", "ns", "degree", "atoms", "col_block", "parallelism", "l2"))
        line = {
            "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
            "scaling": res.get("scaling", "weak"),
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": cfg,
            "hbm_gbs": res["hbm_gbs"],
            "subspace_tflops": res["subspace_tflops"],
            "step_ms": res["step_ms"],
            "filter_frac_of_binding": fr.get("frac_of_binding"), "filter_binding": fr.get("binding"),
            "clocks": short(res["clocks"], ("sm_mhz", "sm_min_mhz", "sm_max_mhz", "power_w_max", "samples", "reasons", "rejected")),
            "e2e": short(res["e2e"], ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "columns", "step_s", "scope", "with_solve")),
            "gpu_launches": res["gpu_launches"],
            "roofline": roof,
            "cpu_baseline": short(res["cpu_baseline"], ("value", "unit", "cores", "kind", "sample")),
        }
        for k in ("comm", "phase_ms"):                  # the shard path's extras, when present and small
            if k in res and len(json.dumps(res[k])) < 600:
                line[k] = res[k]
        try:
            out_dir = os.path.join(ROOT, "gpurun_out")
            os.makedirs(out_dir, exist_ok=True)
            with open(os.path.join(out_dir, "bench_detail.json"), "w") as f:
                json.dump({"headline": line, "detail": detail}, f, indent=1)
        except OSError:
            pass
        sys.stdout.flush()
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="workload: 0-4 = BASELINE.json configs, 5 = finer-mesh degree-33 workload")
    ap.add_argument("--col-block", type=int, default=0)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (profiling runs)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg (profiling runs)")
    ap.add_argument("--per-config", type=int, default=-1,
                    help="1: after the headline workload also time the other workloads (per_config key); default: on for the default workload")
    ap.add_argument("--next-rows", type=int, default=-1,
                    help="1: also time the SURVEY 8(f) rows (gradient / force, eigensolve, k-point operators) under `next_rows`; "
                         "default: on for the default workload")
    ap.add_argument("--parallelism", default="shard", choices=["shard", "replicas"],
                    help="N > 1: 'shard' partitions ONE workload over the ranks as the paper does (strong scaling); "
                         "'replicas' runs N independent copies (weak scaling)")
    ap.add_argument("--force-shard", action="store_true", help="take the shard code path with one rank too (testing)")
    ap.add_argument("--stencil-path", type=int, default=0, help="0 library default, 2 TMA + DFMA kernel, 3 TMA + DMMA hybrid")
    ap.add_argument("--stencil-stages", type=int, default=0, help="TMA ring depth (0 = library default)")
    args = ap.parse_args()
    if args.per_config < 0:
        args.per_config = 1 if args.config == 4 else 0
    if args.next_rows < 0:
        args.next_rows = 1 if args.config == 4 else 0
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: start the N ranks ourselves, exactly as the driver would
        import socket
        sk = socket.socket()
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
        sk.close()
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)]
                 + sys.argv[1:])
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
