#!/usr/bin/env python
"""bench.py — H_eff.psi FP64 throughput at the middle bond (BASELINE.json `metric`).

  python bench.py --gpus N --steps K --warmup W [--config C] [--impl reference]

One "step" is one H_eff.psi (Eq. (7)/(8)) on the two-site problem of BASELINE.json
configs[C] (default C = 3, the U(1)xU(1) D = 4096 problem the north_star target is quoted on; it fits
one GPU).  The line also carries ms per Davidson iteration and one renormalisation step (the other
rows of SURVEY.md 8(a)), the roofline object, the end-to-end number through the host-buffer C call,
and the CPU oracle timed on a bounded sample.  N > 1: replicas only (the path does not shard,
DESIGN.md "Multi-GPU"): every rank runs the same problem on its own GPU, no data-path collective.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores.
"""
from __future__ import annotations

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

METRIC = "heff_apply_fp64_gflops"
UNIT = "GFLOP/s"


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _host_threads():
    try:
        import threadpoolctl
        info = threadpoolctl.threadpool_info()
        return int(max(p["num_threads"] for p in info)) if info else int(os.cpu_count())
    except Exception:
        return int(os.cpu_count())


def time_oracle_sample(d, T, V, mps, psi0, steps, warmup, nblocks=10, max_elems=9000):
    """The CPU oracle (oracle/lean.py: the oracle's own formulas restricted to chosen output blocks) on a BOUNDED
    sample of output blocks of the bench configuration, in the SAME analytic flop count as the GPU line: the flops
    of a block are those of the library's task list for that block (dmrg_block_flops).

    The oracle's block operators at this size cannot be built by the oracle itself in minutes (37 min at D = 4096),
    so they are read from the library's environments (dmrg_env_export_block) BEFORE the timed region, exactly as in
    tests/test_gpu_lean_parity.py, which checks them against the oracle; forming the complementary operators of the
    sampled blocks is setup (the GPU's task-list build is not timed either).  Timed: the oracle's contraction loop
    `_accumulate` (psi' blocks = sum over terms of mL psi mR^T) for the sampled blocks."""
    import importlib.util
    from oracle import dmrg as odmrg
    from oracle import lean
    from paper_2501_18263_b200 import inputs
    spec = importlib.util.spec_from_file_location("lean_helpers", os.path.join(ROOT, "tests", "lean_helpers.py"))
    lh = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(lh)
    pb = inputs.psi_blocks(mps)
    bf = d.block_flops()
    N, k, L = (mps.n_up, mps.n_dn), mps.k, mps.L
    # a fixed spread of block sizes: every 1/nblocks quantile of the blocks below max_elems, by analytic flops
    cand = sorted((i for i in range(len(pb)) if 64 <= pb[i][4] * pb[i][5] <= max_elems), key=lambda i: bf[i])
    if not cand:
        cand = sorted(range(len(pb)), key=lambda i: bf[i])
    idxs = sorted({cand[min(len(cand) - 1, int((q + 0.5) / nblocks * len(cand)))] for q in range(nblocks)})
    Ls = lh.ExportedSide(d, 0, range(0, k - 1), mps.sectors[k - 1], N)
    Rs = lh.ExportedSide(d, 1, range(k + 1, L), {odmrg.qsub(N, q): dim for q, dim in mps.sectors[k + 1].items()}, N)
    qL = {pb[i][0] for i in idxs}
    qR = {odmrg.qsub(N, pb[i][3]) for i in idxs}
    orc = lean.LeanTwoSiteOracle(T, V, mps.n_up, mps.n_dn, k, pb, Ls.block(qL, L), Rs.block(qR, L))
    psi = orc.unflatten(np.asarray(psi0, dtype=np.float64))
    keys = [orc.block_key(i) for i in idxs]
    terms = orc.terms({kk[0] for kk in keys}, {kk[1] for kk in keys})

    def one_pass():
        out = {kk: np.zeros_like(psi[kk]) for kk in keys}
        orc._accumulate(terms, psi, out)
        return out
    for _ in range(warmup):
        one_pass()
    t0 = time.perf_counter()
    for _ in range(steps):
        one_pass()
    dt = (time.perf_counter() - t0) / max(steps, 1)
    flops = float(sum(bf[i] for i in idxs))
    # the same products through the oracle's plain C + OpenMP loop (oracle/cproducts.c: two triple loops per product, no
    # BLAS), list of products gathered before the timed region
    c_line = None
    try:
        from oracle import clevel
        pl = clevel.ProductList(terms, psi, {kk: np.zeros_like(psi[kk]) for kk in keys})
        ref = one_pass()
        got = pl.run()
        err = max(float(np.abs(got[kk] - ref[kk]).max()) / max(1.0, float(np.abs(ref[kk]).max())) for kk in keys)
        t1 = time.perf_counter()
        for _ in range(steps):
            pl.run()
        dtc = (time.perf_counter() - t1) / max(steps, 1)
        c_line = {"value": flops / dtc * 1e-9, "unit": UNIT, "cores": int(os.cpu_count()), "kind": "oracle, contraction loop in "
                  "plain C + OpenMP (oracle/cproducts.c), same sample and flop count", "ms_per_pass": dtc * 1e3,
                  "max_rel_dev_from_numpy_loop": err}
    except Exception as e:      # no C compiler on the box: the numpy figure stands alone
        c_line = {"unavailable": str(e)[:200]}
    return {"value": flops / dt * 1e-9, "unit": UNIT, "cores": _host_threads(), "kind": "oracle",
            "sample": "the bench configuration itself: %d of its %d psi' output blocks (dims %s), %.3f %% of the analytic flops of one "
                      "H_eff.psi, %.2f s of oracle time per pass; flops = the library's task-list count for those blocks "
                      "(dmrg_block_flops), operator blocks exported from the library's environments before the timed region"
                      % (len(idxs), len(pb), ", ".join("%dx%d" % (pb[i][4], pb[i][5]) for i in idxs),
                         100.0 * flops / float(bf.sum()), dt),
            "ms_per_apply": dt * 1e3, "sample_flops": flops, "apply_flops": float(bf.sum()), "c_openmp": c_line}


def _workload(cfg, mps, n_up, n_dn, su2, D):
    return ("BASELINE configs[%d]: L=%d, N=(%d,%d), %s, D=%d%s, middle bond (%d,%d), one H_eff.psi per step"
            % (cfg, mps.L, n_up, n_dn, "SU(2) S=0" if su2 else "U(1)xU(1)", D, " multiplets" if su2 else "", mps.k, mps.k + 1))


def run_reference(args):
    """`--impl reference`: the CPU oracle on the bench configuration (a bounded sample of its output blocks per step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    from paper_2501_18263_b200 import inputs
    from paper_2501_18263_b200.binding import DMRG
    cfg = args.config
    if args.su2 or cfg == 4:
        raise SystemExit("--impl reference: U(1)xU(1) configurations only")
    c = inputs.CONFIGS[cfg]
    D = args.D if args.D else c["D"]
    T, V, mps = inputs.make_config(cfg, D=D)
    psi0 = inputs.make_psi0(mps, c["seed"])
    # the library only supplies the oracle's INPUTS here (the operator blocks of the two environments); see time_oracle_sample
    d = DMRG(mps.L, mps.n_up, mps.n_dn, device=int(os.environ.get("LOCAL_RANK", "0")))
    d.setup(T, V, mps)
    cb = time_oracle_sample(d, T, V, mps, psi0, max(args.steps, 1), min(args.warmup, 3))
    d.close()
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": cb["ms_per_apply"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": _workload(cfg, mps, mps.n_up, mps.n_dn, False, D) + "; CPU oracle, each step a bounded "
                                   "sample of that workload: " + cb["sample"]},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2501_18263_b200 import inputs, replicas
    from paper_2501_18263_b200.binding import DMRG

    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    rank, world = replicas.init("nccl", torch.device("cuda", local))

    cfg = args.config
    su2 = args.su2 or cfg == 4          # config 4 exists in SU(2) form only (BASELINE.json configs[4])
    c = inputs.SU2_CONFIGS[cfg] if su2 else inputs.CONFIGS[cfg]
    D = args.D if args.D else c["D"]
    t0 = time.perf_counter()
    dev = torch.device("cuda", local)
    if su2:
        T, V, mps = inputs.make_config_su2(cfg, D=D)
        n_up = n_dn = mps.N // 2
        psi0 = inputs.make_psi0_su2(mps, c["seed"])
    else:
        T, V, mps = inputs.make_config(cfg, D=D)
        n_up, n_dn = mps.n_up, mps.n_dn
        psi0 = inputs.make_psi0(mps, c["seed"])
    d = DMRG(mps.L, n_up, n_dn, device=local, workspace_bytes=args.workspace_gb << 30, su2=su2)
    d.setup(T, V, mps)
    job_flops = None
    if args.shard and world > 1:
        # strong scaling: the psi' blocks of ONE problem dealt to the ranks, one all-reduce (NCCL) per apply
        from paper_2501_18263_b200 import sharded
        sharded.shard_over_ranks(d)
        d.env_build(mps.k)          # environments come from the cache; only the task list is rebuilt
        job_flops = float(d.shard_info()[1].sum())
    torch.cuda.synchronize()
    setup_s = time.perf_counter() - t0
    st = d.stats()
    n = d.psi_size()
    x = torch.from_numpy(psi0).to(dev)
    y = torch.empty_like(x)
    peak_tf = d.fp64_peak()
    dfma_tf = d.dfma_peak()
    # cuBLAS DGEMM 8192^3 through torch: a yardstick for the FP64 tensor pipe, never on the product path
    ga = torch.randn(8192, 8192, dtype=torch.float64, device=dev)
    gb = torch.randn(8192, 8192, dtype=torch.float64, device=dev)
    torch.matmul(ga, gb)
    ge0, ge1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ge0.record()
    for _ in range(3):
        torch.matmul(ga, gb)
    ge1.record()
    torch.cuda.synchronize()
    dgemm_tf = 3 * 2.0 * 8192.0 ** 3 / (ge0.elapsed_time(ge1) * 1e-3) * 1e-12
    del ga, gb
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        hbm_peak = 6650.0   # fallback of /opt/skills/guides/B200_PROFILING.md

    def barrier():
        replicas.barrier(world)
        torch.cuda.synchronize()

    # ---- device-resident: K applies, each timed with its own CUDA events on the launching stream.  At
    # configs 2-4 the operator working set (GBs) is far larger than the 126 MB L2; at configs 0-1 it fits,
    # so a buffer larger than L2 is rewritten between timed steps (outside the events).
    op_bytes = st["op_bytes_left"] + st["op_bytes_right"]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if op_bytes < (512 << 20) else None
    for _ in range(args.warmup):
        d.heff_apply(x, y)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = d.stats()["total_launches"]
    torch.cuda.profiler.start()     # no-op unless run under ncu --profile-from-start off
    evs = []
    for _ in range(args.steps):
        if flush is not None:
            flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        d.heff_apply(x, y)
        e1.record()
        evs.append((e0, e1))
    barrier()
    torch.cuda.profiler.stop()
    clocks = sampler.stop()
    launches = d.stats()["total_launches"] - l0
    ms = sum(a.elapsed_time(b) for a, b in evs) / args.steps
    ms_max, fl_per_s = replicas.aggregate_throughput(st["flops_apply"], ms, world, dev)
    if job_flops is not None:
        fl_per_s = job_flops / (ms_max * 1e-3)
    value = fl_per_s * 1e-9

    # ---- the dominant kernel alone: every launch of one more apply bracketed by events (serial order)
    _, rec = d.apply_profile(x, y)
    dom = {}
    for r in rec:
        if r["shape"] == 8 and r["phase"] < 3:
            a = dom.setdefault(r["phase"], [0, 0.0, 0.0])
            a[0] += 1; a[1] += r["flops"]; a[2] += r["ms"]
    tot_ms = sum(r["ms"] for r in rec) or 1.0
    # every tile shape, serialised: {"<phase>:<rows>x<cols>": [ms, TFLOP/s]} (shape = 3 * row class + col class)
    per_shape = {}
    for r in rec:
        if 0 <= r["shape"] < 9 and r["flops"] > 0:
            if r["phase"] == 3:      # fused small-sector kernel: shape = N / 8 - 1 of the output blocks
                key = "fused:N=%d" % (8 * (r["shape"] + 1))
            else:
                key = "%d:%dx%d" % (r["phase"], (32, 64, 128)[r["shape"] // 3], (32, 64, 128)[r["shape"] % 3])
            a = per_shape.setdefault(key, [0.0, 0.0])
            a[0] += r["ms"]; a[1] += r["flops"]
    per_shape = {k: [round(v[0], 3), round(v[1] / v[0] * 1e-9, 2)] for k, v in sorted(per_shape.items()) if v[0] > 0}
    dominant = {"kernel": "k_grouped_gemm<128,128> (tile shape 128x128)",
                "share_of_serial_step": sum(v[2] for v in dom.values()) / tot_ms,
                "serial_ms_and_tflops_per_shape": per_shape,
                "per_phase": {str(k): {"launches": v[0], "avg_ms": v[2] / v[0], "flops_per_launch": v[1] / v[0],
                                       "tflops": v[1] / v[2] * 1e-9} for k, v in dom.items() if v[0]}}
    dom_fl = sum(v[1] for v in dom.values())
    dom_ms = sum(v[2] for v in dom.values())

    # ---- end to end through the host-buffer C call (pinned host psi in, psi out)
    hx = torch.from_numpy(psi0.copy()).pin_memory()
    hy = torch.empty_like(hx).pin_memory()
    hxn, hyn = hx.numpy(), hy.numpy()
    d.heff_apply_host(hxn, hyn)
    barrier()
    t1 = time.perf_counter()
    esteps = max(1, min(args.steps, 5))
    for _ in range(esteps):
        d.heff_apply_host(hxn, hyn)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t1) / esteps * 1e3
    e2e_max, e2e_fl = replicas.aggregate_throughput(st["flops_apply"], e2e_ms, world, dev)
    if job_flops is not None:
        e2e_fl = job_flops / (e2e_max * 1e-3)
    e2e_val = e2e_fl * 1e-9

    # the CPU oracle on a sample of this configuration's output blocks (needs the environments of THIS bond: before
    # the renormalisation step below moves the context to the next one)
    cpu_line = None
    if rank == 0 and world == 1 and not args.no_cpu and not su2:
        cpu_line = time_oracle_sample(d, T, V, mps, psi0, 2, 1)
    extra = {}
    if (rank == 0 or job_flops is not None) and not args.quick:    # sharded: Davidson runs in lock-step on all ranks
        # ---- Davidson: fixed 10 iterations from the random start vector
        dg = d.heff_diag()      # start: lowest diagonal element + 1 % random (R20)
        z = 0.01 * x
        z[int(torch.argmin(dg))] += 1.0
        z /= torch.linalg.norm(z)
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        E, it, rn = d.davidson(z, tol=1e-30, max_iter=10, max_basis=12)
        torch.cuda.synchronize()
        extra["davidson"] = {"iters": it, "ms_per_iter": (time.perf_counter() - t2) * 1e3 / it, "energy": E, "resid": rn}
        extra["env_build"] = {"setup_s": setup_s, "last_build_ms": st["last_build_ms"],
                              "last_renorm_step_gflop": st["flops_renorm"] * 1e-9}
        if cfg <= 3 and not su2 and job_flops is None:
            # BASELINE configs[2]: Davidson to 1e-8 and one operator-renormalisation step (site k joins the left block)
            if cfg <= 2:
                z2 = 0.01 * x
                z2[int(torch.argmin(dg))] += 1.0
                z2 /= torch.linalg.norm(z2)
                t3 = time.perf_counter()
                E2, it2, rn2 = d.davidson(z2, tol=1e-8, max_iter=400, max_basis=20)
                torch.cuda.synchronize()
                extra["davidson_1e-8"] = {"iters": it2, "ms_total": (time.perf_counter() - t3) * 1e3, "energy": E2, "resid": rn2}
            d.mps_set_site(mps.k, 0, inputs.make_left_site(mps.sectors, mps.k, c["seed"]))
            d.renormalize(0)
            torch.cuda.synchronize()
            s2 = d.stats()
            extra["renormalize_step"] = {"ms": s2["renorm_ms"], "gflop": s2["flops_renorm"] * 1e-9,
                                         "tflops": s2["flops_renorm"] / (s2["renorm_ms"] * 1e-3) * 1e-12,
                                         "includes": "host planning of the step + all launches + sync; first call: "
                                                     "the caller's allocator has no cached block for the workspace",
                                         "call_wall_ms": s2["last_build_ms"]}
            # the same step in the state a sweep sees: one step back (site k+2 is still right-canonical), then again
            d.renormalize(1)
            d.mps_set_site(mps.k, 0, inputs.make_left_site(mps.sectors, mps.k, c["seed"]))
            d.renormalize(0)
            torch.cuda.synchronize()
            s3 = d.stats()
            extra["renormalize_step"].update({
                "ms_steady": s3["renorm_ms"], "tflops_steady": s3["flops_renorm"] / (s3["renorm_ms"] * 1e-3) * 1e-12,
                "call_wall_ms_steady": s3["last_build_ms"],
                "call_wall_includes": "dmrg_renormalize as a sweep calls it: blocking step + task list, complementary "
                                      "operators and diagonal of the next two-site problem"})

    # DRAM bytes per launch of the dominant kernel: written next to the committed ncu --set full summary of this
    # workload (profiles/gemm128_traffic.json, dram__bytes_read.sum + dram__bytes_write.sum); default config only.
    traffic_detail, traffic = None, None
    if cfg == 3 and not su2 and not args.D:
        try:
            tj = json.load(open(os.path.join(ROOT, "profiles", "gemm128_traffic.json")))
            per = [l["dram_read_bytes"] + l["dram_write_bytes"] for l in tj["launches"]]
            traffic_detail = {"bytes_per_launch": per, "source": tj["source"]}
            traffic = sum(per) / len(per)
        except Exception:
            pass
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_max, "higher_is_better": True,
                "scaling": "strong" if job_flops is not None else "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": "BASELINE configs[%d]: L=%d, N=(%d,%d), %s, D=%d%s, middle bond (%d,%d), "
                                       "one H_eff.psi per step" % (cfg, mps.L, n_up, n_dn,
                                                                   "SU(2) S=0" if su2 else "U(1)xU(1)", D,
                                                                   " multiplets" if su2 else "", mps.k, mps.k + 1),
                           "psi_size": n, "terms": st["n_terms"], "tasks": st["n_tasks"],
                           "flops_per_apply": job_flops if job_flops is not None else st["flops_apply"], "operator_bytes": st["op_bytes_left"] + st["op_bytes_right"],
                           "l2": ("256 MB buffer rewritten between timed steps" if flush is not None
                                  else "operator working set (%.1f GB) >> 126 MB L2, no flush" % (op_bytes / 1e9)),
                           "workspace_chunks": st["n_chunks"], "parallelism": ("psi'-block shards of one problem + one all-reduce per apply" if job_flops is not None
                                           else "replicas" if world > 1 else "single")},
                "clocks": clocks,
                "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 8 * n, "d2h_bytes_per_step": 8 * n,
                        "ms_per_step": e2e_max},
                "gpu_launches": int(launches),
                "roofline": {"bound": "tensor", "achieved": value / world * 1e-3, "peak": peak_tf, "unit": "TFLOP/s",
                             "frac": value / world * 1e-3 / peak_tf, "traffic": traffic,
                             "what": "whole H_eff.psi: analytic task-list flops / event time of the step (all "
                                     "k_grouped_gemm launches of the step, run on the library's worker streams)",
                             "peak_source": "FP64 tensor-pipe (DMMA m8n8k4) register-only loop measured in this run "
                                            "(dmrg_fp64_peak) = 148 SM x 128 flop/clk x SM clock; MEASURED_PEAKS.json "
                                            "has no FP64 entry",
                             "comparison_peaks": {"dmma_loop_tflops": peak_tf, "dfma_loop_tflops": dfma_tf,
                                                  "cublas_dgemm_8192_tflops": dgemm_tf,
                                                  "frac_of_dfma_loop": value / world * 1e-3 / dfma_tf,
                                                  "frac_of_cublas_dgemm": value / world * 1e-3 / dgemm_tf},
                             "dominant_kernel": dict(dominant, achieved=(dom_fl / dom_ms * 1e-9 if dom_ms else None),
                                                     frac=(dom_fl / dom_ms * 1e-9 / peak_tf if dom_ms else None),
                                                     traffic=traffic_detail),
                             "hbm": {"unique_bytes_per_apply": st["bytes_unique"],
                                     "intermediate_bytes_per_apply": st["bytes_intermediate"],
                                     "achieved_gbs": (st["bytes_unique"] + st["bytes_intermediate"]) / (ms_max * 1e-3) * 1e-9,
                                     "peak_gbs": hbm_peak},
                             "flops_executed_per_apply": st["flops_executed"]},
                }
        line.update(extra)
        if cpu_line is not None:
            line["cpu_baseline"] = cpu_line
        print(json.dumps(line))
    d.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--D", type=int, default=0)
    ap.add_argument("--su2", action="store_true", help="SU(2)-adapted form of the config (configs 3 and 4)")
    ap.add_argument("--workspace-gb", type=int, default=0, dest="workspace_gb", help="0 = library default")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--quick", action="store_true", help="skip the Davidson / renormalisation extras")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: shard ONE problem's psi' blocks over the ranks (strong scaling) instead of N replicas")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
