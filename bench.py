#!/usr/bin/env python
"""bench.py -- the hot path of arxiv/paper_2606_24748 on B200, measured.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

One STEP = one pass of the whole hot path over one synthetic elasticity problem (BASELINE.json config 3 by default:
128^3 Q1 hex elements, 6.44 M unknowns, bs 3 -> 6, lognormal modulus, seed 3):
    y = A x (3x3)   y = P x_c (3x6)   y = P^T x (6x3)   A_c = P^T A P numeric recompute (AP = A*P, then A_c = R*AP)
Prints ONE JSON line.  `value` is the algorithmic bytes of the step (from the block format: 8*bs_r*bs_c+4 bytes per
block) divided by the step time, inputs resident in HBM; the per-operation GB/s, ms and roofline
fractions BASELINE.json's metric names are in `ops`.  `e2e` is the same metric through the C ABI's *_host calls with
host buffers (H2D of x vectors and of A's new values, D2H of y vectors and of A_c's values inside the timed region).
`cpu_baseline` is the CPU oracle (oracle/, as it stands) timed on this box's host cores on one pass of the workload.
`--impl reference` times the oracle alone (the reference arm of this tier).  N > 1 (torchrun): every rank runs its own
independent problem of the same shape (weak scaling, no data-path collective); time = max over ranks.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "blocked SpMV GB/s & PtAP-recompute ms at 128^3 elasticity, % of HBM peak"
NOMINAL_HBM_GBS = 8000.0   # the figure north_star names
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def read_traffic() -> dict:
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of each kernel, from the committed ncu --set full
    capture: profiles/ncu_traffic.csv is written by `python -m paper_2606_24748_b200.ncu_summary` (profiles/ncu_traffic.md
    names the commands)."""
    out = {}
    tp = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    try:
        for ln in open(tp).read().splitlines()[1:]:
            f = [t.strip() for t in ln.split(",")]
            if len(f) >= 2 and f[1]:
                out[f[0]] = int(float(f[1]))
    except Exception:
        pass
    return out


def bsr_bytes(M) -> int:
    return M.nnzb * (8 * M.bs_r * M.bs_c + 4) + 4 * (M.nbrows + 1)


def spmv_bytes(M) -> int:
    """nnzb*(8*bs_r*bs_c+4) + 4*(nbrows+1) + 8*bs_c*nbcols + 8*bs_r*nbrows."""
    return bsr_bytes(M) + 8 * M.bs_c * M.nbcols + 8 * M.bs_r * M.nbrows


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [t.strip() for t in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------ workload
def make_problem(cfg: int, ne: int | None = None):
    """Host matrices A (fine operator) and P (smoothed prolongator) of a BASELINE.json config (DESIGN.md recipe)."""
    from paper_2606_24748_b200 import problems as pr
    g = pr.make_generator(cfg, **({"ne": ne} if ne else {}))
    A = g.A(0)
    g.build_prolongator(0)
    return g, A, g.P(0)


def workload_name(cfg: int, A, P, ne=None) -> str:
    from paper_2606_24748_b200 import problems as pr
    base = pr.CONFIGS[cfg]["name"]
    if ne:
        base += f" [sample grid: {ne}^{pr.CONFIGS[cfg]['d']} elements, same recipe]"
    return f"{base}; {A.nbrows * A.bs_r} unknowns, nnzb(A)={A.nnzb}, nnzb(P)={P.nnzb}"


# ------------------------------------------------------------------ the oracle pass (cpu_baseline / --impl reference)
class OraclePass:
    """One pass of the hot path in the CPU oracle as it stands: spmv_fast on A, P and the explicit R = P^T, and PtAP
    form 2 (materialised AP, then R*AP); double accumulators, OpenMP over rows.  Symbolic work is done once here."""

    def __init__(self, A, P, seed: int):
        from oracle import oracle as orc
        from paper_2606_24748_b200 import problems as pr
        self.orc = orc
        self.A, self.P = A, P
        self.f2 = orc.PtapForm2(A, P)
        self.R = self.f2.R
        self.hA, self.hP, self.hR = orc._Held(A), orc._Held(P), orc._Held(self.R)
        self.x = pr.uniform(seed, pr.PURPOSE_FINE, A.nbrows * A.bs_r)
        self.xc = pr.uniform(seed, pr.PURPOSE_COARSE, P.nbcols * P.bs_c)
        self.y = np.empty(A.nbrows * A.bs_r)
        self.yc = np.empty(P.nbcols * P.bs_c)
        nb = lambda n, br, bc, rows: n * (8 * br * bc + 4) + 4 * (rows + 1)
        bAP = nb(self.f2.cap.shape[0], A.bs_r, P.bs_c, A.nbrows)
        bAc = nb(self.f2.cc.shape[0], P.bs_c, P.bs_c, P.nbcols)
        self.bytes = {"spmv_A": spmv_bytes(A), "spmv_P": spmv_bytes(P), "spmv_Pt": spmv_bytes(self.R),
                      "ptap": bsr_bytes(A) + bsr_bytes(P) + bAP + bsr_bytes(self.R) + bAP + bAc}
        self.total_bytes = sum(self.bytes.values())

    def run(self) -> dict:
        t = {}
        t0 = time.perf_counter(); self.orc.spmv_fast(self.A, self.x, self.y, held=self.hA)
        t1 = time.perf_counter(); self.orc.spmv_fast(self.P, self.xc, self.y, held=self.hP)
        t2 = time.perf_counter(); self.orc.spmv_fast(self.R, self.x, self.yc, held=self.hR)
        t3 = time.perf_counter(); self.f2.run()
        t4 = time.perf_counter()
        t["spmv_A"], t["spmv_P"], t["spmv_Pt"], t["ptap"], t["total"] = t1 - t0, t2 - t1, t3 - t2, t4 - t3, t4 - t0
        return t


def omp_threads() -> int:
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v and v.isdigit() else (os.cpu_count() or 1)


def run_reference(args) -> dict:
    """The reference arm of this tier: the oracle alone, on a bounded sample per step."""
    ne = args.ref_ne
    gen, A, P = make_problem(args.config, ne)  # gen owns the arrays A and P view
    from paper_2606_24748_b200 import problems as pr
    op = OraclePass(A, P, pr.CONFIGS[args.config]["seed"])
    for _ in range(args.warmup):
        op.run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        op.run()
    dt = time.perf_counter() - t0
    val = op.total_bytes * args.steps / dt / 1e9
    sample = f"{ne}^3-element grid of the same recipe per step (all four operations, {op.total_bytes / 1e9:.3f} GB)"
    return {"impl": "reference", "metric": METRIC, "value": val, "unit": "GB/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, A, P, ne)},
            "cpu_baseline": {"value": val, "unit": "GB/s", "cores": omp_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


# ------------------------------------------------------------------ ranks (one process per GPU, weak scaling)
def rank_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def max_over_ranks(value: float, world: int, device) -> float:
    """The job's time is the slowest rank's (every rank runs its own independent problem; no data-path collective)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(bytes_per_rank: int, world: int, seconds: float) -> float:
    """Whole-job GB/s: the units all ranks processed divided by the max-over-ranks time."""
    return bytes_per_rank * world / seconds / 1e9


# ------------------------------------------------------------------ strong scaling of ONE problem (row sharding, f3)
def run_sharded(args) -> dict | None:
    """`--sharded`: the config's problem is cut into one slab of block rows per GPU (paper_2606_24748_b200/shard.py;
    PAPER.md:111 "one rank per GPU"); a step is the same hot path, now with its exchanges (x halo, coarse halo,
    restriction reduce, cut rows of A_c) between NVLink neighbours.  value = the GLOBAL problem's algorithmic bytes
    over the slowest rank's time: strong scaling.  Each rank generates the whole problem on the host and keeps its
    slab (stand-in for a distributed assembly)."""
    import torch
    import torch.distributed as dist
    from paper_2606_24748_b200 import bsr, problems as pr, shard

    rank, world, local = rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    bsr.lib()
    cfg = args.config
    seed = pr.CONFIGS[cfg]["seed"]
    gen, A, P = make_problem(cfg)
    agg = gen.level_arrays(0)["agg"].copy()
    comm = shard.DistComm(dev) if world > 1 else shard.SoloComm()
    sh = shard.RowShard(A, P, agg, comm, shard.LibOps(dev))
    sh.ptap_symbolic()
    x = pr.uniform(seed, pr.PURPOSE_FINE, A.nbrows * A.bs_r)
    xc = pr.uniform(seed, pr.PURPOSE_COARSE, P.nbcols * P.bs_c)
    x_ext, xc_ext, yc_ext = sh.new_fine_ext(), sh.new_coarse_ext(), sh.new_coarse_ext()
    sh.fine_local(x_ext).copy_(torch.from_numpy(x[sh.r0 * A.bs_r:sh.r1 * A.bs_r]).to(dev))
    sh.coarse_local(xc_ext).copy_(torch.from_numpy(xc[sh.c0 * P.bs_c:sh.c1 * P.bs_c]).to(dev))
    y = torch.empty(sh.nloc * A.bs_r, dtype=torch.float64, device=dev)
    Rshape = pr.HostBSR(P.nbcols, P.nbrows, P.bs_c, P.bs_r, None, P.colidx, None)

    def allsum(v: int) -> int:
        if world == 1:
            return int(v)
        t = torch.tensor([v], dtype=torch.int64, device=dev)
        dist.all_reduce(t)
        return int(t.item())

    # GLOBAL algorithmic bytes (the figures of the single-GPU line): AP and A_c block counts summed over the slabs
    nnzb_ap = allsum(sh.plan.info()["nnzb_ap"])
    nnzb_c = allsum(sh.coo.nnzb)
    bAP = nnzb_ap * (8 * A.bs_r * P.bs_c + 4) + 4 * (A.nbrows + 1)
    bAc = nnzb_c * (8 * P.bs_c * P.bs_c + 4) + 4 * (P.nbcols + 1)
    nbytes = {"spmv_A": spmv_bytes(A), "spmv_P": spmv_bytes(P), "spmv_Pt": spmv_bytes(Rshape),
              "ptap_numeric": bsr_bytes(A) + bsr_bytes(P) + bAP + bsr_bytes(Rshape) + bAP + bAc}
    names = list(nbytes)

    def step(ev=None):
        if ev: ev[0].record()
        sh.spmv_A(x_ext, y)
        if ev: ev[1].record()
        sh.spmv_P(xc_ext, y)
        if ev: ev[2].record()
        sh.spmv_Pt(sh.fine_local(x_ext), yc_ext)
        if ev: ev[3].record()
        sh.ptap_numeric()
        if ev: ev[4].record()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    l0, _ = bsr.counters()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for k in range(args.steps):
        step(evs[k])
    t1.record()
    barrier()
    l1, _ = bsr.counters()
    clocks = sampler.stop()
    ms_step = max_over_ranks(t0.elapsed_time(t1), world, dev) / args.steps
    per = {n: max_over_ranks(float(np.median([evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(args.steps)])), world, dev)
           for i, n in enumerate(names)}
    sent = {k: allsum(v) for k, v in sh.exchange_bytes().items()}
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return None
    peak, peak_src = measured_peak()
    total = sum(nbytes.values())
    ops = {n: {"ms": per[n], "GB/s": nbytes[n] / (per[n] * 1e-3) / 1e9, "algorithmic_GB": nbytes[n] / 1e9,
               "frac_of_measured_hbm_x_gpus": nbytes[n] / (per[n] * 1e-3) / 1e9 / (peak * world)} for n in names}
    dom = max(names, key=lambda n: per[n])
    return {"metric": METRIC, "value": total / (ms_step * 1e-3) / 1e9, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg, A, P), "parallelism": f"row slabs x{world} (shard.py)",
                       "l2": "inputs exceed L2; no flush", "step": "y=Ax, y=Px_c, y=P^T x, ptap_numeric, with their exchanges"},
            "ops": ops, "exchange_bytes_sent_per_call_all_ranks": sent,
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": ops[dom]["GB/s"], "peak": peak * world,
                         "peak_source": peak_src + f" x {world} GPUs", "unit": "GB/s",
                         "frac": ops[dom]["GB/s"] / (peak * world), "traffic": None},
            "clocks": clocks, "gpu_launches": int(l1 - l0),
            "e2e": {"value": None, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                    "note": "the host-buffer leg is measured by the default (replica) mode"}}


# ------------------------------------------------------------------ the CUDA arm
def run_ours(args) -> dict | None:
    import torch
    import torch.distributed as dist
    from paper_2606_24748_b200 import bsr, problems as pr

    rank, world, local = rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    bsr.lib()  # fails loudly if the CUDA library cannot be built / loaded
    cfg = args.config
    seed = pr.CONFIGS[cfg]["seed"]
    gen, A, P = make_problem(cfg)
    dev = torch.device("cuda", local)
    GA, GP = bsr.Bsr.from_host(A, dev), bsr.Bsr.from_host(P, dev)
    plan = bsr.PtapPlan(GA, GP)                     # cold: symbolic + block coordinate plan
    GP.transpose_prepare()                          # cold: R = P^T cached
    info = plan.info()
    x = torch.from_numpy(pr.uniform(seed, pr.PURPOSE_FINE, A.nbrows * A.bs_r)).to(dev)
    xc = torch.from_numpy(pr.uniform(seed, pr.PURPOSE_COARSE, P.nbcols * P.bs_c)).to(dev)
    y, yc = torch.empty_like(x), torch.empty_like(xc)
    vals_c = plan.new_values()
    Rshape = pr.HostBSR(P.nbcols, P.nbrows, P.bs_c, P.bs_r, None, P.colidx, None)
    nbytes = {"spmv_A": spmv_bytes(A), "spmv_P": spmv_bytes(P), "spmv_Pt": spmv_bytes(Rshape),
              "ptap": info["algorithmic_bytes"]}
    bAP = info["nnzb_ap"] * (8 * A.bs_r * P.bs_c + 4) + 4 * (A.nbrows + 1)
    bAc = plan.nnzb_c * (8 * P.bs_c * P.bs_c + 4) + 4 * (P.nbcols + 1)
    nbytes_k = {"ptap_stage1_AP": bsr_bytes(A) + bsr_bytes(P) + bAP, "ptap_stage2_RAP": bsr_bytes(Rshape) + bAP + bAc}
    total_bytes = sum(nbytes.values())
    names = ["spmv_A", "spmv_P", "spmv_Pt", "ptap_stage1_AP", "ptap_stage2_RAP"]
    # the operator changes between repetitions ("for PtAP change A's values between repetitions"):
    # two device value buffers, A_0 and 1.25 A_0, rebound alternately (bsr_rebind_values bumps the state counter)
    a_bufs = [GA.vals, GA.vals * 1.25]
    step_no = [0]

    def step(ev=None):
        GA.rebind_values(a_bufs[step_no[0] & 1])
        step_no[0] += 1
        if ev: ev[0].record()
        GA.spmv(x, y)
        if ev: ev[1].record()
        GP.spmv(xc, y)
        if ev: ev[2].record()
        GP.spmv_t(x, yc)
        if ev: ev[3].record()
        plan.numeric_stage(1)               # AP = A*P      } together: ptap_numeric (same two launches, same gate)
        if ev: ev[4].record()
        plan.numeric_stage(2, vals_c)       # A_c = R*(AP)  }
        if ev: ev[5].record()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(6)] for _ in range(args.steps)]
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    l0, a0 = bsr.counters()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_start.record()
    for k in range(args.steps):
        step(evs[k])
    t_end.record()
    barrier()
    l1, a1 = bsr.counters()
    clocks = sampler.stop()
    ms_total = t_start.elapsed_time(t_end)
    samples = {n: [evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(args.steps)] for i, n in enumerate(names)}
    per = {n: float(np.median(v)) for n, v in samples.items()}          # median over the timed steps
    per_min = {n: float(np.min(v)) for n, v in samples.items()}
    ms_total = max_over_ranks(ms_total, world, dev)
    ms_step = ms_total / args.steps
    value = job_value(total_bytes, world, ms_step * 1e-3)
    peak, peak_src = measured_peak()

    # ---- e2e: the same step through the C ABI's host-buffer calls (pinned host memory, copies inside the timed region)
    hx = torch.from_numpy(pr.uniform(seed, pr.PURPOSE_FINE, A.nbrows * A.bs_r)).pin_memory()
    hxc = torch.from_numpy(pr.uniform(seed, pr.PURPOSE_COARSE, P.nbcols * P.bs_c)).pin_memory()
    hy, hyc = torch.empty_like(hx).pin_memory(), torch.empty_like(hxc).pin_memory()
    hvals_a = torch.from_numpy(np.ascontiguousarray(A.vals).reshape(-1)).pin_memory()
    hvals_c = torch.empty(vals_c.numel(), dtype=torch.float64).pin_memory()

    def step_host():
        GA.spmv_host(hx.numpy(), hy.numpy())
        GP.spmv_host(hxc.numpy(), hy.numpy())
        GP.spmv_host(hx.numpy(), hyc.numpy(), trans=True)
        plan.numeric_host(hvals_a.numpy(), hvals_c.numpy(), vals_c)

    h2d = 8 * (2 * hx.numel() + hxc.numel() + hvals_a.numel())
    d2h = 8 * (2 * hy.numel() + hyc.numel() + hvals_c.numel())
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    step_host()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        step_host()
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, world, dev)
    e2e_val = job_value(total_bytes * e2e_steps, world, e2e_s)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return None

    ops = {}
    for n in ["spmv_A", "spmv_P", "spmv_Pt"]:
        gbs = nbytes[n] / (per[n] * 1e-3) / 1e9
        ops[n] = {"ms": per[n], "ms_min": per_min[n], "GB/s": gbs, "algorithmic_GB": nbytes[n] / 1e9,
                  "frac_of_measured_hbm": gbs / peak, "frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS}
    ptap_ms = per["ptap_stage1_AP"] + per["ptap_stage2_RAP"]
    gbs = nbytes["ptap"] / (ptap_ms * 1e-3) / 1e9
    ops["ptap_numeric"] = {"ms": ptap_ms, "GB/s": gbs, "algorithmic_GB": nbytes["ptap"] / 1e9,
                           "frac_of_measured_hbm": gbs / peak, "frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS,
                           "stage1_ms": per["ptap_stage1_AP"], "stage2_ms": per["ptap_stage2_RAP"],
                           "ms_min": per_min["ptap_stage1_AP"] + per_min["ptap_stage2_RAP"],
                           "a_values": "alternate between A_0 and 1.25 A_0 every step (bsr_rebind_values)",
                           "GFLOP": 2.0 * (info["n_products_1"] * A.bs_r * A.bs_r * P.bs_c +
                                           info["n_products_2"] * P.bs_c * A.bs_r * P.bs_c) / 1e9}
    ops["ptap_numeric"]["fp64_TFLOPs"] = ops["ptap_numeric"]["GFLOP"] / ptap_ms
    kb = dict(nbytes); kb.update(nbytes_k)
    dom = max(names, key=lambda n: per[n])
    ach = kb[dom] / (per[dom] * 1e-3) / 1e9
    traffic_all = read_traffic()   # profiles/ncu_traffic.csv, written by paper_2606_24748_b200/ncu_summary.py
    traffic = traffic_all.get(dom)
    # the ALU roof beside the HBM roof: fp64 FMA peak measured on this device by the library
    fp64_peak = bsr.fp64_peak_tflops()
    flops_k = {"ptap_stage1_AP": 2.0 * info["n_products_1"] * A.bs_r * A.bs_r * P.bs_c,
               "ptap_stage2_RAP": 2.0 * info["n_products_2"] * P.bs_c * A.bs_r * P.bs_c}
    alu = {n: {"achieved_tflops": f / (per[n] * 1e-3) / 1e12, "peak": fp64_peak,
               "frac": f / (per[n] * 1e-3) / 1e12 / fp64_peak} for n, f in flops_k.items()}
    roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                "frac": ach / peak, "traffic": traffic, "algorithmic_bytes_per_launch": kb[dom],
                "ms_per_launch": per[dom], "share_of_step": per[dom] / sum(per.values()),
                "alu": dict(alu.get(dom, {}), unit="TFLOP/s", peak_source="bsr_measure_fp64_peak (this run)",
                            mma_peak=bsr.fp64_peak_tflops(mma=True), all_kernels=alu),
                "all_kernels": {n: {"ms": per[n], "ms_min": per_min[n], "GB/s": kb[n] / (per[n] * 1e-3) / 1e9,
                                    "frac": kb[n] / (per[n] * 1e-3) / 1e9 / peak, "traffic": traffic_all.get(n)}
                                for n in names}}
    out = {"metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
           "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_name(cfg, A, P), "l2": "inputs exceed L2 (A alone is %.2f GB); no flush" %
                      (bsr_bytes(A) / 1e9), "per_rank": "one independent problem per GPU", "step":
                      "y=Ax, y=Px_c, y=P^T x, ptap_numeric (AP=A*P; A_c=R*AP)"},
           "ops": ops, "roofline": roofline, "clocks": clocks,
           "e2e": {"value": e2e_val, "unit": "GB/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "ms_per_step": e2e_s / e2e_steps * 1e3, "steps": e2e_steps},
           "gpu_launches": int(l1 - l0), "allocs_in_timed_region": int(a1 - a0)}
    if not args.no_next_rows:
        out["next_rows"] = run_next_rows(gen, A, GA, peak)
    if not args.no_vcycle:
        # release the config-3 device arrays first (config 4 is a second, smaller problem)
        del plan, GA, GP, x, xc, y, yc, vals_c, a_bufs
        torch.cuda.empty_cache()
        out["vcycle"] = run_vcycle(peak)
    if not args.no_second_workload:
        import gc
        gc.collect(); torch.cuda.empty_cache()
        out["second_workload"] = run_second_workload(peak)
    if not args.no_cpu_baseline:
        from oracle import oracle as orc
        op = OraclePass(A, P, seed)
        t = op.run()
        ncores = orc.set_threads(0)
        out["cpu_baseline"] = {"value": op.total_bytes / t["total"] / 1e9, "unit": "GB/s", "cores": ncores,
                               "kind": "oracle", "sample": "one full pass of the same workload (all four operations)",
                               "seconds": {k: round(v, 4) for k, v in t.items()}}
        orc.set_threads(1)                                          # once with 1 thread as well
        t1 = op.run()
        orc.set_threads(0)
        out["cpu_baseline"]["one_thread"] = {"value": op.total_bytes / t1["total"] / 1e9, "unit": "GB/s", "cores": 1,
                                             "seconds": {k: round(v, 4) for k, v in t1.items()}}
    if world > 1:
        dist.destroy_process_group()
    return out


def run_next_rows(gen, A, GA, peak: float, reps: int = 10) -> dict:
    """SURVEY.md 8(f) rows f1 and f2 at the same config-3 grid: device prolongator smoothing (one pass over A) and
    the blocked COO assembly of A from 134 M finite-element block contributions; median ms of `reps`, GB/s over the
    algorithmic bytes the library reports, fraction of the measured HBM peak."""
    import torch
    from paper_2606_24748_b200 import bsr

    def timed(fn):
        for _ in range(3):
            fn()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        torch.cuda.synchronize()
        for e0, e1 in evs:
            e0.record(); fn(); e1.record()
        torch.cuda.synchronize()
        t = [e0.elapsed_time(e1) for e0, e1 in evs]
        return float(np.median(t)), float(np.min(t))

    def row(ms, ms_min, nbytes, **kw):
        gbs = nbytes / (ms * 1e-3) / 1e9
        return dict(ms=ms, ms_min=ms_min, algorithmic_GB=nbytes / 1e9, **{"GB/s": gbs}, frac_of_measured_hbm=gbs / peak,
                    frac_of_nominal_8TBs=gbs / NOMINAL_HBM_GBS, **kw)

    out = {}
    Pt = gen.P_tent(0)
    GT = bsr.Bsr.from_host(Pt, GA.vals.device)
    t0 = time.perf_counter()
    sm = bsr.ProlongatorSmoother(GA, GT)
    cold = time.perf_counter() - t0
    vals_p = sm.new_values()
    omega = gen.level_info(0)["omega"]
    ms, mn = timed(lambda: sm.numeric(omega, vals_p))
    inf = sm.info()
    out["prolongator_smooth"] = row(ms, mn, inf["algorithmic_bytes"], symbolic_s=cold, staged=inf["staged"],
                                    n_products=inf["n_products"], launches_per_call=2)
    del sm, GT, vals_p
    d, ne = gen.d, gen.ne
    E, Ke = gen.element_data()
    dev = GA.vals.device
    dKe = torch.from_numpy(Ke.reshape(-1)).to(dev)
    dE = torch.from_numpy(E).to(dev) if E is not None else None
    nel = gen.nelements
    brow, bcol = bsr.fem_q1_coords(d, ne, 0, nel, dev)
    n = (ne + 1) ** d
    t0 = time.perf_counter()
    plan = bsr.BcooPlan(brow, bcol, n, n, d, d)
    cold = time.perf_counter() - t0
    del brow, bcol
    stream = bsr.fem_q1_blocks(d, ne, 0, nel, dKe, dE, True)
    vals = plan.new_values()
    ms, mn = timed(lambda: plan.set_values(stream, vals))
    inf = plan.info()
    out["bcoo_set_values"] = row(ms, mn, inf["algorithmic_bytes"], plan_s=cold, n_contrib=inf["n_contrib"],
                                 nnzb=inf["nnzb"])
    ms, mn = timed(lambda: bsr.fem_q1_blocks(d, ne, 0, nel, dKe, dE, True, stream))
    out["fem_q1_element_blocks"] = row(ms, mn, 8 * stream.numel())
    return out


def run_second_workload(peak: float, reps: int = 10) -> dict:
    """the same hot path on the denser (config 5: Q2 elements, ~185 nonzeros per row) and the
    irregular (config 6: greedy aggregates) operator of the 65^3 node grid -- PAPER.md:206-217 finds that the block
    advantage shrinks as rows get denser; rows beyond the staged PtAP format run the gather kernels (`staged`)."""
    import torch
    from paper_2606_24748_b200 import bsr, problems as pr

    def timed(fn):
        for _ in range(3):
            fn()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        torch.cuda.synchronize()
        for e0, e1 in evs:
            e0.record(); fn(); e1.record()
        torch.cuda.synchronize()
        return float(np.median([e0.elapsed_time(e1) for e0, e1 in evs]))

    out = {}
    for cfg in (5, 6):
        gen, A, P = make_problem(cfg)
        seed = pr.CONFIGS[cfg]["seed"]
        GA, GP = bsr.Bsr.from_host(A), bsr.Bsr.from_host(P)
        plan = bsr.PtapPlan(GA, GP)
        GP.transpose_prepare()
        x = torch.from_numpy(pr.uniform(seed, pr.PURPOSE_FINE, A.nbrows * A.bs_r)).cuda()
        xc = torch.from_numpy(pr.uniform(seed, pr.PURPOSE_COARSE, P.nbcols * P.bs_c)).cuda()
        y, yc, vals_c = torch.empty_like(x), torch.empty_like(xc), plan.new_values()
        R = pr.HostBSR(P.nbcols, P.nbrows, P.bs_c, P.bs_r, None, P.colidx, None)
        ops = {}
        for name, fn, nb in (("spmv_A", lambda: GA.spmv(x, y), spmv_bytes(A)), ("spmv_P", lambda: GP.spmv(xc, y), spmv_bytes(P)),
                             ("spmv_Pt", lambda: GP.spmv_t(x, yc), spmv_bytes(R)),
                             ("ptap_numeric", lambda: plan.numeric(vals_c), plan.info()["algorithmic_bytes"])):
            ms = timed(fn)
            gbs = nb / (ms * 1e-3) / 1e9
            ops[name] = {"ms": ms, "algorithmic_GB": nb / 1e9, "GB/s": gbs, "frac_of_measured_hbm": gbs / peak}
        sched = plan.schedule()
        ops["ptap_numeric"]["staged"] = [bool(sched[1]["staged"]), bool(sched[2]["staged"])]
        out[f"cfg{cfg}"] = {"workload": workload_name(cfg, A, P), "nnz_per_row": A.nnzb * A.bs_c / A.nbrows,
                            "max_blocks_per_row": {"A": int(np.diff(A.rowptr).max()), "P": int(np.diff(P.rowptr).max()),
                                                   "A_c": int(np.diff(plan.rowptr_c.cpu().numpy()).max())},
                            "l2": "A is %.2f GB (exceeds L2)" % (bsr_bytes(A) / 1e9), "ops": ops}
        del plan, GA, GP, x, xc, y, yc, vals_c
        torch.cuda.empty_cache()
    return out


def run_vcycle(peak: float, cfg: int = 4, reps: int = 10) -> dict:
    """BASELINE.json's third number: V-cycle ms at config 4 (96^3, three levels, V(2,2) degree-2 Chebyshev / block
    Jacobi, dense coarsest solve), plus the full hierarchy recompute and one PCG iteration.  The hierarchy is built
    through the library (two ptap plans); the generator only needs the level-1 operator back on the host to form the
    level-2 prolongator (cold setup)."""
    import torch
    from paper_2606_24748_b200 import bsr, problems as pr
    g = pr.make_generator(cfg)
    g.build_prolongator(0)
    A0, P0 = g.A(0), g.P(0)
    G0, GP0 = bsr.Bsr.from_host(A0), bsr.Bsr.from_host(P0)
    plan0 = bsr.PtapPlan(G0, GP0)
    v1 = plan0.numeric()
    A1 = pr.HostBSR(plan0.nbrows_c, plan0.nbrows_c, P0.bs_c, P0.bs_c, plan0.rowptr_c.cpu().numpy(),
                    plan0.colidx_c.cpu().numpy(), v1.cpu().numpy().reshape(-1, P0.bs_c, P0.bs_c))
    g.set_operator(1, A1)
    g.build_prolongator(1)
    P1 = g.P(1)
    G1, GP1 = plan0.coarse_matrix(v1), bsr.Bsr.from_host(P1)
    plan1 = bsr.PtapPlan(G1, GP1)
    v2 = plan1.numeric()
    G2 = plan1.coarse_matrix(v2)
    lams = [g.level_info(0)["lam"], g.level_info(1)["lam"]]
    vc = bsr.VCycle([G0, G1, G2], [GP0, GP1], lams)
    b = torch.from_numpy(pr.uniform(pr.CONFIGS[cfg]["seed"], pr.PURPOSE_RHS, A0.nbrows * A0.bs_r)).cuda()
    xv = torch.empty_like(b)

    def timed(fn, n):
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    ms_v = timed(lambda: vc.apply(b, xv), reps)

    def recompute():
        plan0.numeric(v1); plan1.numeric(v2); vc.refresh(check=False)
    ms_r = timed(recompute, 3)
    ms_pcg = timed(lambda: vc.pcg(b, 5), 2) / 5
    # algorithmic bytes of one application: per non-coarsest level 4 A-SpMVs + restriction +
    # prolongation and four reads of D^-1, plus the two triangular sweeps of the dense coarsest solve
    nbytes = 0
    for Al, Pl in ((A0, P0), (A1, P1)):
        Rl = pr.HostBSR(Pl.nbcols, Pl.nbrows, Pl.bs_c, Pl.bs_r, None, Pl.colidx, None)
        nbytes += 4 * spmv_bytes(Al) + spmv_bytes(Pl) + spmv_bytes(Rl) + 4 * 8 * Al.nbrows * Al.bs_r * Al.bs_r
    nc = plan1.nbrows_c * P1.bs_c
    nbytes += 8 * nc * nc
    gbs = nbytes / (ms_v * 1e-3) / 1e9
    return {"workload": pr.CONFIGS[cfg]["name"], "vcycle_ms": ms_v, "algorithmic_GB": nbytes / 1e9, "GB/s": gbs,
            "frac_of_measured_hbm": gbs / peak, "frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS,
            "hierarchy_recompute_ms": ms_r, "pcg_iteration_ms": ms_pcg, "coarsest_unknowns": nc}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config (3 = the 128^3 headline grid)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-ne", type=int, default=64, help="sample grid of the reference arm (elements per side)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-vcycle", action="store_true", help="skip the config-4 V-cycle timing")
    ap.add_argument("--sharded", action="store_true", help="strong-scale ONE problem over the ranks (row slabs, "
                    "paper_2606_24748_b200/shard.py) instead of one independent problem per rank")
    ap.add_argument("--no-second-workload", action="store_true", help="skip the f4 timings (configs 5 and 6)")
    ap.add_argument("--no-next-rows", action="store_true", help="skip the f1 / f2 timings (prolongator smoothing, "
                    "blocked COO assembly)")
    args = ap.parse_args()
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        print(json.dumps(run_reference(args)), flush=True)
        return
    out = run_sharded(args) if args.sharded else run_ours(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
