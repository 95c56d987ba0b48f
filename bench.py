#!/usr/bin/env python
"""bench.py -- the hot path of arxiv/paper_2606_09200 on B200: GEMM overlapped with a collective stand-in.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cb-ar|mb-ar|cb-a2a|mb-a2a|tiny] [--impl ours|reference]
                    [--per-config all|none]

One "step" = one pass of the whole hot path over one batch of seeded synthetic
input: n_iters pipelined iterations of  K_g^i (tcgen05 GEMM)  ||  K_c^i (allreduce / alltoall stand-in)
under the occupancy / priority setting the sweep (S7) picked during warm-up.  Default workload =
BASELINE.json configs[1] ("cb-ar": GEMM 8192^3 bf16 + allreduce emul P=8 x 16Mi fp32).

Prints ONE JSON line (rank 0).  value = overlapped iterations per second over all GPUs (replicas only:
the path does not shard).  The line also carries serial/overlap/ratio, per-kernel
TFLOP/s and GB/s against MEASURED_PEAKS.json, the combined roofline, `roofline`, `cpu_baseline`, `e2e`, and
-- at N = 1 -- `per_config`: the same protocol on the other four BASELINE.json configs (Tiny, mb-ar, cb-a2a,
mb-a2a with its reserve x budget x priority sweep), each also flattened to one string under `config` so that
a parser which keeps only scalars still sees all five.

Timing protocol.  The K timed steps run at exactly the picked setting with NO per-kernel events (so the
CUDA-graph mode the policy picks for launch-bound steps is honoured); the per-kernel split, the overlap rate
and the dominant kernel's launch time come from an instrumented pass of the same K steps right after it.
The in-place allreduce buffers are refilled from pristine device copies before every run (outside the
timed window), so every iteration reduces finite, full-entropy data.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import ra_inputs  # noqa: E402  (seeded input generator; holds none of the method's arithmetic)

METRIC = "GEMM+collective overlap time vs serial; GEMM TFLOP/s; collective HBM GB/s"
UNIT = "iter/s"
PAPER_CONTEXT = ("paper: up to 25.5% execution-time reduction (priority vs baseline overlap, cb-ar on A40; "
                 "platforms A40/A100/H100/MI250X, PAPER.md:7,122) -- context, not the target")
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "source": "measured"}
    return dict(FALLBACK_PEAKS, source="fallback")


def get_config(name: str):
    for c in ra_inputs.CONFIGS:
        if c.name == name:
            return c
    raise SystemExit(f"unknown config {name}")


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.tmp = None

    def start(self):
        try:
            self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(self.gpu)], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.tmp.flush()
        self.tmp.seek(0)
        sm, mx, reasons, power = [], [], set(), []
        for line in self.tmp.read().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
                power.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.tmp.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(power), power_w_mean=sum(power) / len(power))
        return out


# ------------------------------------------------------------------------------------------------
def host_inputs(cfg, pinned: bool):
    """Seeded synthetic host buffers for one batch (DESIGN.md input recipe).  bf16 as uint16 bits."""
    import torch
    A, B = ra_inputs.gemm_operands(cfg)
    h = {"A": torch.from_numpy(A.view(np.int16)), "B": torch.from_numpy(B.view(np.int16))}
    if cfg.coll == "allreduce":
        h["ar"] = [torch.from_numpy(b) for b in ra_inputs.allreduce_buffers(cfg)]
    else:
        h["a2a"] = torch.from_numpy(ra_inputs.alltoall_payload(cfg).view(np.int64))
    if pinned:
        h["A"], h["B"] = h["A"].pin_memory(), h["B"].pin_memory()
        if "ar" in h:
            h["ar"] = [t.pin_memory() for t in h["ar"]]
        else:
            h["a2a"] = h["a2a"].pin_memory()
    return h


def device_state(ra, cfg, h, pristine=True):
    import torch
    d = {"A": h["A"].cuda(), "B": h["B"].cuda(),
         "C": torch.empty((cfg.M, cfg.N), dtype=torch.int16, device="cuda")}
    budgets = sorted({0, 74, 92, 110, 128, 140, 148})
    wsb = max(ra.ra_gemm_workspace_bytes(0, 1, cfg.M, cfg.N, cfg.K, dict(sm_budget=b)) for b in budgets)
    d["ws"] = torch.empty(max(wsb, 16), dtype=torch.uint8, device="cuda")
    if cfg.coll == "allreduce":
        d["ar"] = [t.cuda() for t in h["ar"]]
        d["ar_pristine"] = [t.cuda() for t in h["ar"]] if pristine else None
    else:
        d["a2a_a"] = h["a2a"].cuda()
        d["a2a_b"] = torch.empty_like(d["a2a_a"])
    return d


def make_workload(ra, cfg, d, n_iters, gemm=True, coll=True):
    g = dict(M=cfg.M, N=cfg.N, K=cfg.K, A=d["A"], B=d["B"], C=d["C"], workspace=d["ws"]) if gemm else None
    kw = {}
    if coll and cfg.coll == "allreduce":
        kw["allreduce"] = d["ar"]
        kw["ar_pristine"] = d.get("ar_pristine")     # the library refills the rank buffers before every run
    elif coll:
        kw["alltoall"] = dict(a=d["a2a_a"], b=d["a2a_b"], P=cfg.P, chunk_bytes=cfg.chunk_bytes)
    return ra.make_workload(gemm=g, n_iters=n_iters, **kw)


def check_finite(cfg, d, where: str):
    """The in-place allreduce multiplies magnitudes by P per iteration (8^20 ~ 1e18 over one step: finite in fp32); the
    library refills the buffers from the pristine copies before every run.  A saturated buffer here means that broke."""
    import torch
    if cfg.coll == "allreduce":
        t = d["ar"][0]
        assert bool(torch.isfinite(t).all()) and float(t.abs().max()) > 0.0, f"allreduce buffers saturated after {where}"


def sweep_candidates(ra, cfg, quick: bool):
    """S7 grid: (smem_reserve_bytes, sm_budget, priority on/off[, coll_sm_budget]).  BASELINE.json config 5:
    reserve 0-200 KB, budget 74-148, priority on/off."""
    info = ra.ra_device_info()
    hi = info["prio_greatest"]
    KB = 1024
    if quick:
        reserves, budgets = (0, 64 * KB), (148, 128, 110)
    else:
        reserves, budgets = (0, 32 * KB, 64 * KB, 96 * KB, 128 * KB, 160 * KB, 200 * KB), (74, 92, 110, 128, 140, 148)
    cands = []
    for r in reserves:
        for b in budgets:
            for prio in (0, hi):
                # collective SM budget: the SMs the GEMM leaves free, or -- with the GEMM on every SM -- a throttled
                # collective on 24-48 SMs that still finishes inside the GEMM's time but disturbs fewer SMs
                for csb in sorted({0, info["sm_count"] - b} if b < info["sm_count"] else ({0, 24, 32, 48} if r == 0 else {0})):
                    base = dict(mode=1, occ=dict(smem_reserve_bytes=r, sm_budget=b), prio_compute=0, prio_comm=prio, coll_sm_budget=csb)
                    # both collectives have a shared-memory-free LDG/STG variant (co-resides on a full GEMM SM) and a TMA-ring
                    # variant whose ring must fit somewhere: INSIDE the reserve (ring + 1 KiB system + barriers) or on SMs
                    # the GEMM leaves free; the alltoall also has the copy engines (no SM residency at all)
                    tma, ldg = (0, 1) if cfg.coll == "alltoall" else (1, 0)
                    if r >= 20 * KB:
                        cands.append(dict(base, coll_variant=tma, coll_smem_bytes=min(r - 4 * KB, 64 * KB), coll_ctas_per_sm=1))
                    elif b < info["sm_count"] or cfg.M <= 128:
                        cands.append(dict(base, coll_variant=tma))
                    cands.append(dict(base, coll_variant=ldg))
                    if csb == 0 and (cfg.coll == "alltoall" or (r == 0 and b == info["sm_count"])):
                        cands.append(dict(base, coll_variant=2))       # copy engines: all of the alltoall / the allreduce's fan-out
    if cfg.M > 128:
        # L2 as the traded resource: the GEMM keeps an X panel in a persisting carve-out of 1/8 .. 5/8 of the L2 (less DRAM
        # traffic, less energy) and the collective streams through what is left (slower alone, but it is the hidden kernel)
        MiB = 1 << 20
        for pb in (15 * MiB, 31 * MiB, 47 * MiB, 79 * MiB):
            for variant in ((0, 1, 2) if cfg.coll == "alltoall" and not quick else (1 if cfg.coll == "alltoall" else 0,)):
                cands.append(dict(mode=1, occ=dict(l2_persist_bytes=pb), prio_compute=0, prio_comm=0, coll_sm_budget=0, coll_variant=variant))
    return cands


def cfg_label(kw):
    o = kw.get("occ", {})
    return {"smem_reserve_bytes": o.get("smem_reserve_bytes", 0), "sm_budget": o.get("sm_budget", 0),
            "tiles_per_cta": o.get("tiles_per_cta", 0), "priority": "on" if kw.get("prio_comm", 0) != kw.get("prio_compute", 0) else "off",
            "coll_sm_budget": kw.get("coll_sm_budget", 0), "coll_smem_bytes": kw.get("coll_smem_bytes", 0),
            "coll_variant": kw.get("coll_variant", 0), "coll_ctas_per_sm": kw.get("coll_ctas_per_sm", 0),
            "use_graph": kw.get("use_graph", 0), "l2_persist_bytes": o.get("l2_persist_bytes", 0)}


def residency_map(ra, w, cfg_kw, n_sms):
    """Per-SM residency during one overlapped step, from the library's %smid/%globaltimer trace
    (ra_set_trace): every CTA of every kernel logs {kernel id, SM, start, end}.  Evidence for co-residency:
    how much of the collective's CTA-time ran on an SM that hosted a GEMM CTA at the same instant."""
    import torch
    cap = 1 << 16
    buf = torch.from_numpy(np.zeros(1 + 4 * cap, dtype=np.int64)).cuda()    # H2D memcpy, no torch fill kernel
    ra.ra_set_trace(buf, cap)
    try:
        ra.ra_overlap_run(w, ra.make_cfg(**cfg_kw))
        torch.cuda.synchronize()
    finally:
        ra.ra_set_trace(None, 0)
    hbuf = buf.cpu().numpy().view(np.uint64)
    n = int(min(int(hbuf[0]), cap))
    rec = hbuf[1:1 + 4 * n].reshape(n, 4)
    kid = (rec[:, 0] >> np.uint64(32)).astype(np.int64)
    sm = (rec[:, 0] & np.uint64(0xFFFFFFFF)).astype(np.int64)
    t0, t1 = rec[:, 2].astype(np.int64), rec[:, 3].astype(np.int64)
    g, c = kid == 1, kid != 1
    out = {"records": n, "gemm_ctas": int(g.sum()), "coll_ctas": int(c.sum()),
           "gemm_sms_used": int(len(set(sm[g]))), "coll_sms_used": int(len(set(sm[c])))}
    co, tot = 0, 0
    per_sm_g = {}
    for s_, a, b in zip(sm[g], t0[g], t1[g]):
        per_sm_g.setdefault(int(s_), []).append((int(a), int(b)))
    for s_, a, b in zip(sm[c], t0[c], t1[c]):
        tot += int(b - a)
        for (ga, gb) in per_sm_g.get(int(s_), ()):
            lo, hi = max(a, ga), min(b, gb)
            if hi > lo:
                co += int(hi - lo)
    out["coll_cta_time_coresident_with_gemm_frac"] = (co / tot) if tot else None
    span = (t1.max() - t0.min()) if n else 0
    out["gemm_sm_busy_frac"] = float((t1[g] - t0[g]).sum() / (span * n_sms)) if span else None
    out["coll_mean_cta_us"] = float((t1[c] - t0[c]).mean() / 1e3) if c.any() else None
    return out


def library_gemm_same_box(cfg, d, n_iters):
    """Yardstick only (never on the product path): the library GEMM (cuBLAS through torch.matmul) on the SAME box, same operands,
    same two protocols as our kernel -- best of 10 single launches, and 6 x n_iters back to back.  MEASURED_PEAKS.json was taken on
    whichever box the driver used; boxes of the pool differ by ~4 %, so this is the like-for-like reference."""
    import torch
    A = d["A"].view(torch.bfloat16)
    B = d["B"].view(torch.bfloat16)
    C = torch.empty((cfg.M, cfg.N), dtype=torch.bfloat16, device="cuda")
    fn = lambda: torch.matmul(A, B.t(), out=C)
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    burst = []
    for _ in range(10):
        time.sleep(0.05)
        e0, e1 = torch.cuda.Event(True), torch.cuda.Event(True)
        e0.record(); fn(); e1.record(); torch.cuda.synchronize()
        burst.append(e0.elapsed_time(e1))
    runs = []
    for r in range(6):
        e0, e1 = torch.cuda.Event(True), torch.cuda.Event(True)
        e0.record()
        for _ in range(n_iters):
            fn()
        e1.record(); torch.cuda.synchronize()
        runs.append(e0.elapsed_time(e1) / n_iters)
    sus = statistics.mean(runs[2:])
    return {"what": "torch.matmul (cuBLAS) bf16, same operands, same box", "burst_ms": min(burst), "burst_tflops": cfg.gemm_flops / min(burst) / 1e9,
            "sustained_ms": sus, "sustained_tflops": cfg.gemm_flops / sus / 1e9}


def kernels_alone(ra, cfg, d, peaks, n_iters, graph: int = 0):
    """Each kernel by itself (CUDA events inside the library, on the stream the kernel runs on)."""
    out = {}
    # burst: single launches with idle gaps, best of 10 (how MEASURED_PEAKS.json's burst figure was taken)
    w1, keep1 = make_workload(ra, cfg, d, 1, coll=False)
    burst = []
    for _ in range(12):
        time.sleep(0.05)
        burst.append(ra.ra_overlap_run(w1, ra.make_cfg(mode=0))["total_ms"])
    gb_ms = min(burst[2:])
    out["gemm_ms_burst"] = gb_ms
    out["gemm_tflops_burst"] = cfg.gemm_flops / gb_ms / 1e9
    out["gemm_frac_of_bf16_peak_burst"] = out["gemm_tflops_burst"] / peaks["bf16_tflops"]
    # sustained: back-to-back launches (power-capped regime)
    w, keep = make_workload(ra, cfg, d, n_iters, coll=False)
    res, _ = ra.ra_overlap_sweep(w, [ra.make_cfg(mode=0, use_graph=graph)], runs=6)
    g_ms = res[0]["total_ms"] / n_iters
    out["gemm_ms"] = g_ms
    out["gemm_tflops"] = cfg.gemm_flops / g_ms / 1e9
    out["gemm_frac_of_bf16_peak_sustained"] = out["gemm_tflops"] / peaks["bf16_tflops_sustained"]
    out["gemm_gbs"] = cfg.gemm_bytes / g_ms / 1e6
    out["gemm_frac_of_hbm_peak"] = out["gemm_gbs"] / peaks["hbm_gbs"]
    out["gemm_plan"] = res[0]["plan"]
    if cfg.M * cfg.N >= 1 << 20:
        out["library_gemm_same_box"] = library_gemm_same_box(cfg, d, n_iters)
    w, keep = make_workload(ra, cfg, d, n_iters, gemm=False)
    # the collective alone is a bandwidth measurement: let the clocks recover from the power-capped GEMM runs first
    import torch
    torch.cuda.synchronize()
    time.sleep(0.5)
    res, _ = ra.ra_overlap_sweep(w, [ra.make_cfg(mode=0, use_graph=graph)], runs=6)
    c_ms = res[0]["total_ms"] / n_iters
    out["coll_ms"] = c_ms
    out["coll_gbs"] = cfg.coll_bytes / c_ms / 1e6
    out["coll_frac_of_hbm_peak"] = out["coll_gbs"] / peaks["hbm_gbs"]
    return out


# ------------------------------------------------------------------------------------------------
_ORACLE_INPUTS = {}


def _oracle_inputs(cfg):
    if cfg.name not in _ORACLE_INPUTS:       # input generation is not part of what is timed
        _ORACLE_INPUTS.clear()               # one workload's operands at a time (8192 x 57344 alone is 1.9 GB)
        _ORACLE_INPUTS[cfg.name] = ra_inputs.gemm_operands(cfg)
    return _ORACLE_INPUTS[cfg.name]


def _oracle_collective_pass(cfg):
    """One full pass of the collective's oracle over the config's buffers; seconds."""
    import oracle
    if cfg.coll == "allreduce":
        bufs = ra_inputs.allreduce_buffers(cfg)
        t0 = time.perf_counter()
        oracle.allreduce(bufs)
        return time.perf_counter() - t0
    send = ra_inputs.alltoall_payload(cfg)
    t0 = time.perf_counter()
    oracle.alltoall(send, cfg.P, cfg.chunk_bytes)
    return time.perf_counter() - t0


def _oracle_gemm_calibrate(cfg, n0: int = 2048):
    """Seconds per C entry of oracle.gemm_samples (each entry = the full K-length fp64 dot product)."""
    import oracle
    A, B = _oracle_inputs(cfg)
    rng = np.random.default_rng(cfg.seed)
    ii, jj = rng.integers(0, cfg.M, n0), rng.integers(0, cfg.N, n0)
    oracle.gemm_samples(0, 1, cfg.M, cfg.N, cfg.K, 1.0, A, B, ii[:64], jj[:64])       # page the operands in
    t0 = time.perf_counter()
    oracle.gemm_samples(0, 1, cfg.M, cfg.N, cfg.K, 1.0, A, B, ii, jj)
    return (time.perf_counter() - t0) / n0


def cpu_oracle_full(cfg, full_limit_s: float = 90.0, sample_budget_s: float = 15.0):
    """cpu_baseline: the oracle as it stands, on the host cores.  One iteration of the hot path = oracle.gemm over the
    whole problem + one oracle pass of the collective.  The GEMM is TIMED IN FULL (one oracle.gemm call over all M x N
    entries) whenever a calibration run puts it under `full_limit_s`; only larger shapes (8192 x 57344 x 8192) fall back
    to oracle.gemm_samples on a bounded random sample, extrapolated by M*N/n and labelled as such.
    Returns (seconds per iteration, description, cores, 'full' | 'sampled')."""
    import oracle
    A, B = _oracle_inputs(cfg)
    per_entry = _oracle_gemm_calibrate(cfg)
    est = per_entry * cfg.M * cfg.N
    t_coll = _oracle_collective_pass(cfg)
    if est <= full_limit_s:
        t0 = time.perf_counter()
        oracle.gemm(0, 1, cfg.M, cfg.N, cfg.K, 1.0, A, B)
        t_gemm = time.perf_counter() - t0
        desc = (f"full: oracle.gemm over all {cfg.M}x{cfg.N} C entries (K={cfg.K}), timed once: {t_gemm:.2f} s "
                f"(calibration predicted {est:.1f} s) + one full oracle {cfg.coll} pass ({t_coll * 1e3:.0f} ms); serial sum")
        return t_gemm + t_coll, desc, oracle.num_threads(), "full"
    rng = np.random.default_rng(cfg.seed + 1)
    n = int(min(cfg.M * cfg.N, max(2048, sample_budget_s / per_entry)))
    ii, jj = rng.integers(0, cfg.M, n), rng.integers(0, cfg.N, n)
    t0 = time.perf_counter()
    oracle.gemm_samples(0, 1, cfg.M, cfg.N, cfg.K, 1.0, A, B, ii, jj)
    t_s = time.perf_counter() - t0
    t_gemm = t_s * (cfg.M * cfg.N / n)
    desc = (f"sampled: oracle.gemm_samples on {n} of {cfg.M * cfg.N} C entries (K={cfg.K} each, {t_s:.2f} s, extrapolated "
            f"x{cfg.M * cfg.N / n:.1f} -> {t_gemm:.1f} s; a full pass would exceed {full_limit_s:.0f} s) + one full oracle "
            f"{cfg.coll} pass ({t_coll * 1e3:.0f} ms); serial sum")
    return t_gemm + t_coll, desc, oracle.num_threads(), "sampled"


def run_reference(args, cfg):
    """--impl reference: the CPU oracle is the reference arm of this tier (there is no reference code).

    A step of this arm is a BOUNDED SAMPLE of one iteration of the workload: oracle.gemm_samples on a fixed fraction f
    of the C entries (each the full K-length fp64 dot product) plus the same fraction of the collective's oracle pass
    (allreduce: the first f*count elements of every rank buffer; alltoall: f of each chunk).  ms_per_step is the time
    that step really took; value = f / t_step, i.e. iterations per second at the sampled rate.  f is sized once, from a
    calibration run, so that warmup + steps fit in `--ref-budget-s` seconds."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    A, B = _oracle_inputs(cfg)
    n_steps = args.warmup + args.steps
    per_entry = _oracle_gemm_calibrate(cfg)
    t_coll_full = _oracle_collective_pass(cfg)
    t_iter_est = per_entry * cfg.M * cfg.N + t_coll_full
    f = min(1.0, (args.ref_budget_s / max(n_steps, 1)) / t_iter_est)
    n = max(64, int(f * cfg.M * cfg.N))
    f = n / (cfg.M * cfg.N)
    rng = np.random.default_rng(cfg.seed + 2)
    ii, jj = rng.integers(0, cfg.M, n), rng.integers(0, cfg.N, n)
    if cfg.coll == "allreduce":
        cnt = max(4, int(f * cfg.ar_count))
        bufs0 = [b[:cnt].copy() for b in ra_inputs.allreduce_buffers(cfg)]
    else:
        cb = max(16, int(f * cfg.chunk_bytes) // 16 * 16)
        send = ra_inputs.alltoall_payload(cfg, chunk_bytes=cb)
    times = []
    for s in range(n_steps):
        if cfg.coll == "allreduce":
            bufs = [b.copy() for b in bufs0]
        t0 = time.perf_counter()
        oracle.gemm_samples(0, 1, cfg.M, cfg.N, cfg.K, 1.0, A, B, ii, jj)
        if cfg.coll == "allreduce":
            oracle.allreduce(bufs)
        else:
            oracle.alltoall(send, cfg.P, cb)
        dt = time.perf_counter() - t0
        if s >= args.warmup:
            times.append(dt)
    t = statistics.mean(times)
    v = f / t
    cores = oracle.num_threads()
    desc = (f"each step = fraction f={f:.5f} of one iteration: oracle.gemm_samples on {n} of {cfg.M * cfg.N} C entries "
            f"(K={cfg.K} each) + the same fraction of the oracle {cfg.coll} pass; {t:.3f} s per step measured; "
            f"value = f / t (a full iteration at this rate: {t / f:.1f} s)")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "gemm": [cfg.M, cfg.N, cfg.K], "collective": cfg.coll, "P": cfg.P,
                       "iterations_per_step": f, "step": "bounded sample of one iteration (see cpu_baseline.sample)"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def dist_setup(n_gpus: int):
    """Replicas only (the path does not shard): torch.distributed is used for the barrier and max-over-ranks."""
    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if torch.cuda.is_available():
        torch.cuda.set_device(local % max(torch.cuda.device_count(), 1))
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group(backend="nccl" if torch.cuda.is_available() else "gloo")
    return world, rank, local


def max_over_ranks(x: float, world: int, device) -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier(world: int):
    import torch
    if torch.cuda.is_available():
        torch.cuda.synchronize()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    if torch.cuda.is_available():
        torch.cuda.synchronize()


def self_launch(argv, n: int) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start the N ranks ourselves (one process per
    GPU, rendezvous on 127.0.0.1) and pass their output through."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    return subprocess.call(cmd)


# ------------------------------------------------------------------------------------------------
def config5_grid(ra, cfg):
    """BASELINE.json configs[4]: 'sweep smem_reserve 0-200 KB, SM budget 74-148, priority on/off' -- the corners and
    midpoints of the full grid (bench.py --config mb-a2a --sweep full runs all 7 x 6 x 2), sized for ~1 minute."""
    info = ra.ra_device_info()
    hi, KB = info["prio_greatest"], 1024
    cands = []
    for r in (0, 64 * KB, 128 * KB, 200 * KB):
        for b in (74, 110, 148):
            for prio in (0, hi):
                base = dict(mode=1, occ=dict(smem_reserve_bytes=r, sm_budget=b), prio_compute=0, prio_comm=prio)
                if r >= 20 * KB:      # TMA ring sized into the reserve, one ring CTA per SM
                    cands.append(dict(base, coll_variant=0, coll_smem_bytes=min(r - 4 * KB, 64 * KB), coll_ctas_per_sm=1))
                else:
                    cands.append(dict(base, coll_variant=0))
                cands.append(dict(base, coll_variant=1))                         # LDG/STG, no shared memory
                if b < info["sm_count"]:                                          # collective on the SMs the GEMM leaves free
                    cands.append(dict(base, coll_variant=0, coll_sm_budget=info["sm_count"] - b))
    cands.append(dict(mode=1, coll_variant=2))                                   # copy engines
    return cands


def sweep_marginals(cand_kws, results, n_iters):
    """Best overlap time per reserve, per budget, and priority on / off at otherwise equal settings (Norm. time)."""
    by_r, by_b, pairs = {}, {}, {}
    for kw, r in zip(cand_kws, results):
        if kw.get("mode") != 1:
            continue
        lab, ms = cfg_label(kw), r["total_ms"] / n_iters
        rk, bk = lab["smem_reserve_bytes"] // 1024, lab["sm_budget"] or 148
        by_r[rk] = min(by_r.get(rk, 1e30), ms)
        by_b[bk] = min(by_b.get(bk, 1e30), ms)
        key = tuple(sorted((k, v) for k, v in lab.items() if k != "priority"))
        pairs.setdefault(key, {})[lab["priority"]] = ms
    norm = [p["on"] / p["off"] for p in pairs.values() if "on" in p and "off" in p]
    return {"best_ms_by_reserve_kb": {str(k): round(v, 4) for k, v in sorted(by_r.items())},
            "best_ms_by_sm_budget": {str(k): round(v, 4) for k, v in sorted(by_b.items())},
            "norm_time_priority_on_over_off": {"n_pairs": len(norm), "min": min(norm) if norm else None,
                                               "median": statistics.median(norm) if norm else None,
                                               "max": max(norm) if norm else None}}


def measure_config(ra, cfg, args, peaks, world, dev, headline: bool):
    """The whole protocol on one workload: warm-up, S7 (sweep + pick, the model's pick inside it), each kernel alone,
    K timed steps at the picked setting (no per-kernel events), the same K steps serial, an instrumented pass for the
    per-kernel split / overlap rate; for the headline workload also the residency trace and the e2e leg."""
    import torch
    n_iters = args.n_iters or cfg.n_iters
    steps = args.steps
    h = host_inputs(cfg, pinned=headline)
    d = device_state(ra, cfg, h)
    torch.cuda.synchronize()
    info = ra.ra_device_info()

    # ---- W plain steps, then S7 (sweep + pick; the serial schedule is one of the settings) ----
    w, keep = make_workload(ra, cfg, d, n_iters)
    for _ in range(max(args.warmup, 3)):
        ra.ra_overlap_run(w, ra.make_cfg(mode=1))
    sweep = args.sweep if headline or args.sweep in ("none", "auto") else ("config5" if cfg.name == "mb-a2a" else "quick")
    if sweep in ("none", "auto"):
        cands = []
    elif sweep == "config5":
        cands = config5_grid(ra, cfg)
    else:
        cands = sweep_candidates(ra, cfg, quick=(sweep == "quick"))
    if sweep == "auto":       # the library's own short list: model pick + neighbours (ra_overlap_autotune)
        auto_cfg, _, _ = ra.ra_overlap_autotune(w, peaks["bf16_tflops_sustained"], peaks["hbm_gbs"], runs=args.sweep_runs)
        cands = [ra.cfg_to_kw(auto_cfg)]
    # S7': the model-based policy's pick runs inside the same sweep so that its regret is measured, not assumed
    sug = ra.ra_overlap_suggest(w, peaks["bf16_tflops_sustained"], peaks["hbm_gbs"])
    graph = int(sug["kw"].get("use_graph", 0))            # launch-bound workload (Tiny): every candidate is graph-replayed
    if graph:
        cands = [dict(kw, use_graph=1) for kw in cands]
    cand_kws = [dict(mode=0, use_graph=graph)] + [dict(mode=1, use_graph=graph)] + [sug["kw"]] + cands
    runs = args.sweep_runs if sweep != "config5" else max(6, args.sweep_runs - 3)
    results, best = ra.ra_overlap_sweep(w, [ra.make_cfg(**kw) for kw in cand_kws], runs=runs)
    sweep_argmin = best
    # Final: the sweep's three fastest overlap settings and the policy's pick (index 2) are timed again with the paper's own
    # protocol -- 30 runs each, the first third warm-up -- because the minimum over ~50 settings of a noisy
    # quantity (a power-capped step wanders by 2-3 % over tenths of a second) is biased low.  Argmin of the final; settings
    # within 2.5 % of the policy's are a tie and the tie goes to the policy, so that the timed setting is not chosen by noise.
    final = None
    if sweep != "none" and len(cand_kws) > 4:
        order = sorted((i for i, kw in enumerate(cand_kws) if kw["mode"] == 1), key=lambda i: results[i]["total_ms"])
        finalists = list(dict.fromkeys(order[:3] + [2]))
        fres, fbest = ra.ra_overlap_sweep(w, [ra.make_cfg(**cand_kws[i]) for i in finalists], runs=30)
        best = finalists[fbest]
        pol_ms = fres[finalists.index(2)]["total_ms"]
        if pol_ms <= 1.025 * fres[fbest]["total_ms"]:
            best = 2
        final = {"settings": [cfg_label(cand_kws[i]) for i in finalists], "ms_per_iter": [r["total_ms"] / n_iters for r in fres],
                 "runs": 30, "picked": finalists.index(best)}
        for i, r in zip(finalists, fres):
            results[i] = dict(results[i], total_ms=r["total_ms"], median_ms=r["median_ms"], min_ms=r["min_ms"])
    elif sweep != "none" and results[2]["total_ms"] <= 1.025 * results[best]["total_ms"]:
        best = 2
    best_kw = cand_kws[best]
    sweep_serial_ms = results[0]["total_ms"] / n_iters
    sweep_table = [dict(cfg_label(kw), mode=kw["mode"], ms_per_iter=r["total_ms"] / n_iters, median=r["median_ms"] / n_iters,
                        min=r["min_ms"] / n_iters, stages=r["plan"]["stages"], tile_n=r["plan"]["tile_n"], grid=r["plan"]["grid"])
                   for kw, r in zip(cand_kws, results)]
    # priority on vs off at the best occupancy setting ("Norm. time")
    norm_time = None
    lab = cfg_label(best_kw)
    for kw, r in zip(cand_kws, results):
        l2 = cfg_label(kw)
        if kw["mode"] == 1 and all(l2[k] == lab[k] for k in lab if k != "priority") and l2["priority"] != lab["priority"]:
            on, off = (results[best]["total_ms"], r["total_ms"]) if lab["priority"] == "on" else (r["total_ms"], results[best]["total_ms"])
            norm_time = on / off
    policy = {"setting": cfg_label(sug["kw"]), "predicted_ms_per_iter": sug["t_overlap_ms"], "measured_ms_per_iter": results[2]["total_ms"] / n_iters,
              "sweep_best_ms_per_iter": results[sweep_argmin]["total_ms"] / n_iters, "sweep_argmin_setting": cfg_label(cand_kws[sweep_argmin]),
              "regret": results[2]["total_ms"] / results[best]["total_ms"] - 1.0, "final": final,
              "timed_setting_is": "policy (tie within 2.5 %)" if best == 2 and sweep_argmin != 2 else ("policy" if best == 2 else "sweep final argmin"), "gemm_bound": sug["gemm_bound"],
              "model_roofline_ms": sug["t_roofline_ms"], "settings_in_sweep": len(cand_kws) - 1}
    alone = kernels_alone(ra, cfg, d, peaks, n_iters, graph=graph)
    residency = residency_map(ra, w, best_kw, info["sm_count"])
    residency_ring = None
    if cfg.coll == "alltoall" and cfg.M * cfg.N >= 1 << 20:
        # the collective whose co-residency DEPENDS on the reserve: one TMA-ring alltoall CTA per SM (64 KiB ring) living inside
        # the shared memory a 72 KiB smem_reserve_bytes makes the GEMM leave free
        residency_ring = residency_map(ra, w, dict(mode=1, occ=dict(smem_reserve_bytes=72 * 1024), coll_variant=0, coll_smem_bytes=64 * 1024,
                                                   coll_ctas_per_sm=1, prio_compute=0, prio_comm=info["prio_greatest"]), info["sm_count"])

    # ---- timed region: exactly K steps of the overlapped hot path at exactly the picked setting ----
    best_cfg = ra.make_cfg(**best_kw)
    # W untimed warm-up steps at the picked setting IMMEDIATELY before the timed ones: the timed steps then start in the
    # clock / power state the step itself sustains, not in the one the stand-alone collective timing above left behind
    for _ in range(max(args.warmup, 3)):
        ra.ra_overlap_run(w, best_cfg)
    ra.ra_gemm_residency(reset=True)
    sampler = ClockSampler(torch.cuda.current_device())
    barrier(world)
    sampler.start()
    t_wall0 = time.perf_counter()
    step_ms = []
    for _ in range(steps):
        r = ra.ra_overlap_run(w, best_cfg)          # synchronous; total_ms from CUDA events on its own streams
        step_ms.append(r["total_ms"])
    barrier(world)
    wall_ms = (time.perf_counter() - t_wall0) * 1e3
    clocks = sampler.stop()
    plan = r["plan"]
    check_finite(cfg, d, "the timed region")
    max_resident = ra.ra_gemm_residency()
    dev_ms_total = max_over_ranks(sum(step_ms), world, dev)
    ms_per_step = dev_ms_total / steps
    over_ms = ms_per_step / n_iters

    # instrumented pass (not part of `value`): the same K steps with an event pair around every kernel, on the stream
    # the kernel is launched on -> per-kernel launch time inside the overlapped step, overlap rate
    inst_cfg = ra.make_cfg(**dict(best_kw, record_kernel_times=1))
    g_ms, c_ms, orate, inst_ms = [], [], [], []
    for _ in range(steps):
        r = ra.ra_overlap_run(w, inst_cfg)
        g_ms.append(r["gemm_ms_sum"] / n_iters)
        c_ms.append(r["coll_ms_sum"] / n_iters)
        orate.append(r["overlap_rate"])
        inst_ms.append(r["total_ms"] / n_iters)
    # serial schedule at the same setting, same protocol (TimeRatio = t_overlap / t_sequential)
    ser_cfg = ra.make_cfg(**dict(best_kw, mode=0))
    ser = [ra.ra_overlap_run(w, ser_cfg)["total_ms"] for _ in range(steps)]
    serial_ms = statistics.mean(ser) / n_iters
    check_finite(cfg, d, "the serial pass")

    flops, gbytes, cbytes = cfg.gemm_flops, cfg.gemm_bytes, cfg.coll_bytes
    compute_bound = flops / (peaks["bf16_tflops"] * 1e12) > gbytes / (peaks["hbm_gbs"] * 1e9)
    comb = {k: max(flops / (peaks[k] * 1e9), (gbytes + cbytes) / (peaks["hbm_gbs"] * 1e6)) for k in ("bf16_tflops", "bf16_tflops_sustained")}
    gemm_in_step_ms = statistics.mean(g_ms)
    coll_launches = 0 if (cfg.coll == "alltoall" and best_kw.get("coll_variant", 0) == 2) else 1
    out = {
        "workload": cfg.name, "gemm": [cfg.M, cfg.N, cfg.K], "collective": cfg.coll, "P": cfg.P, "n_iters_per_step": n_iters,
        "steps": steps, "ms_per_step": ms_per_step, "value": world * n_iters * steps / (dev_ms_total / 1e3),
        "overlap_ms_per_iter": over_ms, "serial_ms_per_iter": serial_ms, "sweep_serial_ms_per_iter": sweep_serial_ms,
        "time_ratio_same": over_ms / serial_ms, "time_ratio_best": over_ms / (alone["gemm_ms"] + alone["coll_ms"]),
        "norm_time_priority": norm_time, "overlap_rate": statistics.mean(orate),
        "gemm_in_step_ms": gemm_in_step_ms, "coll_in_step_ms": statistics.mean(c_ms),
        "instrumented_ms_per_iter": statistics.mean(inst_ms),
        "alone": alone, "combined_roofline_ms": {"burst": comb["bf16_tflops"], "sustained": comb["bf16_tflops_sustained"]},
        "overlap_vs_roofline": {"burst": over_ms / comb["bf16_tflops"], "sustained": over_ms / comb["bf16_tflops_sustained"]},
        "best_setting": cfg_label(best_kw), "plan": plan, "sweep": sweep, "policy": policy, "clocks": clocks,
        "gemm_max_ctas_on_one_sm": max_resident, "wall_ms_timed_region": wall_ms,
        "gpu_launches": steps * n_iters * (1 + coll_launches), "compute_bound": compute_bound,
    }
    if sweep == "config5":
        out["sweep_marginals"] = sweep_marginals(cand_kws, results, n_iters)
    if residency is not None:
        out["residency"] = residency
    if residency_ring is not None:
        out["residency_tma_ring_in_72k_reserve"] = residency_ring
    if args.table and headline:
        with open(args.table, "w") as f:
            json.dump(sweep_table, f, indent=1)

    if headline:
        # ---- e2e: the same steps through the C ABI's host-buffer entry point (ra_overlap_run_host): every step copies
        # its inputs from pinned host memory and its results back; the library pipelines H2D(s+1) || compute(s) || D2H(s-1)
        # over two device buffer sets.  Timed by the host clock around the one synchronous call.
        hC = torch.empty((cfg.M, cfg.N), dtype=torch.int16).pin_memory()
        h_out = (torch.empty_like(h["ar"][0]) if cfg.coll == "allreduce" else torch.empty_like(h["a2a"])).pin_memory()
        h2d = h["A"].numel() * 2 + h["B"].numel() * 2 + (sum(t.numel() * 4 for t in h["ar"]) if cfg.coll == "allreduce" else h["a2a"].numel() * 8)
        d2h = hC.numel() * 2 + h_out.numel() * h_out.element_size()
        e2e_cfg = ra.make_cfg(**dict(best_kw, use_graph=0))      # host-buffer steps are enqueued directly, not graph-replayed
        d2 = device_state(ra, cfg, h, pristine=False)
        w2, keep2 = make_workload(ra, cfg, d2, n_iters)
        if cfg.coll == "allreduce":
            io, keep_io = ra.make_host_io(A=h["A"], B=h["B"], C=hC, ar_in=h["ar"], ar_out=h_out)
        else:
            io, keep_io = ra.make_host_io(A=h["A"], B=h["B"], C=hC, a2a_in=h["a2a"], a2a_out=h_out)
        ra.ra_overlap_run_host(w, w2, io, e2e_cfg, 2)            # warm-up
        barrier(world)
        t0 = time.perf_counter()
        e2e_res = ra.ra_overlap_run_host(w, w2, io, e2e_cfg, steps)
        barrier(world)
        e2e_s = max_over_ranks(time.perf_counter() - t0, world, dev)
        out["e2e"] = {"value": world * n_iters * steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                      "api": "ra_overlap_run_host (pinned host buffers; H2D, compute and D2H of consecutive steps pipelined over two device sets)",
                      "gpu_ms_per_step": e2e_res["total_ms"] / steps}
        del d2, w2, io, keep_io, hC, h_out
    del w, keep, d, h
    ra.ra_shutdown()                    # drops cached graphs / tensor maps that point into the freed buffers
    torch.cuda.empty_cache()
    return out


def flat_summary(m, peaks):
    """One config's report lines as a single string: survives a parser that keeps only scalars."""
    a, b = m["alone"], m["best_setting"]
    gem = (f"gemm alone {a['gemm_tflops_burst']:.0f} TF/s burst={a['gemm_frac_of_bf16_peak_burst']:.3f} of bf16 peak, "
           f"{a['gemm_tflops']:.0f} sustained={a['gemm_frac_of_bf16_peak_sustained']:.3f}"
           + (f" (cuBLAS same box {a['library_gemm_same_box']['burst_tflops']:.0f} / {a['library_gemm_same_box']['sustained_tflops']:.0f})"
              if "library_gemm_same_box" in a else "") if m["compute_bound"] else
           f"gemm alone {a['gemm_gbs']:.0f} GB/s={a['gemm_frac_of_hbm_peak']:.3f} of HBM peak ({a['gemm_tflops']:.0f} TF/s"
           + (f"; cuBLAS same box {a['library_gemm_same_box']['sustained_tflops']:.0f}" if "library_gemm_same_box" in a else "") + ")")
    return (f"serial {m['serial_ms_per_iter'] * 1e3:.1f} us/iter | overlap {m['overlap_ms_per_iter'] * 1e3:.1f} | "
            f"time_ratio_same {m['time_ratio_same']:.3f} best {m['time_ratio_best']:.3f} | {gem} | "
            f"coll alone {a['coll_gbs']:.0f} GB/s={a['coll_frac_of_hbm_peak']:.3f} of HBM peak | "
            f"overlap/roofline {m['overlap_vs_roofline']['sustained']:.3f} sustained {m['overlap_vs_roofline']['burst']:.3f} burst "
            f"(roofline {m['combined_roofline_ms']['sustained'] * 1e3:.1f}/{m['combined_roofline_ms']['burst'] * 1e3:.1f} us) | "
            f"setting reserve={b['smem_reserve_bytes'] // 1024}K budget={b['sm_budget']} prio={b['priority']} coll_sm={b['coll_sm_budget']} "
            f"variant={b['coll_variant']} graph={b['use_graph']} of {m['policy']['settings_in_sweep']} | overlap_rate {m['overlap_rate']:.2f} | "
            f"sm {m['clocks'].get('sm_mhz')} MHz {','.join(m['clocks'].get('reasons', [])) or 'no-throttle'} | "
            f"gemm_ctas_per_sm_seen {m['gemm_max_ctas_on_one_sm']}")


LINE_LIMIT = 2900   # bytes: the whole line fits in the last 3 kB of stdout, whichever way a reader cuts it


def _finite(x):
    """NaN / Inf -> None, recursively: the line must be strict JSON (json.dumps(..., allow_nan=False))."""
    if isinstance(x, float):
        return x if math.isfinite(x) else None
    if isinstance(x, dict):
        return {k: _finite(v) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_finite(v) for v in x]
    return x


def _r(x, n=4):
    return None if x is None or not math.isfinite(x) else float(f"{x:.{n}g}") if abs(x) < 1e15 else x


def short_summary(m):
    """One config in ~200 bytes: serial / overlapped us per iteration, their ratio, each kernel alone as a fraction of its
    peak (GEMM: burst bf16 peak if compute-bound, HBM peak otherwise), overlapped time over the combined roofline."""
    a, b = m["alone"], m["best_setting"]
    g = a["gemm_frac_of_bf16_peak_burst"] if m["compute_bound"] else a["gemm_frac_of_hbm_peak"]
    return (f"ser {m['serial_ms_per_iter'] * 1e3:.1f} ov {m['overlap_ms_per_iter'] * 1e3:.1f} us r {m['time_ratio_same']:.3f}; "
            f"gemm {g:.3f} {'tensor' if m['compute_bound'] else 'hbm'}; coll {a['coll_frac_of_hbm_peak']:.3f} hbm; "
            f"ov/roof {m['overlap_vs_roofline']['sustained']:.3f}s {m['overlap_vs_roofline']['burst']:.3f}b; "
            f"res{b['smem_reserve_bytes'] // 1024}K sm{b['sm_budget']} prio-{b['priority']} cv{b['coll_variant']}")


def contract_line(cfg, m, per_config, peaks, cpu, world, steps, warmup, sweep, total_bench_s=None, detail_path=""):
    """The ONE stdout line of the bench contract (small: the contract keys, `roofline`, `cpu_baseline`, `e2e`, `clocks`, the
    serial / overlap scalars and one short string per config) and the detail document (everything measured) that goes to
    --detail.  `m` is measure_config's result for the headline workload, `per_config` the other workloads' results."""
    flops, gbytes, cbytes = cfg.gemm_flops, cfg.gemm_bytes, cfg.coll_bytes
    alone, over_ms, gemm_in_step_ms = m["alone"], m["overlap_ms_per_iter"], m["gemm_in_step_ms"]
    # dominant kernel = the GEMM: 0.8 of the step's kernel time on cb-*, the HBM stream on mb-*; launch_ms = CUDA events
    # around every K_g launch, on the compute stream, in the instrumented pass of the same K steps after the timed region
    if m["compute_bound"]:
        ach = flops / gemm_in_step_ms / 1e9
        roof = {"kernel": "ra::gemm_kernel", "bound": "tensor", "achieved": ach, "peak": peaks["bf16_tflops_sustained"], "unit": "TFLOP/s",
                "frac": ach / peaks["bf16_tflops_sustained"], "traffic": None, "peak_kind": f"{peaks['source']}, sustained (kernel timed inside a long step)",
                "launch_ms": gemm_in_step_ms, "frac_of_burst_peak": ach / peaks["bf16_tflops"],
                "alone_burst": {"achieved": alone["gemm_tflops_burst"], "peak": peaks["bf16_tflops"], "frac": alone["gemm_frac_of_bf16_peak_burst"]}}
    else:
        ach = gbytes / gemm_in_step_ms / 1e6
        roof = {"kernel": "ra::gemm_kernel", "bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                "traffic": None, "peak_kind": peaks["source"], "launch_ms": gemm_in_step_ms,
                "alone": {"achieved": alone["gemm_gbs"], "peak": peaks["hbm_gbs"], "frac": alone["gemm_frac_of_hbm_peak"]}}
    roof["algorithmic_bytes"] = gbytes
    tpath = os.path.join(ROOT, "profiles", "traffic.json")   # dram bytes per launch from the committed ncu --set full capture
    if os.path.exists(tpath):
        with open(tpath) as f:
            t = json.load(f).get(cfg.name, {})
        # the capture that matches the timed setting: with or without the L2 carve-out (profiles/r02_l2_persist.md)
        persist = m["best_setting"].get("l2_persist_bytes", 0) >= 79 << 20
        roof["traffic"] = t.get("gemm_dram_bytes_l2_persist_79MiB" if persist else "gemm_dram_bytes")
        roof["traffic_source"] = "profiles/traffic.json (one ncu capture, another box; not this run)"
    # both kernels share HBM inside the overlapped step, so a kernel's in-step rate understates the memory system's use:
    # the whole iteration's algorithmic bytes over its time is the figure to hold against the HBM peak
    step_gbs = (gbytes + cbytes) / over_ms / 1e6
    combined_step = {"bound": "hbm", "achieved": step_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": step_gbs / peaks["hbm_gbs"],
                     "bytes_per_iter": gbytes + cbytes}

    b = m["best_setting"]
    config = {"workload": cfg.name, "gemm": [cfg.M, cfg.N, cfg.K], "collective": cfg.coll, "P": cfg.P, "coll_bytes_moved": cbytes,
              "n_iters_per_step": m["n_iters_per_step"], "l2": "inputs_exceed_l2 (no flush needed)", "multi_gpu": "replicas only",
              "sweep": sweep, "setting": {k: b[k] for k in ("smem_reserve_bytes", "sm_budget", "priority", "coll_sm_budget", "coll_variant", "use_graph") if k in b},
              "configs_in_this_run": [cfg.name] + list(per_config), "detail": detail_path or None}
    config["cfg." + cfg.name] = short_summary(m)
    for name, pm in per_config.items():
        config["cfg." + name] = short_summary(pm)
    e2e = m.get("e2e")
    line = {
        "metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": m["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic", "gpu_launches": m["gpu_launches"], "config": config,
        "serial_ms_per_iter": _r(m["serial_ms_per_iter"]), "overlap_ms_per_iter": _r(over_ms), "time_ratio": _r(m["time_ratio_same"]),
        "time_ratio_vs_kernels_alone": _r(m["time_ratio_best"]), "norm_time_priority": _r(m["norm_time_priority"]),
        "overlap_rate": _r(m["overlap_rate"]), "coll_alone_frac_of_hbm_peak": _r(alone["coll_frac_of_hbm_peak"]),
        "combined_roofline_ms": {k: _r(v) for k, v in m["combined_roofline_ms"].items()},
        "overlap_vs_roofline": {k: _r(v) for k, v in m["overlap_vs_roofline"].items()},
        "wall_ms_timed_region": _r(m["wall_ms_timed_region"], 6), "paper_context": "paper: up to 25.5% less time, priority vs baseline overlap, A40 (PAPER.md:7,122): context, not the target",
        "roofline": {k: (_r(v, 6) if isinstance(v, float) and abs(v) < 1e6 else v) for k, v in roof.items()},
        "cpu_baseline": None if cpu is None else {"value": cpu["value"], "unit": cpu["unit"], "cores": cpu["cores"], "kind": cpu["kind"],
                                                  "sample": cpu["sample"][:160]},
        "e2e": None if e2e is None else {k: e2e[k] for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step")},
        "clocks": {k: m["clocks"].get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons")},
    }
    line["roofline"]["alone_burst" if m["compute_bound"] else "alone"] = {k: _r(v, 5) for k, v in roof["alone_burst" if m["compute_bound"] else "alone"].items()}
    line = _finite(line)
    # never let the line outgrow a 3 kB tail: the optional parts go first (they are all in the detail file)
    for drop in ("paper_context", "cfgs", "time_ratio_vs_kernels_alone", "combined_roofline_ms"):
        if len(dumps_line(line)) <= LINE_LIMIT:
            break
        if drop == "cfgs":
            for k in [k for k in line["config"] if k.startswith("cfg.")]:
                del line["config"][k]
        else:
            line.pop(drop, None)
    detail = {"line": line, "headline": m, "per_config": per_config, "roofline": dict(roof, combined_step=combined_step),
              "cpu_baseline": cpu, "peaks": peaks, "total_bench_s": total_bench_s, "paper_context": PAPER_CONTEXT,
              "cfg_long": dict({cfg.name: flat_summary(m, peaks)}, **{n: flat_summary(pm, peaks) for n, pm in per_config.items()})}
    return line, detail


def dumps_line(line) -> str:
    return json.dumps(line, allow_nan=False, separators=(", ", ": "))


def run_ours(args, cfg):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the hot path has no CPU fallback")
    import paper_2606_09200_b200 as ra   # builds/loads libra.so; raises if the CUDA extension is missing

    world, rank, local = dist_setup(args.gpus)
    dev = torch.device("cuda", torch.cuda.current_device())
    peaks = load_peaks()
    t_start = time.perf_counter()
    m = measure_config(ra, cfg, args, peaks, world, dev, headline=True)

    per_config = {}
    if world == 1 and args.per_config == "all":
        for other in ra_inputs.CONFIGS[:5]:
            if other.name != cfg.name:
                per_config[other.name] = measure_config(ra, other, args, peaks, world, dev, headline=False)
    if rank != 0:
        return

    cpu = None
    if args.gpus == 1 and not args.no_cpu_baseline:
        t_iter, desc, cores, kind = cpu_oracle_full(cfg)
        cpu = {"value": 1.0 / t_iter, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds_per_iter": t_iter,
               "timed": kind}
    line, detail = contract_line(cfg, m, per_config, peaks, cpu, world, args.steps, max(args.warmup, 3), args.sweep,
                                 total_bench_s=time.perf_counter() - t_start, detail_path=args.detail)
    if args.detail:
        os.makedirs(os.path.dirname(os.path.abspath(args.detail)), exist_ok=True)
        with open(args.detail, "w") as f:
            json.dump(_finite(detail), f, indent=1, allow_nan=False)
        print(f"bench.py: per-config results, sweep, policy, residency and peaks are in {args.detail}", file=sys.stderr, flush=True)
    print(dumps_line(line), flush=True)


# ------------------------------------------------------------------------------------------------
# Diagnostics behind profiles/ (not part of the bench contract): --mode gemm-only is the command the ncu traffic
# captures run; --mode power-table is the energy accounting of the overlapped compute-bound step.
def _occ_from_args(args):
    occ = {}
    if args.l2_persist_mib:
        occ["l2_persist_bytes"] = args.l2_persist_mib << 20
    if args.sm_budget:
        occ["sm_budget"] = args.sm_budget
    if args.smem_reserve_kib:
        occ["smem_reserve_bytes"] = args.smem_reserve_kib << 10
    if args.tile_k:
        occ["tile_k"] = args.tile_k
    if args.static_order:
        occ["tile_order"] = 1
    return occ


def run_gemm_only(args, cfg):
    """The config's GEMM alone at the given occupancy knobs: a few single launches (what ncu captures), then the
    best-of-10 burst time and a back-to-back sustained time.  One JSON line."""
    import torch
    import paper_2606_09200_b200 as ra
    peaks = load_peaks()
    d = device_state(ra, cfg, host_inputs(cfg, pinned=False), pristine=False)
    occ = _occ_from_args(args)
    w1, keep1 = make_workload(ra, cfg, d, 1, coll=False)
    c1 = ra.make_cfg(mode=0, occ=occ)
    burst = []
    for _ in range(12):
        time.sleep(0.05)
        burst.append(ra.ra_overlap_run(w1, c1)["total_ms"])
    n_iters = args.n_iters or cfg.n_iters
    w, keep = make_workload(ra, cfg, d, n_iters, coll=False)
    res, _ = ra.ra_overlap_sweep(w, [ra.make_cfg(mode=0, occ=occ)], runs=max(args.sweep_runs, 6))
    g_ms, gb_ms = res[0]["total_ms"] / n_iters, min(burst[2:])
    torch.cuda.synchronize()
    print(json.dumps({"mode": "gemm-only", "workload": cfg.name, "gemm": [cfg.M, cfg.N, cfg.K], "occ": occ, "plan": res[0]["plan"],
                      "gemm_ms_burst": gb_ms, "gemm_tflops_burst": cfg.gemm_flops / gb_ms / 1e9,
                      "gemm_ms_sustained": g_ms, "gemm_tflops_sustained": cfg.gemm_flops / g_ms / 1e9,
                      "frac_of_bf16_peak_burst": cfg.gemm_flops / gb_ms / 1e9 / peaks["bf16_tflops"],
                      "algorithmic_bytes": cfg.gemm_bytes}))


def run_tile_k_table(args):
    """N3, the paper's tile-size study (Figs. 5-6: execution time of the larger-TILE_K configuration
    opt2 normalised to opt1, with priority-aware overlap) restated for this GEMM: occ.tile_k = 64 (opt2) against 32 (opt1)
    on the four full-size configs -- K_g alone, serial, overlapped without and with priority.  Each setting timed as one block by
    ra_overlap_sweep (warm-up runs first).  One JSON line; --table writes markdown."""
    import torch
    import paper_2606_09200_b200 as ra
    hi = ra.ra_device_info()["prio_greatest"]
    out = []
    for cfg in ra_inputs.CONFIGS[1:5]:
        d = device_state(ra, cfg, host_inputs(cfg, pinned=False))
        n_iters = args.n_iters or cfg.n_iters
        w_both, k0 = make_workload(ra, cfg, d, n_iters)
        w_gemm, k1 = make_workload(ra, cfg, d, n_iters, coll=False)
        variant = 1 if cfg.coll == "alltoall" and cfg.M > 128 else 0
        row = {"workload": cfg.name}
        for label, w, kw in (("gemm_alone", w_gemm, dict(mode=0)), ("serial", w_both, dict(mode=0, coll_variant=variant)),
                             ("overlap", w_both, dict(mode=1, coll_variant=variant)),
                             ("overlap_priority", w_both, dict(mode=1, coll_variant=variant, prio_comm=hi))):
            cfgs = [ra.make_cfg(**dict(kw, occ=dict(tile_k=tk))) for tk in (64, 32)]
            res, _ = ra.ra_overlap_sweep(w, cfgs, runs=max(args.sweep_runs, 9))
            t64, t32 = res[0]["total_ms"] / n_iters, res[1]["total_ms"] / n_iters
            row[label] = {"tile_k_64_ms": t64, "tile_k_32_ms": t32, "norm_64_over_32": t64 / t32,
                          "stages": [res[0]["plan"]["stages"], res[1]["plan"]["stages"]],
                          "dyn_smem_bytes": [res[0]["plan"]["dyn_smem_bytes"], res[1]["plan"]["dyn_smem_bytes"]]}
        out.append(row)
        del d, w_both, w_gemm
        torch.cuda.empty_cache()
    print(json.dumps({"mode": "tile-k-table", "rows": out}))
    if args.table:
        with open(args.table, "w") as f:
            f.write("| workload | stages x stage bytes (64 / 32) | K_g alone ms (64 / 32) | norm | serial ms | norm | overlap ms | norm | overlap + priority ms | norm |\n")
            f.write("|---|---|---|---|---|---|---|---|---|---|\n")
            for r in out:
                g = r["gemm_alone"]
                cells = [r["workload"], f"{g['stages'][0]} / {g['stages'][1]} stages, dyn smem {g['dyn_smem_bytes'][0]} / {g['dyn_smem_bytes'][1]} B"]
                for k in ("gemm_alone", "serial", "overlap", "overlap_priority"):
                    cells += [f"{r[k]['tile_k_64_ms']:.4f} / {r[k]['tile_k_32_ms']:.4f}", f"{r[k]['norm_64_over_32']:.3f}"]
                f.write("| " + " | ".join(cells) + " |\n")


def run_power_table(args, cfg):
    """Board power, SM clock and time per iteration of K_g alone, K_c alone and the overlapped step, each from a loop of
    >= --loop-s seconds (nvidia-smi sampled every 20 ms during the loop).  Energy per iteration = mean power x time.
    Prints one JSON line; --table writes the same rows as a markdown table."""
    import torch
    import paper_2606_09200_b200 as ra
    d = device_state(ra, cfg, host_inputs(cfg, pinned=False))
    n_iters = args.n_iters or cfg.n_iters
    hi = ra.ra_device_info()["prio_greatest"]
    MiB = 1 << 20
    w_both, k0 = make_workload(ra, cfg, d, n_iters)
    w_gemm, k1 = make_workload(ra, cfg, d, n_iters, coll=False)
    w_coll, k2 = make_workload(ra, cfg, d, n_iters, gemm=False)
    variants = (0, 1, 2)
    rows = [("K_g alone", w_gemm, dict(mode=0)),
            ("K_g alone, X panel in L2 (79 MiB carve-out)", w_gemm, dict(mode=0, occ=dict(l2_persist_bytes=79 * MiB)))]
    for v in variants:
        for csb in (0, 24, 32, 48):
            if v == 2 and csb:
                continue
            rows.append((f"K_c alone, variant {v}, coll_sm_budget {csb}", w_coll, dict(mode=0, coll_variant=v, coll_sm_budget=csb)))
    rows.append(("serial K_g ; K_c", w_both, dict(mode=0)))
    for v in variants:
        for csb in (0, 24, 32, 48):
            if v == 2 and csb:
                continue
            rows.append((f"overlap, variant {v}, coll_sm_budget {csb}", w_both, dict(mode=1, coll_variant=v, coll_sm_budget=csb)))
    rows.append(("overlap, variant 0, priority on", w_both, dict(mode=1, prio_comm=hi)))
    for pb in (15, 31, 47, 79):
        rows.append((f"overlap, variant {variants[0]}, X panel in L2 ({pb} MiB carve-out)", w_both,
                     dict(mode=1, coll_variant=variants[0], occ=dict(l2_persist_bytes=pb * MiB))))
    out = []
    for label, w, kw in rows:
        c = ra.make_cfg(**kw)
        for _ in range(3):
            ra.ra_overlap_run(w, c)
        torch.cuda.synchronize()
        time.sleep(1.0)                                   # every row starts from the same (cooled) state
        sampler = ClockSampler(torch.cuda.current_device())
        sampler.start()
        t0, ms, runs = time.perf_counter(), [], 0
        while time.perf_counter() - t0 < args.loop_s or runs < 30:
            ms.append(ra.ra_overlap_run(w, c)["total_ms"] / n_iters)
            runs += 1
        clocks = sampler.stop()
        mean_ms = sum(ms) / len(ms)
        sd = statistics.pstdev(ms)
        pw = clocks.get("power_w_mean")
        out.append({"setting": label, "runs": runs, "ms_per_iter": mean_ms, "ms_sd": sd, "ms_min": min(ms), "power_w_mean": pw,
                    "power_w_max": clocks.get("power_w_max"), "sm_mhz_median": clocks.get("sm_mhz"),
                    "mj_per_iter": (pw * mean_ms) if pw else None, "reasons": clocks.get("reasons")})
    line = {"mode": "power-table", "workload": cfg.name, "n_iters_per_run": n_iters, "loop_s": args.loop_s, "rows": out}
    print(json.dumps(line))
    if args.table:
        with open(args.table, "w") as f:
            f.write(f"| setting ({cfg.name}, {n_iters} iterations per run) | runs | ms/iter mean | sd | min | board W mean | W max | SM MHz median | mJ/iter |\n")
            f.write("|---|---|---|---|---|---|---|---|---|\n")
            for r in out:
                mj = f"{r['mj_per_iter']:.0f}" if r["mj_per_iter"] is not None else "-"
                pw = f"{r['power_w_mean']:.0f}" if r["power_w_mean"] is not None else "-"
                pm = f"{r['power_w_max']:.0f}" if r["power_w_max"] is not None else "-"
                f.write(f"| {r['setting']} | {r['runs']} | {r['ms_per_iter']:.4f} | {r['ms_sd']:.4f} | {r['ms_min']:.4f} | {pw} | {pm} | "
                        f"{r['sm_mhz_median']} | {mj} |\n")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cb-ar")
    ap.add_argument("--n-iters", type=int, default=0, help="iterations per step (default: the config's, 20)")
    ap.add_argument("--sweep", default="quick", choices=["none", "auto", "quick", "full"])
    ap.add_argument("--sweep-runs", type=int, default=9)
    ap.add_argument("--per-config", default="all", choices=["all", "none"],
                    help="at N=1 also run the other four BASELINE.json configs (default) or only --config")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--detail", default=os.path.join("gpurun_out", "bench_detail.json"),
                    help="everything the run measured (per-config results, sweep, policy, residency, peaks) goes to this JSON "
                         "file; stdout carries only the short contract line ('' = do not write it)")
    ap.add_argument("--ref-budget-s", type=float, default=90.0, help="--impl reference: CPU seconds for warmup + steps")
    ap.add_argument("--table", default="", help="write the sweep table (JSON; --mode power-table: markdown) here")
    ap.add_argument("--static-order", action="store_true", help="--mode gemm-only: occ.tile_order = 1 (static tile assignment)")
    ap.add_argument("--tile-k", type=int, default=0, help="--mode gemm-only: occ.tile_k (32 or 64)")
    ap.add_argument("--mode", default="bench", choices=["bench", "gemm-only", "power-table", "tile-k-table"],
                    help="gemm-only / power-table: diagnostics behind profiles/ (one GPU, not the bench contract)")
    ap.add_argument("--l2-persist-mib", type=int, default=0, help="--mode gemm-only: occ.l2_persist_bytes in MiB")
    ap.add_argument("--sm-budget", type=int, default=0, help="--mode gemm-only: occ.sm_budget")
    ap.add_argument("--smem-reserve-kib", type=int, default=0, help="--mode gemm-only: occ.smem_reserve_bytes in KiB")
    ap.add_argument("--loop-s", type=float, default=3.0, help="--mode power-table: seconds per row")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(self_launch(sys.argv[1:], args.gpus))
    cfg = get_config(args.config)
    if args.mode == "gemm-only":
        return run_gemm_only(args, cfg)
    if args.mode == "power-table":
        return run_power_table(args, cfg)
    if args.mode == "tile-k-table":
        return run_tile_k_table(args)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
