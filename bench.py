#!/usr/bin/env python
"""bench.py -- C[f] evaluations per second on BASELINE config 3 (N=256 log grid, B=64 members, mediator |M|^2, fp64).

A step is one pass of the whole hot path over one batch: kx_collide on f[B,N], which is ONE cooperative kernel of libkx
(contraction on the FP64 tensor pipe -> grid barrier -> raw operator).  `value` = all ranks' B*K evaluations /
max-over-ranks device time, inputs resident in HBM, L2 flushed before every timed step; `e2e` = the same through
kx_collide_host (pinned host f in, C out, copies inside the timed region).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--mode log|linear] [--project]
                    [--config 3|4|1|2|5] [--storage tiled|rows] [--statistics classical|bose|fermi] [--no-extra]
    torchrun --nproc-per-node N ... bench.py --gpus N ...

--config 3 (default) is the headline; 4 is the N=512 small-batch side measurement (HBM roofline); 1, 2, 5 time the
integrators (kx_evolve; stages per second).  The default run also carries the side measurements as `extra` (short runs).
N > 1: the path partitions over independent distributions, so every rank evaluates its own batch of B members
(weak scaling, no data-path collective).  --impl reference times the CPU oracle as it stands (rank 0 only).
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

import kx_inputs as kin  # noqa: E402

METRIC = "C[f] evals/s (fp64, N=256, B=64)"
UNIT = "C[f]/s"
WORKLOAD = "cfg3: N=256 log p/T in [1e-3,50], B=64 seeded bimodal f, |M|^2 ~ 1/(1+q^2/m_med^2)^2, m_med=0.5"
WORKLOADS = {3: WORKLOAD,
             4: "cfg4: N=512 log p/T in [1e-3,100], seeded bimodal f, constant |M|^2 (not the headline: HBM-bound side measurement)",
             1: "cfg1: N=32 uniform p/T in [0.05,10], B=1, explicit Euler (side measurement: stages/s)",
             2: "cfg2: N=128 uniform p/T in [0.02,20], B=1, RK4 (side measurement: stages/s)",
             5: "cfg5: N=256 log p/T in [1e-3,100], B=8, RK4 with m(u)=x (tensor rebuilt at every stage), two sources (side measurement: stages/s)"}
# Algorithmic work of the fused kernel k_dmma: one FMA (2 flop) per stored entry and member for the
# gain, one per (i, bracket, Chebyshev node) and member for the loss.  Padding of the tiled layout, the f_n scaling and
# the operand preparation are NOT counted.
LOSS_NODES = {"log": 24, "linear": 2}
SM_COUNT, FP64_LANES_PER_SM = 148, 64      # B200: 64 FP64 FMA lanes per SM; DMMA.8x8x4 runs at the same 37.2 TFLOP/s
# dram__bytes_read.sum + dram__bytes_write.sum of one k_dmma launch, from the committed `ncu --set full` capture named in
# TRAFFIC_SOURCE (cfg3, LOG, B=64, raw operator); null for every other configuration
NCU_TRAFFIC = {("log", 64): 61.27e6}
TRAFFIC_SOURCE = "profiles/r02_k_dmma_full.md"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return json.load(open(path)), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for k, nm in enumerate(names):
                if len(r) > 2 + k and r[2 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _inputs(rank: int, B: int, cfg: int = 3):
    from paper_2607_00755_b200 import shard
    c = kin.config(cfg, B=B)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank:   # every rank its own members: global member g has seed 1000*cfg + g
        c["f"] = np.stack([kin._random_bimodal(c["p"], 1000 * cfg + int(g)) for g in shard.weak_member_ids(B, rank, world)])
    return c


def cpu_oracle(c, members: int, steps: int = 1, warmup: int = 0):
    """The oracle as it stands, timed on the host cores on a bounded sample: dense tables built once (timed
    separately), then `members` members of the batch evaluated per step (evaluate phase O8-O9)."""
    import oracle
    t0 = time.perf_counter()
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    t_build = time.perf_counter() - t0
    fs = np.ascontiguousarray(c["f"][:members])
    for _ in range(warmup):
        oracle.collide(T, fs, oracle.LOG)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.collide(T, fs, oracle.LOG)
    dt = (time.perf_counter() - t0) / max(steps, 1)
    return dict(value=members / dt, unit=UNIT, cores=os.cpu_count(), kind="oracle",
                sample=f"{members} of {len(c['f'])} members of cfg3 per step, evaluate phase (O8-O9) over the dense N^3 tables, "
                       f"{steps} step(s); table build (O1-O7) {t_build:.1f} s not included",
                ms_per_step=dt * 1e3, build_s=t_build)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c = _inputs(0, 64)
    members = 16
    cb = cpu_oracle(c, members, steps=args.steps, warmup=min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": cb["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": cb["sample"]},
            "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


class Flusher:
    """Write 256 MiB (evicts everything), then read another 256 MiB so that L2 is left holding CLEAN lines: the write-back
    of the flusher's own dirty lines would otherwise be charged to the kernel that follows."""

    def __init__(self, torch, dev, mode="write+read"):
        self.mode = mode
        self.buf = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)    # 256 MiB > 126 MB L2
        self.rd = torch.zeros(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)
        self.sink = torch.zeros(1, dtype=torch.float64, device=dev)

    def __call__(self):
        self.buf.zero_()
        if self.mode == "write+read":
            self.sink.copy_(self.rd.sum(dim=0, keepdim=True))


def time_collide(torch, h, f, C, flags, K, Wm, flusher, barrier, reps=5, calls=200):
    """The timing protocol of one operator configuration.  Returns seconds:
       t_cold    sum over K steps of the CUDA-event time of one kx_collide, L2 flushed before each (profiling off)
       kern_cold mean device time of the fused kernel in a second flushed pass, from CUDA events recorded by the library on
                 the launching stream around the launch (kx_profile); kern_warm: the same back to back
       t_warm    K calls back to back (the tensor stays in L2, as inside an integrator)
       t_med     median over `reps` repeats of `calls` back-to-back calls, per call (SURVEY.md 8(d) protocol)"""
    stream = torch.cuda.current_stream()

    def step():
        h.collide(f, flags=flags, out=C)
    for _ in range(Wm):
        flusher()
        step()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    h.fallback_members()                     # reset the counter: the timed region reports its own
    barrier()
    for k in range(K):
        flusher()
        ev[k][0].record(stream)
        step()
        ev[k][1].record(stream)
    barrier()
    t_cold = sum(a.elapsed_time(b) for a, b in ev) * 1e-3
    fb = h.fallback_members()
    # the kernel alone, same flushed protocol, events recorded by the library around the launch
    h.profile(True)
    for k in range(K):
        flusher()
        step()
    kern_ms, kern_n = h.profile_read()
    h.profile(False)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    a.record(stream)
    for k in range(K):
        step()
    b.record(stream)
    barrier()
    t_warm = a.elapsed_time(b) * 1e-3
    h.profile(True)
    for k in range(K):
        step()
    kern_warm_ms, kern_warm_n = h.profile_read()
    h.profile(False)
    meds = []
    for _ in range(reps):
        a.record(stream)
        for k in range(calls):
            step()
        b.record(stream)
        b.synchronize()
        meds.append(a.elapsed_time(b) * 1e-3 / calls)
    return dict(t_cold=t_cold, t_warm=t_warm, kern_cold=kern_ms * 1e-3 / max(kern_n, 1),
                kern_warm=kern_warm_ms * 1e-3 / max(kern_warm_n, 1), t_med=float(np.median(meds)), fallback=fb)


def trace_phases(torch, h, f, C, flags, flusher, reps=5):
    """Phases of the fused tensor-core kernel from its own clock stamps (kx_trace: %globaltimer per CTA), L2 flushed before
    every traced launch; microseconds since the first CTA entered, median over `reps` launches."""
    h.trace(True)
    out = []
    for _ in range(reps):
        flusher()
        h.collide(f, flags=flags, out=C)
        torch.cuda.synchronize()
        tr = h.trace_read().astype(np.int64).reshape(160, 32)
        ent = tr[:, 0][tr[:, 0] > 0]
        if ent.size == 0:
            continue
        t0 = ent.min()

        def last(slot):
            v = tr[:, slot][tr[:, slot] > 0]
            return float(v.max() - t0) * 1e-3 if v.size else float("nan")
        out.append((last(1), last(2), last(3), last(5)))
    h.trace(False)
    if not out:
        return None
    m = np.median(np.array(out), axis=0)
    return {"prologue_done_us": m[0], "dmma_phase_done_us": m[1], "barrier_passed_us": m[2], "kernel_done_us": m[3],
            "how": "last CTA to reach each point, microseconds since the first CTA entered (kx_trace), L2 flushed, median of %d" % len(out)}


def roofline(info, B, mode, streaming, stat, kern_s, peaks, peak_src, probe):
    """Roofline of the fused kernel for this configuration."""
    sm_max_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    nnz, N = info["nnz"], info["N"]
    Q = LOSS_NODES[mode]
    if streaming:
        # k_stream: FP64-pipe instructions per (entry, member) counted in the SASS of the inner loop:
        # 12 classical LOG, 3 LINEAR, 22 with quantum statistics; peak = 148 SMs x 64 FP64 lanes x max clock
        c_inst = 22 if stat != 0 else (12 if mode == "log" else 3)
        ach = nnz * B * c_inst / kern_s / 1e12
        peak = SM_COUNT * FP64_LANES_PER_SM * sm_max_hz / 1e12
        return {"bound": "alu", "achieved": ach, "peak": peak, "unit": "T FP64 inst/s", "frac": ach / peak,
                "fp64_inst_per_entry_member": c_inst, "work_per_launch": float(nnz) * B * c_inst,
                "kernel": "k_stream (exact streaming kernel: gather, exp2, FMA per entry and member; barrier; finishing phase)"}
    peak_nominal = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max_hz / 1e12
    peak = max(peak_nominal, probe["dmma"]) if probe else peak_nominal
    flop = 2.0 * (nnz + N * (N - 1) * Q) * B
    ach = flop / kern_s / 1e12
    hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
    t_hbm = info["tensor_bytes"] / (hbm_gbs * 1e9)
    t_flop = flop / (peak * 1e12)
    kname = "k_dmma (one cooperative kernel per evaluation: gain + Chebyshev-node loss on FP64 DMMA.8x8x4, grid barrier, finishing phase)"
    if t_hbm > t_flop:      # small batches: the tensor stream bounds the kernel (cfg4)
        ach_gbs = info["tensor_bytes"] / kern_s / 1e9
        return {"bound": "hbm", "achieved": ach_gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": ach_gbs / hbm_gbs,
                "peak_source": f"{peak_src} copy bandwidth (MEASURED_PEAKS.json hbm_gbs)", "tflops": ach,
                "work_per_launch": float(info["tensor_bytes"]), "kernel": kname}
    return {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
            "peak_source": f"FP64 tensor pipe: 148 SMs x 64 FMA/clk x 2 x {sm_max_hz / 1e6:.0f} MHz (clocks.max.sm, {peak_src})"
                           + (f"; probe in this run: DMMA {probe['dmma']:.1f}, DFMA {probe['dfma']:.1f} TFLOP/s" if probe else ""),
            "work_per_launch": flop, "hbm_time_us_at_peak": t_hbm * 1e6, "tensor_time_us_at_peak": t_flop * 1e6,
            "kernel": kname}


def side_collide(torch, kx, dev, local, peaks, peak_src, flusher, barrier, *, cfg, B, mode="log", project=False,
                 storage="tiled", statistics="classical", precision="fp64", K=10):
    """One short side measurement of the operator (same protocol as the headline, fewer steps)."""
    c = kin.config(cfg, B=B)
    stat = {"classical": kx.STAT_CLASSICAL, "bose": kx.STAT_BOSE, "fermi": kx.STAT_FERMI}[statistics]
    fp32 = precision == "fp32"
    streaming = storage == "rows" or stat != 0 or fp32
    if stat != 0:
        c["f"] = c["f"] / np.abs(c["f"]).max(axis=1, keepdims=True) * (0.8 if stat < 0 else 2.5)
    h = kx.Handle(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"], device=local,
                  interp=kx.INTERP_LOG if mode == "log" else kx.INTERP_LINEAR,
                  storage=kx.STORE_SYM_ROWS if streaming else kx.STORE_TILED, statistics=stat,
                  precision=kx.FP32 if fp32 else kx.FP64)
    f = torch.tensor(c["f"], dtype=torch.float64, device=dev)
    C = torch.empty_like(f)
    t = time_collide(torch, h, f, C, kx.PROJECT if project else 0, K, 3, flusher, barrier, reps=3, calls=50)
    info = h.info()
    roof = roofline(info, B, mode, streaming, stat, t["kern_cold"], peaks, peak_src, None)
    if fp32:    # fp32 contraction: 4 FP32-pipe FMA/MUL per (entry, member) + one MUFU.EX2; peak 148 SMs x 128 lanes x max clock
        peak32 = SM_COUNT * 128 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
        ach32 = info["nnz"] * B * 4 / t["kern_cold"] / 1e12
        roof.update({"bound": "alu", "achieved": ach32, "peak": peak32, "unit": "T FP32 inst/s", "frac": ach32 / peak32})
    h.close()
    return {"N": info["N"], "B": B, "mode": mode, "projected": project, "storage": "rows" if streaming else storage,
            "statistics": statistics, "precision": precision,
            "evals_per_s": B * K / t["t_cold"], "ms_per_step": t["t_cold"] / K * 1e3,
            "ms_per_step_l2_warm": t["t_warm"] / K * 1e3, "ms_per_call_median": t["t_med"] * 1e3,
            "kernel_ms": t["kern_cold"] * 1e3, "bound": roof["bound"], "frac": roof["frac"], "achieved": roof["achieved"],
            "peak": roof["peak"], "unit": roof["unit"], "fallback_members": t["fallback"]}


def time_evolve(torch, kx, dev, local, cfg, steps=None, with_oracle=False):
    """kx_evolve on config 1, 2 or 5: device time per Runge-Kutta stage (CUDA events around the whole call, which ends with
    the library's own stream synchronisation)."""
    stream = torch.cuda.current_stream()
    if cfg == 5:
        B = 8
        c = kin.config(5, B=B)
        S = steps or 300
        full = kin.config5_schedule(c["p"], c["p"] ** 2 * c["dp"], B=B, S=10_000)
        k0 = 3900                             # around x = 1: source 1 on, then off
        sch = dict(tau=full["tau"][k0:k0 + S + 1], rate=full["rate"][2 * k0:2 * (k0 + S) + 1],
                   mass=full["mass"][2 * k0:2 * (k0 + S) + 1], amp=np.ascontiguousarray(full["amp"][:, k0:k0 + S]))
        h = kx.Handle(c["p"], c["dp"], c["m"], device=local)
        G = torch.tensor(full["G"], dtype=torch.float64, device=dev)
        f0 = torch.tensor(np.stack([1e-3 * kin.bimodal(c["p"], (3.0, 30.0), (1.0, 3.0))] * B), dtype=torch.float64, device=dev)
        kw = dict(method=kx.RK4, rate=sch["rate"], mass=sch["mass"], kappa=full["kappa"], G=G, amp=sch["amp"])
        tau, nstage, method = sch["tau"], 4, "RK4"
    else:
        c = kin.config(cfg)
        h = kx.Handle(c["p"], c["dp"], c["m"], device=local)
        f0 = torch.tensor(c["f"], dtype=torch.float64, device=dev)
        loss = h.collide_parts(f0)[1].cpu().numpy()[0]
        numax = float((loss / c["f"][0]).max())
        S = steps or (2000 if cfg == 1 else 500)
        dt = (0.2 if cfg == 1 else 0.5) / numax
        tau = np.arange(S + 1) * dt
        kw = dict(method=kx.EULER if cfg == 1 else kx.RK4)
        nstage, method, B = (1 if cfg == 1 else 4), ("EULER" if cfg == 1 else "RK4"), 1
    f = f0.clone()
    best = None
    for _ in range(3):                        # the first repeat also warms up; the best of the three counts
        f.copy_(f0)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(stream)
        h.evolve(f, tau, **kw)
        b.record(stream)
        b.synchronize()
        t = a.elapsed_time(b) * 1e-3
        best = t if best is None or t < best else best
    info = h.info()
    out = {"workload": WORKLOADS[cfg], "N": info["N"], "B": B, "method": method, "steps": S, "stages": S * nstage,
           "us_per_stage": best / (S * nstage) * 1e6, "stages_per_s": S * nstage / best,
           "member_stages_per_s": B * S * nstage / best, "finite": bool(torch.isfinite(f).all())}
    if cfg == 5:
        # per stage: rebuild of a1-a3 for the stage's mass (about 80 FP64 operations per entry) and the
        # exact streaming contraction (12 FP64 instructions per entry and member)
        nnz = info["nnz"]
        out["fp64_inst_per_stage_contraction"] = float(nnz) * B * 12
        out["note"] = "every stage rebuilds the kernel tensor for m(u) and streams it once (KX_STORE_SYM_ROWS path)"
    h.close()
    if with_oracle:
        import oracle
        So = 3 if cfg == 5 else (200 if cfg == 1 else 10)
        t0 = time.perf_counter()
        if cfg == 5:
            oracle.evolve(c["p"], c["dp"], f0.cpu().numpy(), m=float(sch["mass"][0]), method=oracle.RK4, tau=sch["tau"][:So + 1],
                          rate=sch["rate"][:2 * So + 1], mass=sch["mass"][:2 * So + 1], kappa=full["kappa"], G=full["G"],
                          amp=np.ascontiguousarray(sch["amp"][:, :So]))
        else:
            oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], method=oracle.EULER if cfg == 1 else oracle.RK4, tau=tau[:So + 1])
        dto = time.perf_counter() - t0
        out["cpu_oracle"] = {"stages_per_s": So * nstage / dto, "cores": os.cpu_count(), "kind": "oracle",
                             "sample": f"{So} steps of the same schedule"}
    return out


def run_evolve(args):
    import torch
    import paper_2607_00755_b200 as kx
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libkx has no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if int(os.environ.get("RANK", "0")) != 0:
        return
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    sampler = ClockSampler(local)
    sampler.start()
    r = time_evolve(torch, kx, dev, local, args.config, steps=None, with_oracle=not args.no_cpu_baseline)
    clocks = sampler.stop()
    line = {"metric": f"Runge-Kutta stages/s (kx_evolve, fp64, N={r['N']}, B={r['B']})", "value": r["stages_per_s"], "unit": "stages/s",
            "n_gpus": 1, "steps": r["steps"], "warmup": 1, "ms_per_step": r["us_per_stage"] * 1e-3 * (r["stages"] / r["steps"]),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": r["workload"]}, "evolve": r, "clocks": clocks,
            "gpu_launches": r["stages"] * (5 if args.config == 5 else 1)}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="kx", choices=["kx", "reference"])
    ap.add_argument("--mode", default="log", choices=["log", "linear"])
    ap.add_argument("--project", action="store_true", help="time the projected operator (App. C) instead of the raw one")
    ap.add_argument("--batch", type=int, default=None, help="members per GPU (default: 64 for cfg3, 8 for cfg4)")
    ap.add_argument("--flush", default="write+read", choices=["write", "write+read"],
                    help="L2 flush before every timed step: a 256 MiB write, optionally followed by a 256 MiB read that "
                         "leaves L2 holding clean lines (default)")
    ap.add_argument("--storage", default="tiled", choices=["tiled", "rows"],
                    help="rows = the exact streaming kernel alone (one exp per entry and member): FP64-ALU roofline")
    ap.add_argument("--statistics", default="classical", choices=["classical", "bose", "fermi"],
                    help="quantum statistics of eq. 4.3 (side measurement; streaming kernel, FP64-ALU roofline)")
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5],
                    help="3 = the headline workload; 4 = the N=512 small-batch workload (HBM roofline); 1, 2, 5 = kx_evolve")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the side measurements carried in `extra`")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.config in (1, 2, 5):
        return run_evolve(args)

    import torch
    import paper_2607_00755_b200 as kx

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libkx has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    B = args.batch if args.batch else (64 if args.config == 3 else 8)
    K, Wm = args.steps, max(args.warmup, 3)
    c = _inputs(rank, B, args.config)
    stat = {"classical": kx.STAT_CLASSICAL, "bose": kx.STAT_BOSE, "fermi": kx.STAT_FERMI}[args.statistics]
    streaming = args.storage == "rows" or stat != 0
    if stat != 0:    # occupations of order one, Fermi below 1: where the quantum factors matter
        c["f"] = c["f"] / np.abs(c["f"]).max(axis=1, keepdims=True) * (0.8 if stat < 0 else 2.5)
    h = kx.Handle(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"], device=local,
                  interp=kx.INTERP_LOG if args.mode == "log" else kx.INTERP_LINEAR,
                  storage=kx.STORE_SYM_ROWS if streaming else kx.STORE_TILED, statistics=stat)
    info = h.info()
    dev = torch.device("cuda", local)
    f = torch.tensor(c["f"], dtype=torch.float64, device=dev)
    C = torch.empty_like(f)
    flags = kx.PROJECT if args.project else 0
    flusher = Flusher(torch, dev, args.flush)
    h.reserve(B)

    sampler = ClockSampler(local)
    sampler.start()
    t = time_collide(torch, h, f, C, flags, K, Wm, flusher, barrier)
    phases = trace_phases(torch, h, f, C, flags, flusher) if not streaming else None

    # ---- end to end through host buffers
    fh = torch.tensor(c["f"], dtype=torch.float64).pin_memory()
    Ch = torch.empty_like(fh).pin_memory()
    for _ in range(3):
        h.collide_host(fh, Ch, flags=flags)
    barrier()
    t0 = time.perf_counter()
    for k in range(K):
        h.collide_host(fh, Ch, flags=flags)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    clocks = sampler.stop()

    from paper_2607_00755_b200 import shard
    t_cold, t_warm, t_e2e, t_kern = shard.max_over_ranks([t["t_cold"], t["t_warm"], t_e2e, t["kern_cold"]], dist, dev)
    same = bool(torch.isfinite(C).all())
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # context for kernel_ms: what two CUDA events around an (almost) empty kernel measure on this box
    stream = torch.cuda.current_stream()
    tiny = torch.zeros(1, device=dev)
    ev_over = []
    for _ in range(20):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream); tiny.add_(1.0); e1.record(stream); e1.synchronize()
        ev_over.append(e0.elapsed_time(e1))
    ev_over_us = float(np.min(ev_over[3:])) * 1e3
    peaks, peak_src = _peaks()
    probe = {"dmma": h.probe_flops(1), "dfma": h.probe_flops(0)}
    roof = roofline(info, B, args.mode, streaming, stat, t_kern, peaks, peak_src, probe)
    headline = (not args.project and args.config == 3 and not streaming)
    roof.update({
        "traffic": NCU_TRAFFIC.get((args.mode, B)) if headline else None,
        "traffic_source": TRAFFIC_SOURCE if headline and (args.mode, B) in NCU_TRAFFIC else None,
        "kernel_ms": t_kern * 1e3, "kernel_ms_l2_warm": t["kern_warm"] * 1e3,
        "step_frac": roof["work_per_launch"] / (t_cold / K) / (roof["peak"] * (1e9 if roof["unit"] == "GB/s" else 1e12)),
        "event_pair_around_empty_kernel_us": ev_over_us, "tensor_bytes_per_launch": info["tensor_bytes"]})
    if phases is not None:
        # the contraction alone (what round 1's k_dmma was): work over the time the last CTA needs to write its partials
        phases["dmma_phase_frac"] = roof["work_per_launch"] / (phases["dmma_phase_done_us"] * 1e-6) / (roof["peak"] * (1e9 if roof["unit"] == "GB/s" else 1e12))
        roof["phases"] = phases
    Ngrid = info["N"]
    line = {
        "metric": METRIC if args.config == 3 and B == 64 and stat == 0 else f"C[f] evals/s (fp64, N={Ngrid}, B={B})",
        "value": shard.aggregate_rate(B, world, K, t_cold), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": t_cold / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config], "N": Ngrid, "B_per_gpu": B, "mode": args.mode,
                   "statistics": args.statistics, "projected": bool(args.project), "nnz": info["nnz"],
                   "tensor_bytes": info["tensor_bytes"], "storage": "rows (streaming)" if streaming else "tiled",
                   "loss_nodes": LOSS_NODES[args.mode],
                   "l2": "flushed before every timed step (256 MiB write" + (", then a 256 MiB read so that no dirty lines are left)" if args.flush == "write+read" else ")"),
                   "parallelism": f"independent batches x{world}" if world > 1 else "single GPU"},
        "value_l2_warm": world * B * K / t_warm, "ms_per_step_l2_warm": t_warm / K * 1e3,
        "ms_per_call_median_of_5x200_back_to_back": t["t_med"] * 1e3,
        "calls_per_s": world * K / t_cold,
        "e2e": {"value": world * B * K / t_e2e, "unit": UNIT, "h2d_bytes_per_step": B * Ngrid * 8,
                "d2h_bytes_per_step": B * Ngrid * 8, "ms_per_step": t_e2e / K * 1e3},
        "gpu_launches": K, "kernels_per_step": 1, "fallback_members": t["fallback"],
        "clocks": clocks, "roofline": roof, "finite": same,
    }
    if not args.no_cpu_baseline and world == 1 and args.config == 3:
        cb = cpu_oracle(c, members=B, steps=10, warmup=1)
        line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
    else:
        line["cpu_baseline"] = None
    h.close()
    if not args.no_extra and world == 1 and headline and B == 64:
        # side measurements, short runs of the same protocol (driver-observed; none of them is the headline)
        extra = {}
        sc = dict(torch=torch, kx=kx, dev=dev, local=local, peaks=peaks, peak_src=peak_src, flusher=flusher, barrier=barrier)
        try:
            extra["cfg3_linear"] = side_collide(**sc, cfg=3, B=64, mode="linear")
            extra["cfg3_projected"] = side_collide(**sc, cfg=3, B=64, project=True)
            extra["cfg3_rows"] = side_collide(**sc, cfg=3, B=64, storage="rows", K=5)
            extra["cfg3_bose"] = side_collide(**sc, cfg=3, B=64, statistics="bose", K=5)
            extra["cfg3_fp32"] = side_collide(**sc, cfg=3, B=64, precision="fp32", K=5)
            extra["cfg4_b8"] = side_collide(**sc, cfg=4, B=8)
            extra["cfg4_b1"] = side_collide(**sc, cfg=4, B=1)
            for cfg in (1, 2, 5):
                extra[f"cfg{cfg}_evolve"] = time_evolve(torch, kx, dev, local, cfg, steps={1: 1000, 2: 200, 5: 100}[cfg])
        except Exception as e:      # a side measurement must not take the headline down
            extra["error"] = repr(e)
        line["extra"] = extra
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
