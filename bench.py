#!/usr/bin/env python
"""bench.py -- C[f] evaluations per second on BASELINE config 3 (N=256 log grid, B=64 members, mediator |M|^2, fp64).

A step is one pass of the whole hot path over one batch: kx_collide on f[B,N] (prep -> gain/loss contraction ->
reduction + raw operator).  `value` = all ranks' B*K evaluations / max-over-ranks device time, inputs resident in
HBM; `e2e` = the same through kx_collide_host (pinned host f in, C out, copies inside the timed region).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--mode log|linear] [--project]
    torchrun --nproc-per-node N ... bench.py --gpus N ...

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
# Algorithmic work of the dominant kernel k_dmma: one FMA (2 flop) per stored entry and member
# for the gain, one per (i, bracket, Chebyshev coefficient) and member for the loss.  Padding of the tiled layout,
# the f_n scaling and the operand preparation are NOT counted.
# dram__bytes_read.sum + dram__bytes_write.sum of one k_dmma launch from the committed `ncu --set full` capture
# (profiles/r01c_tiled_dmma.md; LINEAR from the working capture of the same round); null for configurations that were
# not captured.
NCU_TRAFFIC = {("log", 64): 61.43e6, ("linear", 64): 48.72e6}
# kernels of one kx_collide on the tiled path: k_dmma, k_reduce, k_contract (exact fallback, exits at once when no member
# is flagged; LOG only), k_finish
LOSS_NODES = {"log": 24, "linear": 2}
SM_COUNT, FP64_LANES_PER_SM = 148, 64      # B200: 64 FP64 FMA lanes per SM; DMMA.8x8x4 runs at the same 37.2 TFLOP/s


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
                                          "--format=csv,noheader,nounits", "-lms", "100"],
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


WORKLOADS = {3: WORKLOAD,
             4: "cfg4: N=512 log p/T in [1e-3,100], seeded bimodal f, constant |M|^2 (not the headline: HBM-bound side measurement)"}


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
    ap.add_argument("--config", type=int, default=3, choices=[3, 4],
                    help="3 = the headline workload; 4 = the N=512 small-batch workload (side measurement, HBM roofline)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

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
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)    # 256 MiB > 126 MB L2
    flush_rd = torch.zeros(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)
    flush_sink = torch.zeros(1, dtype=torch.float64, device=dev)

    def flush_l2():
        """Write 256 MiB (evicts everything), then read another 256 MiB so that L2 is left holding CLEAN lines: the
        write-back of the flusher's own dirty lines would otherwise be charged to the kernels that follow."""
        flush.zero_()
        if args.flush == "write+read":
            flush_sink.copy_(flush_rd.sum(dim=0, keepdim=True))
    stream = torch.cuda.current_stream()

    def step():
        h.collide(f, flags=flags, out=C)

    for _ in range(Wm):
        flush_l2()
        step()
    barrier()

    # ---- timed region: K steps, L2 flushed before each, device time from CUDA events on the launching stream
    sampler = ClockSampler(local)
    sampler.start()
    h.profile(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    barrier()
    for k in range(K):
        flush_l2()
        ev[k][0].record(stream)
        step()
        ev[k][1].record(stream)
    barrier()
    t_cold = sum(a.elapsed_time(b) for a, b in ev) * 1e-3
    kern_ms, kern_n = h.profile_read()
    h.profile(False)

    # ---- same K steps back to back (tensor L2-resident, as inside an integrator)
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
    t_cold, t_warm, t_e2e, t_kern = shard.max_over_ranks([t_cold, t_warm, t_e2e, kern_ms * 1e-3], dist, dev)
    same = bool(torch.isfinite(C).all())
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # context for kernel_ms: what two CUDA events around an (almost) empty kernel measure on this box
    tiny = torch.zeros(1, device=dev)
    ev_over = []
    for _ in range(20):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream); tiny.add_(1.0); e1.record(stream); e1.synchronize()
        ev_over.append(e0.elapsed_time(e1))
    ev_over_us = float(np.min(ev_over[3:])) * 1e3
    peaks, peak_src = _peaks()
    sm_max_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    nnz = info["nnz"]
    kern_s = t_kern / max(kern_n, 1)
    Q = LOSS_NODES[args.mode]
    Ngrid = info["N"]
    # FP64 tensor pipe (DMMA.8x8x4): 148 SMs x 64 FMA/clk x 2 flop x max SM clock; the library's own probe
    # (kx_probe_flops) measures it on this GPU in the same run.  The guide's nominal ratio applied to the measured
    # bf16 peak (45/2250 x bf16_tflops) is given as peak_alt.
    peak_nominal = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max_hz / 1e12
    probe = {"dmma": h.probe_flops(1), "dfma": h.probe_flops(0)}
    peak = max(peak_nominal, probe["dmma"])
    flop = 2.0 * (nnz + Ngrid * (Ngrid - 1) * Q) * B
    ach = flop / kern_s / 1e12
    hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
    t_hbm = info["tensor_bytes"] / (hbm_gbs * 1e9)
    t_flop = flop / (peak * 1e12)
    if t_hbm > t_flop:      # small batches: the tensor stream bounds the kernel (cfg4)
        ach_gbs = info["tensor_bytes"] / kern_s / 1e9
        roof_head = {"bound": "hbm", "achieved": ach_gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": ach_gbs / hbm_gbs,
                     "peak_source_hbm": f"{peak_src} copy bandwidth (MEASURED_PEAKS.json hbm_gbs)", "tflops": ach}
    else:
        roof_head = {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak}
    if streaming:
        # k_contract: FP64-pipe instructions per (entry, member) counted in the SASS of the inner loop (DESIGN.md
        # section 5): 12 classical LOG, 3 LINEAR, 22 with quantum statistics; peak = 148 SMs x 64 FP64 lanes x max clock
        c_inst = 22 if stat != 0 else (12 if args.mode == "log" else 3)
        ach_inst = nnz * B * c_inst / kern_s / 1e12
        peak_inst = SM_COUNT * FP64_LANES_PER_SM * sm_max_hz / 1e12
        roof_head = {"bound": "alu", "achieved": ach_inst, "peak": peak_inst, "unit": "T FP64 inst/s",
                     "frac": ach_inst / peak_inst, "fp64_inst_per_entry_member": c_inst}
        flop = float(nnz) * B * c_inst
    roof = {**roof_head,
            "traffic": NCU_TRAFFIC.get((args.mode, B)) if (not args.project and args.config == 3 and not streaming) else None,
            "kernel": ("k_contract (exact streaming kernel: gather, exp2, FMA per entry and member)" if streaming
                       else "k_dmma (FP64 DMMA.8x8x4: gain + Chebyshev-moment loss, coefficients computed in the kernel)"),
            "kernel_ms": kern_s * 1e3, "kernel_ms_l2_warm": kern_warm_ms / max(kern_warm_n, 1),
            "event_pair_around_empty_kernel_us": ev_over_us, "flop_per_launch": flop,
            "peak_source": f"FP64 tensor pipe: 148 SMs x 64 FMA/clk x 2 x {sm_max_hz / 1e6:.0f} MHz (clocks.max.sm, {peak_src}); "
                           f"probe in this run: DMMA {probe['dmma']:.1f}, DFMA {probe['dfma']:.1f} TFLOP/s",
            "peak_alt": {"value": float(peaks.get("bf16_tflops", 1590.0)) * 45.0 / 2250.0,
                         "how": f"{peak_src} bf16_tflops x guide nominal ratio 45/2250 (the rule for a contraction in another "
                                "dtype); `peak` is the stricter figure the DMMA probe reaches",
                         "frac": ach / (float(peaks.get("bf16_tflops", 1590.0)) * 45.0 / 2250.0)},
            "tensor_bytes_per_launch": info["tensor_bytes"],
            "hbm_time_us_at_peak": t_hbm * 1e6, "tensor_time_us_at_peak": t_flop * 1e6}
    line = {
        "metric": METRIC if args.config == 3 and B == 64 and stat == 0 else f"C[f] evals/s (fp64, N={Ngrid}, B={B})", "value": shard.aggregate_rate(B, world, K, t_cold), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": t_cold / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config], "N": Ngrid, "B_per_gpu": B, "mode": args.mode, "statistics": args.statistics, "projected": bool(args.project),
                   "nnz": nnz, "tensor_bytes": info["tensor_bytes"], "storage": "rows (streaming)" if streaming else "tiled", "loss_nodes": Q, "l2": "flushed before every timed step (256 MiB write" + (", then a 256 MiB read so that no dirty lines are left)" if args.flush == "write+read" else ")"),
                   "parallelism": f"independent batches x{world}" if world > 1 else "single GPU"},
        "value_l2_warm": world * B * K / t_warm, "ms_per_step_l2_warm": t_warm / K * 1e3,
        "calls_per_s": world * K / t_cold,
        "e2e": {"value": world * B * K / t_e2e, "unit": UNIT, "h2d_bytes_per_step": B * Ngrid * 8,
                "d2h_bytes_per_step": B * Ngrid * 8, "ms_per_step": t_e2e / K * 1e3},
        "gpu_launches": (3 if streaming else (4 if args.mode == "log" else 3)) * K, "clocks": clocks, "roofline": roof, "finite": same,
    }
    if not args.no_cpu_baseline and world == 1 and args.config == 3:
        cb = cpu_oracle(c, members=B, steps=10, warmup=1)
        line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")}
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line), flush=True)
    h.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
