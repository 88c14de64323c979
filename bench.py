#!/usr/bin/env python
"""bench.py -- collision pairs/s of the neural DSMC collision step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--chi table|mlp|mlp_tc] [--impl reference]

A "step" is one pass of the whole hot path: dsmc_bin (a1) on the
unsorted resident particle arrays, then the fused ab initio collision step (a2-a9) on the
cell-sorted arrays, on the Mach-10 cylinder-shaped population of BASELINE.json (cfg 5:
400x200 cells, 2e7 particles, pairs = floor(N_k/2) per cell).  Inputs are synthetic and seeded
(paper_2602_21244_b200/workloads.py).  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "collision_pairs_per_s"
UNIT = "pairs/s"
NX, NY, N_TOTAL = 400, 200, 20_000_000
TABLE_N = 1024
B_MAX = 1e-9


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--chi", default="table", choices=["table", "mlp", "mlp_tc"])
    ap.add_argument("--scale", type=float, default=1.0, help="shrink the population (debug only; marks the line)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-variants", action="store_true")
    ap.add_argument("--no-loop", action="store_true", help="skip the couette_loop section (SURVEY 8(f4))")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d["hbm_gbs"], d["bf16_tflops"], d.get("bf16_tflops_sustained", d["bf16_tflops"]), "measured"
    return 6650.0, 1590.0, 1400.0, "fallback"


TRAFFIC_FILE = "profiles/r02_kernel_traffic.json"


def measured_traffic(chi):
    """dram__bytes_read.sum + dram__bytes_write.sum of the fused collide kernel, per launch, from the committed
    `ncu --set full` capture named in TRAFFIC_FILE (not measured in this run: ncu cannot run inside a timed bench);
    returns (bytes or None, where the number comes from)."""
    p = os.path.join(ROOT, TRAFFIC_FILE)
    if os.path.exists(p):
        e = json.load(open(p)).get(chi, {})
        if e.get("dram_bytes_per_launch") is not None:
            return e["dram_bytes_per_launch"], "%s: %s" % (TRAFFIC_FILE, e.get("capture", "ncu --set full capture"))
    return None, "no capture for this variant"


def population(args, rank=0):
    from paper_2602_21244_b200 import workloads as wl
    s = args.scale
    nx, ny = max(8, int(round(NX * s ** 0.5))), max(4, int(round(NY * s ** 0.5)))
    return wl.mach10_cylinder(seed=4 + 1000 * rank, nx=nx, ny=ny, n_total=int(N_TOTAL * s))


def config_dict(args, pop, pairs):
    return {"workload": "cfg5 Mach-10 cylinder population %dx%d cells, %d particles, %d pairs/step, ab initio chi "
                        "by %s + rotation + moment matching; step = dsmc_bin + fused collide" % (
                            NX if args.scale == 1.0 else -1, NY if args.scale == 1.0 else -1, pop.n, pairs, args.chi),
            "chi_mode": args.chi, "n_particles": pop.n, "n_cells": pop.n_cells, "pairs_per_step": pairs,
            "table": "%dx%d fp32 LJ 12-6 (quadrature; device-built in the product arm, oracle-built in the reference arm)" % (TABLE_N, TABLE_N),
            "l2_policy": "inputs larger than L2 (%.0f MB touched per step)" % (pop.n * 48 / 1e6),
            "scale": args.scale}


# ----------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on a bounded sample of the same workload
# ----------------------------------------------------------------------------------------------
def oracle_sample(pop, chi, target_pairs=150_000):
    """Contiguous cell range holding about target_pairs pairs, starting at the first shock-band cell
    row so the sample mixes freestream, shock and wake cells like the whole population."""
    counts = pop.counts
    half = counts // 2
    cum = np.cumsum(half)
    k0 = int(pop.n_cells * 0.30)
    base = cum[k0 - 1] if k0 > 0 else 0
    k1 = int(np.searchsorted(cum, base + target_pairs))
    k1 = min(max(k1, k0 + 1), pop.n_cells)
    keep = (pop.cell >= k0) & (pop.cell < k1)
    return k0, k1, keep


def time_oracle(pop, chi, table, mlp_w, steps, warmup, target_pairs=150_000):
    import oracle
    k0, k1, keep = oracle_sample(pop, chi, target_pairs)
    cell = (pop.cell[keep] - k0).astype(np.int32)
    vx, vy, vz = pop.vx[keep], pop.vy[keep], pop.vz[keep]
    K = k1 - k0
    pairs = int((pop.counts[k0:k1] // 2).sum())
    otab = oracle.ChiTable(table.chi, table.lnE_min, table.lnE_max)
    net = oracle.Mlp(mlp_w[0], mlp_w[1], oracle.ACT_SILU)
    prm = oracle.AbinitioParams(chi_mode=0 if chi == "table" else 1)
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        rc, perm, cs = oracle.bin_particles(cell, K)
        v = [a[perm].astype(np.float64) for a in (vx, vy, vz)]
        oracle.collide_abinitio(cs, *v, prm, 4, it, net=net, table=otab)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    t = float(np.mean(times))
    return pairs / t, t, pairs, "cells [%d,%d) of the cfg5 population: %d particles, %d pairs, bin + fused ab initio " \
                               "(%s) step, fp64 single thread" % (k0, k1, int(keep.sum()), pairs, chi)


_MP = {}


def _oracle_worker(args):
    """One process of the all-cores oracle run: bin + fused step on its own contiguous cell range.  cell_base keeps
    the Philox counters global, so the union of the workers' results is the single-thread result (cells are
    independent)."""
    import oracle
    k0, k1, it = args
    pop, chi, table, mlp_w = _MP["pop"], _MP["chi"], _MP["table"], _MP["mlp_w"]
    lo, hi = int(_MP["cum"][k0]), int(_MP["cum"][k1])
    idx = _MP["order"][lo:hi]
    cell = (pop.cell[idx] - k0).astype(np.int32)
    otab = oracle.ChiTable(table.chi, table.lnE_min, table.lnE_max)
    net = oracle.Mlp(mlp_w[0], mlp_w[1], oracle.ACT_SILU)
    prm = oracle.AbinitioParams(chi_mode=0 if chi == "table" else 1, cell_base=k0)
    rc, perm, cs = oracle.bin_particles(cell, k1 - k0)
    v = [a[idx][perm].astype(np.float64) for a in (pop.vx, pop.vy, pop.vz)]
    oracle.collide_abinitio(cs, *v, prm, 4, it, net=net, table=otab)
    return hi - lo


def time_oracle_all_cores(pop, chi, table, mlp_w, target_pairs_per_core):
    """The same oracle on every host core: N processes over contiguous cell ranges of one sample.
    Returns pairs/s, seconds, pairs, cores, description."""
    import multiprocessing as mp
    cores = len(os.sched_getaffinity(0))
    k0, k1, keep = oracle_sample(pop, chi, target_pairs_per_core * cores)
    order = np.argsort(pop.cell, kind="stable")
    cum = np.concatenate([[0], np.cumsum(pop.counts)])
    half = np.cumsum(pop.counts[k0:k1] // 2)
    cuts = [k0] + [k0 + int(np.searchsorted(half, half[-1] * (w + 1) / cores)) for w in range(cores - 1)] + [k1]
    cuts = sorted(set(min(max(c, k0), k1) for c in cuts))
    _MP.update(pop=pop, chi=chi, table=table, mlp_w=mlp_w, order=order, cum=cum)
    pairs = int((pop.counts[k0:k1] // 2).sum())
    ctx = mp.get_context("fork")
    with ctx.Pool(len(cuts) - 1) as pool:
        pool.map(_oracle_worker, [(a, b, 0) for a, b in zip(cuts[:-1], cuts[1:])])  # warm-up: pages, library
        t0 = time.perf_counter()
        pool.map(_oracle_worker, [(a, b, 1) for a, b in zip(cuts[:-1], cuts[1:])])
        t = time.perf_counter() - t0
    return pairs / t, t, pairs, len(cuts) - 1, "cells [%d,%d) of the cfg5 population split into %d contiguous ranges, one " \
        "process each: %d pairs, bin + fused ab initio (%s) step, fp64" % (k0, k1, len(cuts) - 1, pairs, chi)


def host_info():
    model = "unknown"
    try:
        for l in open("/proc/cpuinfo"):
            if l.startswith("model name"):
                model = l.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "usable_cores": len(os.sched_getaffinity(0)), "cpu_model": model,
            "oracle_build": "gcc -O2 -std=c99 (no fast-math), oracle/dsmc_oracle.c"}


def build_operators(chi_needed=True):
    """chi table by the oracle's quadrature (allowed: it is an INPUT, built once, outside timing)
    and the random-init chi-MLP 2->128->128->1 (seed 3)."""
    import oracle
    from paper_2602_21244_b200 import workloads as wl
    t0 = time.perf_counter()
    table = oracle.build_chi_table(oracle.lj_argon(), TABLE_N, TABLE_N, b_max=B_MAX, n_panels=1)
    Ws, bs = wl.random_mlp(3, [2, 128, 128, 1])
    return table, (Ws, bs), time.perf_counter() - t0


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons sampled DURING the timed region: NVML (one query ~ 0.1 ms, every 1 ms) when
    nvidia_ml_py can be initialised, else the nvidia-smi command line (one query ~ 100 ms)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag = index, False
        self.sm, self.sm_max, self.reasons, self.source = [], None, set(), "nvidia-smi"
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.nvml, self.source = pynvml, "nvml"
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        self.sm.append(float(n.nvmlDeviceGetClockInfo(self.h, n.NVML_CLOCK_SM)))
        r = n.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        for name, bit in (("hw_slowdown", n.nvmlClocksEventReasonHwSlowdown),
                          ("hw_thermal_slowdown", n.nvmlClocksEventReasonHwThermalSlowdown),
                          ("sw_thermal_slowdown", n.nvmlClocksEventReasonSwThermalSlowdown),
                          ("sw_power_cap", n.nvmlClocksEventReasonSwPowerCap)):
            if r & bit:
                self.reasons.add(name)

    def _sample_smi(self):
        out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                              "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
        r = [x.strip() for x in out.strip().split(",")]
        if len(r) >= 7 and r[0].replace(".", "").isdigit():
            self.sm.append(float(r[0]))
            self.sm_max = max(self.sm_max or 0.0, float(r[1]))
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    self.reasons.add(name)

    def run(self):
        while not self.stop_flag:
            try:
                if self.nvml is not None:
                    self._sample_nvml()
                    time.sleep(0.001)
                else:
                    self._sample_smi()
                    time.sleep(0.05)
            except Exception:
                time.sleep(0.01)

    def mark(self):
        """forget what was sampled so far (called when the timed region starts)"""
        self.sm, self.reasons = [], set()

    def summary(self):
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.sm_max,
                "reasons": sorted(self.reasons), "samples": len(self.sm), "source": self.source}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    pop = population(args)
    table, mlp_w, _ = build_operators()
    chi = "table" if args.chi == "table" else "mlp"
    v, t, pairs, sample = time_oracle(pop, chi, table, mlp_w, args.steps, args.warmup,
                                      target_pairs=2_000_000 if chi == "table" else 150_000)
    total_pairs = pop.pairs_per_step(-1)
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(args, pop, total_pairs),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_2602_21244_b200 import dsmc

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hbm_peak, tc_burst, tc_sust, peak_src = peaks()

    pop = population(args, rank)       # weak scaling: every rank owns one full cfg-5 population
    # the product arm builds its chi table with the product (dsmc_build_chi_table_lj: the LJ quadrature on the
    # device); oracle/ is touched only by the cpu_baseline leg at the end
    from paper_2602_21244_b200 import workloads as wl
    mlp_w = wl.random_mlp(3, [2, 128, 128, 1])
    pairs = pop.pairs_per_step(-1)
    ctx = dsmc.Context(pop.n, pop.n_cells, device=local)
    t0 = time.perf_counter()
    ctx.build_chi_table_lj(TABLE_N, TABLE_N, b_max=B_MAX)
    torch.cuda.synchronize()
    t_table = time.perf_counter() - t0
    ctx.set_mlp(1, mlp_w[0], mlp_w[1], dsmc.ACT_SILU)
    dev = torch.device("cuda", local)
    cell = torch.from_numpy(pop.cell).to(dev)
    vin = [torch.from_numpy(a).to(dev) for a in (pop.vx, pop.vy, pop.vz)]
    out = (torch.empty(pop.n, dtype=torch.float32, device=dev), torch.empty(pop.n, dtype=torch.float32, device=dev),
           torch.empty(pop.n, dtype=torch.float32, device=dev), torch.empty(pop.n, dtype=torch.int32, device=dev),
           torch.empty(pop.n_cells + 1, dtype=torch.int32, device=dev))

    def params(chi):
        flags = dsmc.F_MOMENT_MATCH | (dsmc.F_BF16_TC if chi.startswith("mlp_tc") else 0) | \
            (dsmc.F_TC_ONE_KERNEL if chi == "mlp_tc_one_kernel" else 0) | \
            (dsmc.F_PAIR_REPLACE if chi.endswith("_replace") else 0)
        return dsmc.AbinitioParams(chi_mode=0 if chi.startswith("table") else 1, flags=flags, b_max=B_MAX)

    def one_step(chi, t, ev=None):
        ctx.bin(cell, *vin, pop.n_cells, out=out)
        if ev is not None:
            ev[0].record()
        ctx.collide_abinitio(out[4], out[0], out[1], out[2], params(chi), seed=4, step=t)
        if ev is not None:
            ev[1].record()

    def timed(chi, steps, warmup, sampler=None):
        for t in range(warmup):
            one_step(chi, t)
        ctx.check()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        if sampler is not None:
            sampler.mark()
        l0 = ctx.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for t in range(steps):
            one_step(chi, warmup + t, evs[t])
        e1.record()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        ms = e0.elapsed_time(e1)
        coll_ms = float(np.mean([a.elapsed_time(b) for a, b in evs]))
        if world > 1:
            tt = torch.tensor([ms], device=dev)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            ms = tt.item()
        return ms / steps, coll_ms, ctx.launch_count() - l0

    sampler = ClockSampler(local)
    sampler.start()
    ms_step, coll_ms, launches = timed(args.chi, args.steps, args.warmup, sampler)
    sampler.stop_flag = True
    sampler.join(timeout=2)
    st = ctx.sync_status()
    if st != 0:
        raise SystemExit("device status %d (%s)" % (st, dsmc.strerror(st)))

    # end to end through the C-ABI host entry point: pinned host buffers, H2D + D2H inside the timing
    hcell = torch.from_numpy(pop.cell).pin_memory()
    hv = [torch.from_numpy(a).pin_memory() for a in (pop.vx, pop.vy, pop.vz)]
    hout = [torch.empty(pop.n, dtype=torch.float32).pin_memory() for _ in range(3)] + \
           [torch.empty(pop.n, dtype=torch.int32).pin_memory(), torch.empty(pop.n_cells + 1, dtype=torch.int32).pin_memory()]
    e2e_steps = max(6, min(args.steps, 12))
    for t in range(2):
        ctx.step_host(hcell, *hv, pop.n_cells, hout, abi=params(args.chi), seed=4, step=t)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for t in range(e2e_steps):
        ctx.step_host(hcell, *hv, pop.n_cells, hout, abi=params(args.chi), seed=4, step=10 + t)
    torch.cuda.synchronize()
    e2e_sync_s = (time.perf_counter() - t0) / e2e_steps
    # the same through three contexts on three streams fed in turn (dsmc_step_host_submit / dsmc_sync_status): every
    # step still copies its inputs in and its results out, but the H2D of one batch runs under the D2H of an earlier one
    # and under the kernels of another (two lanes leave the link idle while a lane computes)
    N_LANES = 3
    extra_ctx = []
    lanes = [(ctx, torch.cuda.Stream(device=dev), hout)]
    for _ in range(N_LANES - 1):
        cx = dsmc.Context(pop.n, pop.n_cells, device=local)
        cx.build_chi_table_lj(TABLE_N, TABLE_N, b_max=B_MAX)
        cx.set_mlp(1, mlp_w[0], mlp_w[1], dsmc.ACT_SILU)
        extra_ctx.append(cx)
        lanes.append((cx, torch.cuda.Stream(device=dev), [torch.empty_like(t).pin_memory() for t in hout]))
    torch.cuda.synchronize()

    def pipelined(first, count):
        busy = [False] * N_LANES
        for t in range(count):
            k = t % N_LANES
            c, st, ho = lanes[k]
            if busy[k]:
                with torch.cuda.stream(st):
                    c.check()
            with torch.cuda.stream(st):
                c.step_host(hcell, *hv, pop.n_cells, ho, abi=params(args.chi), seed=4, step=first + t, submit_only=True)
            busy[k] = True
        for k in range(N_LANES):
            if busy[k]:
                with torch.cuda.stream(lanes[k][1]):
                    lanes[k][0].check()

    pipelined(100, N_LANES)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    pipelined(110, e2e_steps)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    for cx in extra_ctx:
        cx.close()
    if world > 1:
        tt = torch.tensor([e2e_s, e2e_sync_s], device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e_s, e2e_sync_s = tt.tolist()
    h2d = pop.n * 16
    d2h = pop.n * 16 + (pop.n_cells + 1) * 4

    variants = {}
    if not args.no_variants and rank == 0 or (not args.no_variants and world > 1):
        # table_replace: the same step with pairs drawn WITH replacement (DSMC_F_PAIR_REPLACE)
        for chi in ("table", "mlp", "mlp_tc", "mlp_tc_one_kernel", "table_replace", "mlp_tc_replace"):
            if chi == args.chi:
                variants[chi] = {"pairs_per_s": pairs / (ms_step * 1e-3), "collide_ms": coll_ms, "step_ms": ms_step}
                continue
            try:
                m, c, _ = timed(chi, max(3, args.steps // 4), 2)
                variants[chi] = {"pairs_per_s": pairs / (m * 1e-3), "collide_ms": c, "step_ms": m}
            except dsmc.DsmcError as e:
                variants[chi] = {"unavailable": str(e)}

    # cfg 4 (a10): chi for 1e7 independent pairs, table and tensor-core MLP (context for the MLP engine alone)
    cfg4 = {}
    if not args.no_variants and rank == 0:
        from paper_2602_21244_b200 import workloads as wl
        n4 = int(10_000_000 * args.scale)
        E4, b4 = wl.abinitio_pair_batch(seed=3, n=n4)
        E4d, b4d = torch.from_numpy(E4).to(dev), torch.from_numpy(b4).to(dev)
        o4 = torch.empty_like(E4d)
        for name, mode, fl in (("table", 0, 0), ("mlp_tc", 1, dsmc.F_BF16_TC)):
            for _ in range(3):
                ctx.chi_batch(E4d, b4d, mode, B_MAX, flags=fl, out=o4)
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a0.record()
            for _ in range(10):
                ctx.chi_batch(E4d, b4d, mode, B_MAX, flags=fl, out=o4)
            a1.record()
            torch.cuda.synchronize()
            ms4 = a0.elapsed_time(a1) / 10
            cfg4[name] = {"ms": ms4, "pairs_per_s": n4 / (ms4 * 1e-3)}
        # the computation the operators above replace: deflection-integral quadrature per pair
        for _ in range(2):
            ctx.chi_exact_batch(E4d, b4d, out=o4)
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a0.record()
        for _ in range(3):
            ctx.chi_exact_batch(E4d, b4d, out=o4)
        a1.record()
        torch.cuda.synchronize()
        msx = a0.elapsed_time(a1) / 3
        cfg4["exact_quadrature_fp64"] = {"ms": msx, "pairs_per_s": n4 / (msx * 1e-3),
                                         "table_speedup": msx / cfg4["table"]["ms"],
                                         "mlp_tc_speedup": msx / cfg4["mlp_tc"]["ms"]}
        # (f2) the 1024 x 1024 LJ table generated on the device by the same quadrature (the oracle builds it on one
        # host core in table_build_s seconds; the paper's exact 512 x 512 table took hours on a CPU cluster)
        ctx_t = dsmc.Context(16, 1, device=local)
        ctx_t.build_chi_table_lj(TABLE_N, TABLE_N, b_max=B_MAX)
        torch.cuda.synchronize()
        tb0 = time.perf_counter()
        ctx_t.build_chi_table_lj(TABLE_N, TABLE_N, b_max=B_MAX)
        torch.cuda.synchronize()
        cfg4["table_build_on_device_ms"] = (time.perf_counter() - tb0) * 1e3
        # (f2 as the paper states it) the table generated by the chi-MLP on its nodes; paper: "< 1.0 s" for 512 x 512
        ctx_t.set_mlp(1, mlp_w[0], mlp_w[1], dsmc.ACT_SILU)
        for key, nn_, fl in (("table_build_from_mlp_512_tc_ms", 512, dsmc.F_BF16_TC), ("table_build_from_mlp_512_fp32_ms", 512, 0),
                             ("table_build_from_mlp_1024_tc_ms", TABLE_N, dsmc.F_BF16_TC)):
            ctx_t.build_chi_table_mlp(nn_, nn_, flags=fl)
            torch.cuda.synchronize()
            tb0 = time.perf_counter()
            ctx_t.build_chi_table_mlp(nn_, nn_, flags=fl)
            torch.cuda.synchronize()
            cfg4[key] = (time.perf_counter() - tb0) * 1e3
        ctx_t.close()
        fl4 = n4 * 2 * (2 * 128 + 128 * 128 + 128)
        cfg4["mlp_tc"]["tensor_frac"] = fl4 / (cfg4["mlp_tc"]["ms"] * 1e-3) / 1e12 / tc_sust
        cfg4["table"]["hbm_frac"] = n4 * 12 / (cfg4["table"]["ms"] * 1e-3) / 1e9 / hbm_peak
        del E4d, b4d, o4

    # (f4) the whole DSMC loop around the step on the same population laid out as a 1-D channel: move + Maxwell walls
    # -> bin -> gather x -> fused collide (table) -> sample, on the device (dsmc_couette_run); the input of every
    # bin is the previous step's sorted order after one free flight, as in a running simulation
    loop = {}
    if not args.no_loop and rank == 0:
        rng = np.random.default_rng(11)
        rt = float((pop.vx.astype(np.float64) ** 2 + pop.vy.astype(np.float64) ** 2 + pop.vz.astype(np.float64) ** 2).mean() / 3)
        dx = 1.0e-4
        geo = dsmc.CouetteParams(L=dx * pop.n_cells, dt=0.3 * dx / math.sqrt(rt), u_wall=500.0, rt_wall=rt,
                                 accommodation=1.0, n_cells=pop.n_cells)
        xs = torch.from_numpy(((pop.cell + rng.random(pop.n)) * dx).astype(np.float32)).to(dev)
        vs = [v.clone() for v in vin]
        acc = torch.zeros((pop.n_cells, 8), dtype=torch.float64, device=dev)
        n_loop = max(5, args.steps // 2)
        ctx.couette_run(xs, *vs, geo, 3, abi=params("table"), seed=4, step0=0, sample_from=0, acc=acc)
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        l0 = ctx.launch_count()
        a0.record()
        ctx.couette_run(xs, *vs, geo, n_loop, abi=params("table"), seed=4, step0=3, sample_from=0, acc=acc)
        a1.record()
        torch.cuda.synchronize()
        loop = {"ms_per_step": a0.elapsed_time(a1) / n_loop, "steps": n_loop,
                "launches_per_step": (ctx.launch_count() - l0) / n_loop}
        cellb = torch.empty(pop.n, dtype=torch.int32, device=dev)
        for name, fn in (("move_ms", lambda t: ctx.move_couette(xs, *vs, geo, seed=4, step=100 + t, cell=cellb)),
                         ("gather_ms", lambda t: ctx.gather_f32(out[3], xs, out=out[0])),
                         ("sample_ms", lambda t: ctx.sample_cells(out[4], out[0], out[1], out[2], acc))):
            fn(0)
            torch.cuda.synchronize()
            a0.record()
            for t in range(5):
                fn(1 + t)
            a1.record()
            torch.cuda.synchronize()
            loop[name] = a0.elapsed_time(a1) / 5
        loop["pairs_per_s"] = pairs / (loop["ms_per_step"] * 1e-3)
        del xs, vs, acc, cellb

    # the paper's other two population shapes (north_star: "Couette, cavity and Mach 10 cylinder"): cfg 2 and cfg 3
    # with the VHS-surrogate MLP 8->128->128->3 (random init), FP32 and tensor-core paths; step = bin + fused collide.
    # These are 1e5 / 5e5 pairs per step: launch- and latency-bound, reported for completeness (not the headline).
    other = {}
    if not args.no_variants and rank == 0:
        from paper_2602_21244_b200 import workloads as wl
        for name, popf, ppc, sw in (("cfg2_couette_200x1000", wl.couette, 500, 1), ("cfg3_cavity_100x100x100", wl.cavity, 50, 2)):
            p2 = popf()
            c2 = dsmc.Context(p2.n, p2.n_cells, device=local)
            Ws, bs = wl.random_mlp(sw, [8, 128, 128, 3])
            c2.set_mlp(0, Ws, bs, dsmc.ACT_TANH)
            cell2 = torch.from_numpy(p2.cell).to(dev)
            v2 = [torch.from_numpy(a).to(dev) for a in (p2.vx, p2.vy, p2.vz)]
            o2 = (torch.empty(p2.n, dtype=torch.float32, device=dev), torch.empty(p2.n, dtype=torch.float32, device=dev),
                  torch.empty(p2.n, dtype=torch.float32, device=dev), torch.empty(p2.n, dtype=torch.int32, device=dev),
                  torch.empty(p2.n_cells + 1, dtype=torch.int32, device=dev))
            pairs2 = p2.pairs_per_step(ppc)
            other[name] = {"pairs_per_step": int(pairs2)}
            for path, fl in (("fp32", 0), ("bf16_tc", dsmc.F_BF16_TC)):
                prm2 = dsmc.VhsParams(sigma_v=wl.SIGMA_V, pairs_per_cell=ppc,
                                      flags=dsmc.F_NOISE | dsmc.F_ENERGY_SHELL | dsmc.F_MOMENT_MATCH | fl)
                for t in range(3):
                    c2.bin(cell2, *v2, p2.n_cells, out=o2)
                    c2.collide_vhs_nn(o2[4], o2[0], o2[1], o2[2], prm2, seed=sw, step=t)
                a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
                a0.record()
                for t in range(20):
                    c2.bin(cell2, *v2, p2.n_cells, out=o2)
                    ev2[t][0].record()
                    c2.collide_vhs_nn(o2[4], o2[0], o2[1], o2[2], prm2, seed=sw, step=3 + t)
                    ev2[t][1].record()
                a1.record()
                torch.cuda.synchronize()
                ms2 = a0.elapsed_time(a1) / 20
                other[name][path] = {"step_ms": ms2, "collide_ms": float(np.mean([a.elapsed_time(b) for a, b in ev2])),
                                     "pairs_per_s": pairs2 / (ms2 * 1e-3)}
            st2 = c2.sync_status()
            if st2 != 0:
                other[name]["status"] = int(st2)
            c2.close()
            del cell2, v2, o2

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # roofline of the dominant kernel (the fused collide kernel), north_star definition:
    # the slower of the MLP FLOPs at tensor peak and the gathered + written bytes at HBM bandwidth
    bytes_alg = pop.n * 24 + (pop.n_cells + 1) * 4
    flops_alg = pairs * 2 * (2 * 128 + 128 * 128 + 128) if args.chi != "table" else 0
    t_hbm = bytes_alg / (hbm_peak * 1e9)
    t_tc = flops_alg / (tc_sust * 1e12)
    if t_tc > t_hbm:
        roof = {"bound": "tensor", "achieved": flops_alg / (coll_ms * 1e-3) / 1e12, "peak": tc_sust, "unit": "TFLOP/s"}
    else:
        roof = {"bound": "hbm", "achieved": bytes_alg / (coll_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    if args.chi != "table":
        # extended bound: one MUFU per hidden activation, 16 / clk / SM (measured), at the
        # SM clock sampled during the run
        clk = (sampler.summary().get("sm_mhz") or 1965.0) * 1e6
        t_xu = pairs * 256 / (16.0 * 148 * clk)
        roof["xu_bound"] = {"ms": t_xu * 1e3, "frac": t_xu / (coll_ms * 1e-3)}
    roof["traffic"], roof["traffic_source"] = measured_traffic("table" if args.chi == "table" else args.chi)
    roof["kernel"] = {"table": "fused collide: dsmc::k_cells (+ k_cell_lists, k_cells_big)",
                      "mlp_tc": "fused collide, three passes: dsmc::k_cells<3> | k_chi_batch_tc | k_cells<4> (+ k_cell_lists x2, k_cells_big x2)"}.get(args.chi, "fused collide: dsmc::k_collide<fp32 MLP>")
    roof["kernel_ms"] = coll_ms
    roof["peak_source"] = peak_src
    roof["algorithmic"] = {"bytes_per_launch": bytes_alg, "flops_per_launch": flops_alg}
    bin_ms = ms_step - coll_ms
    roof["bin"] = {"ms": bin_ms, "achieved_gbs": pop.n * 36 / (bin_ms * 1e-3) / 1e9, "frac": pop.n * 36 / (bin_ms * 1e-3) / 1e9 / hbm_peak}

    line = {"metric": METRIC, "value": world * pairs / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32" if args.chi != "mlp_tc" else "bf16", "data": "synthetic",
            "config": config_dict(args, pop, pairs), "clocks": sampler.summary(),
            "e2e": {"value": world * pairs / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_s * 1e3,
                    "api": "dsmc_step_host_submit + dsmc_sync_status, three contexts on three streams fed in turn "
                           "(pinned host buffers; every step copies its inputs in and its results out)",
                    "single_context_sync": {"value": world * pairs / e2e_sync_s, "ms_per_step": e2e_sync_s * 1e3,
                                            "api": "dsmc_step_host"}},
            "gpu_launches": int(launches), "roofline": roof, "variants": variants, "cfg4_chi_batch": cfg4, "couette_loop": loop, "other_workloads": other,
            "table_build_s": t_table}
    if not args.no_cpu_baseline and world >= 1:
        chi = "table" if args.chi == "table" else "mlp"
        table, _, _ = build_operators()
        v, t, sp, sample = time_oracle(pop, chi, table, mlp_w, steps=3, warmup=1,
                                       target_pairs=4_000_000 if chi == "table" else 300_000)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                                "host": host_info()}
        try:  # the same oracle on every host core (it is a baseline, not the target)
            va, ta, pa, ca, sa = time_oracle_all_cores(pop, chi, table, mlp_w, 400_000 if chi == "table" else 30_000)
            line["cpu_baseline"]["all_cores"] = {"value": va, "unit": UNIT, "cores": ca, "seconds": ta, "sample": sa}
        except Exception as e:  # a host without fork / affinity: the single-thread figure stands
            line["cpu_baseline"]["all_cores"] = {"unavailable": repr(e)[:200]}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
