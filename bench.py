#!/usr/bin/env python
"""bench.py -- times the whole near-field hot path (nf_bin + nf_accel, all SURVEY.md 8(a) rows) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference] [--per-config LIST]

One "step" = one pass of the whole hot path over one batch of synthetic input: nf_bin (cell ids, histogram,
prefix sums, stable sort, gather, scheduling) followed by nf_accel (direct sum + scatter to input order).
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "near_field_pair_interactions_per_s"
UNIT = "interactions/s"
FLOPS_PER_INTERACTION = 25      # 3 add + 8 fma(2) + 3 mul + 1 min + rsqrt(2): SURVEY.md 8(a) S6; the paper counts 26
FLOPS_EXECUTED_MIN = 19         # the Newtonian body (3 add + 6 fma + 2 mul + rsqrt) the kernel runs where no pair is inside eps_s
L2_BYTES = 126 * 1024 * 1024
# ncu numbers are never measured by this run: they are READ from the committed capture summaries (one row per workload:
# workload, dram bytes read, dram bytes written per direct_kernel launch, FMA-pipe busy %, issue-slot %, file of origin)
NCU_TABLE = os.path.join(ROOT, "profiles", "r2_direct_kernel_counters.csv")


def ncu_counters(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum (and the pipe counters) of one direct_kernel launch from the committed
    `ncu --set full` capture of this workload, or None when no capture of it is committed."""
    try:
        import csv
        with open(NCU_TABLE) as f:
            for row in csv.DictReader(l for l in f if not l.startswith("#")):
                if row["workload"] == workload:
                    return {"traffic": int(float(row["dram_bytes_read"])) + int(float(row["dram_bytes_write"])),
                            "fma_pipe_busy_pct": float(row["sm__pipe_fma_cycles_active_pct"]),
                            "issue_active_pct": float(row["smsp__issue_active_pct"]),
                            "source": "profiles/" + row["source"]}
    except (OSError, KeyError, ValueError):
        pass
    return None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config (1-based); default 3 = uniform 256^3")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--per-config", default="1,2,4,5",
                    help="extra configs reported in 'per_config' (N=1 only, 3 warm-ups + 3 steps; config 5: 1 + 1); '' = none")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-density", action="store_true", help="skip the fused-density timing")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slabs"],
                    help="N > 1: 'replicas' (the contract: one GPU per problem, no sharding) or 'slabs' (ONE box split "
                         "into x-slab ranges with an R-slab halo exchange inside every step: strong scaling)")
    ap.add_argument("--occupancy-sweep", default=None, metavar="CPD[,CPD...]",
                    help="instead of a config: 200^3 uniform particles binned into CPD^3 cells for every CPD of the list "
                         "(default list with an empty string: 49,63,79,100,126,159 = 68 ... 2 particles per cell), nf_accel only: "
                         "the void regime of the direct kernel (PAPER.md:512)")
    ap.add_argument("--variant", type=int, default=None)
    ap.add_argument("--fastpath", type=int, default=None)
    ap.add_argument("--heavy-first", type=int, default=None)
    ap.add_argument("--ctas-per-sm", type=int, default=None)
    ap.add_argument("--window", type=int, default=None, help="sink slots per work unit (nf_set_option window)")
    ap.add_argument("--flat-below", type=int, default=None, help="nf_set_option flat_below (0: never take the flat loop)")
    return ap.parse_args()


# ------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.1):
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self.period = period
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "hw_power_brake_slowdown": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_min_mhz": min(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------ oracle leg
def oracle_sample_rate(pos_np, cfg, target_s=12.0):
    """Times the oracle as it stands on a bounded sink sample of this workload (about target_s of CPU work).
    Returns (interactions/s, description, seconds, cores)."""
    import numpy as np
    import oracle
    t0 = time.time()
    b = oracle.bin_particles(pos_np, cfg.cpd, cfg.L)
    t_bin = time.time() - t0
    rng = np.random.default_rng(12345)
    n = pos_np.shape[0]
    cnt = b["count"].astype(np.int64).reshape(cfg.cpd, cfg.cpd, cfg.cpd)
    box = np.zeros_like(cnt)
    R = cfg.R
    for ox in range(-R, R + 1):
        for oy in range(-R, R + 1):
            for oz in range(-R, R + 1):
                box += np.roll(cnt, (ox, oy, oz), axis=(0, 1, 2))
    per_sink = box.reshape(-1)[b["cid"]]                   # sources per sink
    # pilot to get the rate, then size the sample
    pilot = rng.choice(n, size=min(n, 2000), replace=False)
    t0 = time.time()
    oracle.accel(pos_np, cfg.cpd, cfg.L, cfg.eps, cfg.R, sinks=pilot, binning=b)
    dt = max(time.time() - t0, 1e-4)
    rate = per_sink[pilot].sum() / dt
    want = rate * target_s
    m = int(min(n, max(2000, want / max(per_sink.mean(), 1.0))))
    sinks = rng.choice(n, size=m, replace=False)
    t0 = time.time()
    oracle.accel(pos_np, cfg.cpd, cfg.L, cfg.eps, cfg.R, sinks=sinks, binning=b)
    dt = time.time() - t0
    inter = int(per_sink[sinks].sum())
    desc = (f"{m} random sinks of {cfg.name} (all {n} particles binned by the oracle in {t_bin:.1f}s, "
            f"{inter:.3e} pair interactions summed in {dt:.1f}s)")
    return inter / dt, desc, dt, oracle.num_threads(), inter, m


# ------------------------------------------------------------------------------------ GPU arm
def fp32_peak_tflops(stats):
    """SM count x 128 lanes x 2 flops x max SM clock, read from the device (BASELINE.json north_star)."""
    return stats["sm_count"] * 128 * 2 * stats["clock_khz"] * 1e3 / 1e12


def apply_options(plan, args):
    for key, val in (("variant", args.variant), ("fastpath", args.fastpath), ("heavy_first", args.heavy_first),
                     ("ctas_per_sm", args.ctas_per_sm), ("window", args.window), ("flat_below", args.flat_below)):
        if val is not None:
            plan.set_option(key, val)


def time_device_steps(plan, pos, acc, steps, warmup, flush, dist=None):
    """W warm-up steps, then exactly K timed steps between barrier + synchronize on both sides.
    Returns (total_ms, [accel_ms per step], [bin_ms per step])."""
    import torch
    for _ in range(warmup):
        plan.bin(pos)
        plan.accel(acc)
    torch.cuda.synchronize()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    for k in range(steps):
        if flush is not None:
            flush.add_(1)                      # > L2 bytes written between iterations
        ev[k][0].record()
        plan.bin(pos)
        ev[k][1].record()
        plan.accel(acc)
        ev[k][2].record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    bin_ms = [e[0].elapsed_time(e[1]) for e in ev]
    acc_ms = [e[1].elapsed_time(e[2]) for e in ev]
    total = sum(bin_ms) + sum(acc_ms)          # excludes the L2 flush writes, includes every kernel of the path
    return total, acc_ms, bin_ms


def time_e2e_steps(plan, pos_host, acc_host, steps, warmup):
    """Same metric through the C-ABI with HOST (pinned) buffers: H2D of the positions and D2H of the
    accelerations are inside every timed step.  Wall clock around synchronous calls (nf_accel_host syncs)."""
    import torch
    for _ in range(max(1, min(warmup, 2))):
        plan.bin_host(pos_host)
        plan.accel_host(acc_host)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        plan.bin_host(pos_host)
        plan.accel_host(acc_host)
    torch.cuda.synchronize()
    return (time.perf_counter() - t0) * 1e3


def time_e2e_two_in_flight(make_plan, pos_host, steps):
    """The same host-buffer calls with TWO independent problems in flight: two plans, two streams, two host threads (ctypes
    releases the GIL in the calls), each looping nf_bin_host + nf_accel_host on its own pinned output buffer.  The PCIe
    copies of one problem run under the kernel of the other -- inside one call they cannot: the binning needs every position
    before the first unit starts and the accelerations are complete only when the last unit ends.  Returns (ms, steps done)."""
    import threading
    import torch
    plans = [make_plan(), make_plan()]
    streams = [torch.cuda.Stream() for _ in plans]
    outs = [torch.empty(pos_host.shape, dtype=pos_host.dtype, pin_memory=True) for _ in plans]
    per_thread = max(6, 2 * steps)                  # the first H2D and the last D2H have nothing to hide behind
    gate = threading.Barrier(3)
    errs = []

    def work(i):
        try:
            torch.cuda.set_device(pos_dev_index)
            with torch.cuda.stream(streams[i]):
                plans[i].bin_host(pos_host)
                plans[i].accel_host(outs[i])           # warm-up: staging buffers, workspace
                gate.wait()
                for _ in range(per_thread):
                    plans[i].bin_host(pos_host)
                    plans[i].accel_host(outs[i])
        except Exception as e:                         # noqa: BLE001
            errs.append(e)
            try:
                gate.abort()
            except Exception:                          # noqa: BLE001
                pass

    pos_dev_index = torch.cuda.current_device()
    th = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    try:
        gate.wait()
    except threading.BrokenBarrierError:
        pass
    t0 = time.perf_counter()
    for t in th:
        t.join()
    torch.cuda.synchronize()
    ms = (time.perf_counter() - t0) * 1e3
    same = bool(torch.equal(outs[0], outs[1]))
    for pl in plans:
        pl.close()
    if errs:
        raise errs[0]
    return ms, 2 * per_thread, same


def max_over_ranks(values, dist=None, device="cpu"):
    """Replicas only: the ranks share no data; the one collective of the harness is the MAX of the timings."""
    import torch
    if dist is None:
        return list(values)
    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def aggregate_value(world, interactions, steps, total_ms):
    """Whole-job interactions/s of `world` independent replicas that each ran `steps` steps in `total_ms` (max over ranks)."""
    return world * interactions * steps / (total_ms / 1e3)


def occupancy_stats(plan, cfg):
    """Realised cell occupancy of the workload and where the interactions sit; harness-side torch."""
    import torch
    cnt = plan.binning()["count"].to(torch.int64).reshape(cfg.cpd, cfg.cpd, cfg.cpd)
    box = torch.zeros_like(cnt)
    for ox in range(-cfg.R, cfg.R + 1):
        for oy in range(-cfg.R, cfg.R + 1):
            for oz in range(-cfg.R, cfg.R + 1):
                box += torch.roll(cnt, (ox, oy, oz), (0, 1, 2))
    inter = (cnt * box).reshape(-1)
    top = max(1, inter.numel() // 100)
    heavy = torch.topk(inter, top).values.sum().item()
    c = cnt.reshape(-1)
    return {"max_per_cell": int(c.max().item()), "median_per_cell": float(c.median().item()),
            "mean_per_cell": float(c.double().mean().item()), "empty_cells": int((c == 0).sum().item()),
            "interactions_check": int(inter.sum().item()),
            "share_of_interactions_in_heaviest_1pct_cells": heavy / max(1, inter.sum().item())}


def run_config(idx, args, device_index, dist=None, with_e2e=True, steps=None, warmup=None):
    import torch
    import nf_inputs
    import paper_2110_11398_b200 as nf
    cfg = nf_inputs.config(idx)
    steps = steps or args.steps
    warmup = warmup if warmup is not None else args.warmup
    gen_dev = "cuda" if cfg.n > 20_000_000 else "cpu"
    pos = nf_inputs.generate(cfg, device=gen_dev).cuda()
    torch.cuda.empty_cache()                   # the generator's temporaries (FFT grids) go back to the driver
    acc = torch.empty_like(pos)
    input_bytes = pos.numel() * 4
    flush = None
    if input_bytes * 3 < 2 * L2_BYTES:         # small configs: flush L2 between timed iterations
        flush = torch.zeros(2 * L2_BYTES // 4, dtype=torch.int32, device="cuda")
    out = {"name": cfg.name, "n": cfg.n, "cpd": cfg.cpd}
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
        apply_options(plan, args)
        with ClockSampler(device_index) as clk:
            total_ms, acc_ms, bin_ms = time_device_steps(plan, pos, acc, steps, warmup, flush, dist)
        st = plan.stats()
        out["clocks"] = clk.summary()
        I = st["interactions"]
        out.update(stats=st, interactions=I, total_ms=total_ms, accel_ms=acc_ms, bin_ms=bin_ms, steps=steps,
                   l2="flushed between iterations (256 MiB write)" if flush is not None else "inputs exceed L2")
        out["occupancy"] = occupancy_stats(plan, cfg)
        a = acc.double()
        out["sum_check"] = float((a.sum(0).abs().max() / a.abs().sum()).item())   # total force ~ 0 at any size
        if with_e2e and not args.no_density:
            # the same pass with the fused kernel density estimate (b = 0.4 spacings)
            rho = torch.empty(pos.shape[0], dtype=torch.float32, device="cuda")
            b = 0.4 * cfg.L / cfg.n_side
            evd = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            for _ in range(2):
                plan.accel_density(b, acc, rho)
            torch.cuda.synchronize()
            evd[0].record()
            for _ in range(steps):
                plan.accel_density(b, acc, rho)
            evd[1].record()
            torch.cuda.synchronize()
            out["density_ms_accel"] = evd[0].elapsed_time(evd[1]) / steps
            out["density_mean"] = float(rho.double().mean().item())
            del rho
            # kick and per-cell max |a| fused into the epilogue
            vel = torch.zeros_like(pos)
            amax = torch.empty(cfg.cpd ** 3, dtype=torch.float32, device="cuda")
            nf.nf_accel_kick(plan._h, acc, vel, 1e-6, amax)
            torch.cuda.synchronize()
            evd[0].record()
            for _ in range(steps):
                nf.nf_accel_kick(plan._h, acc, vel, 1e-6, amax)
            evd[1].record()
            torch.cuda.synchronize()
            out["kick_ms_accel"] = evd[0].elapsed_time(evd[1]) / steps
            out["amax_global"] = float(amax.max().item())
            del vel, amax
            # per-particle source masses (nf_set_masses; fourth staged array, one FMUL2 per pair)
            mass = nf_inputs.masses(cfg, device="cuda")
            evm = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            plan.set_masses(mass)
            plan.accel(acc)
            torch.cuda.synchronize()
            evm[0].record()
            plan.set_masses(mass)
            evm[1].record()
            for _ in range(steps):
                plan.accel(acc)
            evm[2].record()
            torch.cuda.synchronize()
            out["mass_ms_set"] = evm[0].elapsed_time(evm[1])
            out["mass_ms_accel"] = evm[1].elapsed_time(evm[2]) / steps
            plan.set_masses(None)
            del mass
        if with_e2e:
            # nf_rebin (the same particles after a drift of 0.004 cell widths rms, ~1 % of them change
            # cell) beside the full nf_bin, for the generated (random) input order and for a caller that keeps its arrays in
            # the library's cell order (pos[perm]); restores the timed binning afterwards
            g = torch.Generator(device="cuda").manual_seed(4242)
            cell = cfg.L / cfg.cpd
            q = pos.clone()
            rb = {}
            for label in ("input_order_as_generated", "input_in_cell_order"):
                plan.bin(q)
                plan.bin(q)
                full_ms = plan.stats()["ms_bin"]
                t, movers, paths = [], [], []
                for _ in range(3):
                    q = torch.remainder(q + torch.randn(q.shape, generator=g, device="cuda") * (0.004 * cell), cfg.L)
                    q[q >= cfg.L] = 0
                    q = q.contiguous()
                    torch.cuda.synchronize()
                    plan.rebin(q)
                    sr = plan.stats()
                    t.append(sr["ms_bin"]); movers.append(sr["rebin_movers"]); paths.append(sr["rebin_path"])
                rb[label] = {"ms_nf_bin": full_ms, "ms_nf_rebin": statistics.median(t), "speedup": full_ms / statistics.median(t),
                             "movers_frac": statistics.median(movers) / cfg.n, "path": paths}
                q = q[plan.binning()["perm"].long()].contiguous()
            out["rebin"] = rb
            del q
            plan.bin(pos)
            pos_h = torch.empty(pos.shape, dtype=pos.dtype, pin_memory=True)
            pos_h.copy_(pos)
            acc_h = torch.empty(pos.shape, dtype=pos.dtype, pin_memory=True)
            del pos, acc, a                    # the host path stages through plan-owned device buffers
            pos = acc = None
            torch.cuda.empty_cache()
            e_steps = max(1, min(steps, 3))
            out["e2e_ms"] = time_e2e_steps(plan, pos_h, acc_h, e_steps, warmup)
            out["e2e_steps"] = e_steps
            if cfg.n <= 64_000_000:            # two more plans: 2 x (workspace + two staging buffers)
                def make_plan():
                    pl = nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R)
                    apply_options(pl, args)
                    return pl
                try:                           # an extra figure: its failure must not cost the line
                    out["e2e2_ms"], out["e2e2_steps"], out["e2e2_same"] = time_e2e_two_in_flight(make_plan, pos_h, e_steps)
                except Exception as e:         # noqa: BLE001
                    sys.stderr.write(f"two_problems_in_flight leg skipped: {e!r}\n")
            out["pos_host"] = pos_h
    del pos, acc
    torch.cuda.empty_cache()
    return out, cfg


def summarise(r):
    st = r["stats"]
    I, n = r["interactions"], r["n"]
    t = r["total_ms"] / 1e3 / r["steps"]
    ta = statistics.mean(r["accel_ms"]) / 1e3
    peak = fp32_peak_tflops(st)
    return {
        "workload": r["name"], "n": n, "interactions": I,
        "interactions_per_s": I / t, "particle_updates_per_s": n / t,
        "accel_only_interactions_per_s": I / ta,
        "ms_per_step": t * 1e3, "ms_bin": statistics.mean(r["bin_ms"]), "ms_accel": ta * 1e3,
        "fp32_peak_frac_25flop": FLOPS_PER_INTERACTION * I / ta / 1e12 / peak,
        "fp32_peak_frac_26flop_paper": 26 * I / ta / 1e12 / peak,
        "sum_check": r["sum_check"], "l2": r["l2"], "clocks": r["clocks"], "occupancy": r["occupancy"],
    }


def main_b200(args):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    r, cfg = run_config(args.config, args, local, dist)
    st = r["stats"]
    t_total = r["total_ms"]
    e2e_ms = r["e2e_ms"]
    t_total, e2e_ms = max_over_ranks([t_total, e2e_ms], dist, "cuda")   # replicas only, no data-path collective
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    s = summarise(r)
    I, n, K = r["interactions"], r["n"], r["steps"]
    value = aggregate_value(world, I, K, t_total)
    ta = statistics.mean(r["accel_ms"]) / 1e3
    peak = fp32_peak_tflops(st)
    achieved = FLOPS_PER_INTERACTION * I / ta / 1e12
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": t_total / K, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg.name, "n": n, "cpd": cfg.cpd, "R": cfg.R, "eps": cfg.eps, "L": cfg.L,
                   "interactions_per_step": I, "l2": r["l2"], "multi_gpu": "replicas only (no collective)",
                   "occupancy": r["occupancy"],
                   "flops_per_interaction": FLOPS_PER_INTERACTION},
        "particle_updates_per_s": world * n * K / (t_total / 1e3),
        "fp32_peak_frac": s["fp32_peak_frac_25flop"], "fp32_peak_frac_26flop_paper": s["fp32_peak_frac_26flop_paper"],
        "ms_bin": s["ms_bin"], "ms_accel": s["ms_accel"],
        "e2e": {"value": world * I * r["e2e_steps"] / (e2e_ms / 1e3), "unit": UNIT, "h2d_bytes_per_step": 12 * n,
                "d2h_bytes_per_step": 12 * n, "steps": r["e2e_steps"], "ms_per_step": e2e_ms / r["e2e_steps"],
                "api": "nf_bin_host + nf_accel_host (pinned host buffers)",
                "frac_of_device_value": (world * I * r["e2e_steps"] / (e2e_ms / 1e3)) / value,
                "bound": "serial inside one call: the binning needs every position, the accelerations (scattered 12-byte rows in "
                         "input order) are complete when the last unit ends; the two PCIe copies cannot overlap the kernel"},
        "gpu_launches": K * (st["kernel_launches_bin"] + st["kernel_launches_accel"]),
        "clocks": r["clocks"],
        "roofline": {"bound": "alu", "kernel": "nf::direct_kernel<packed f32x2>", "achieved": achieved, "peak": peak,
                     "unit": "TFLOP/s", "frac": achieved / peak, "traffic": (ncu_counters(cfg.name) or {}).get("traffic"),
                     "ncu": ncu_counters(cfg.name),
                     "executed": {"flops_per_interaction": FLOPS_EXECUTED_MIN,
                                  "achieved": achieved * FLOPS_EXECUTED_MIN / FLOPS_PER_INTERACTION,
                                  "frac": achieved * FLOPS_EXECUTED_MIN / FLOPS_PER_INTERACTION / peak,
                                  "note": "lower bound: quads with a pair inside eps_s execute the 25-flop body"},
                     "body_in_isolation": "the pair body alone (LDS.128 + the packed arithmetic, no scheduling) reaches 0.87 of this peak "
                                          "at the kernel's 4 consumer warps per sub-partition: profiles/r2_ubench_fp32_pipe.md",
                     "peak_source": "SM count x 128 FP32 lanes x 2 x max SM clock read from the device (DESIGN.md)",
                     "sm_count": st["sm_count"], "clock_khz": st["clock_khz"], "launch_ms": ta * 1e3,
                     "grid": st["accel_grid"], "block": st["accel_block"]},
        "sum_check": r["sum_check"],
    }
    if "e2e2_ms" in r:
        v2 = world * I * r["e2e2_steps"] / (r["e2e2_ms"] / 1e3)
        line["e2e"]["two_problems_in_flight"] = {
            "value": v2, "unit": UNIT, "steps": r["e2e2_steps"], "ms_per_step": r["e2e2_ms"] / r["e2e2_steps"],
            "frac_of_device_value": v2 / value, "outputs_equal": r["e2e2_same"],
            "api": "the same two calls on two plans from two host threads (two streams): the copies of one problem run under "
                   "the kernel of the other; rank-local, not max-reduced over ranks"}
    if "density_ms_accel" in r:
        line["fused_density"] = {"call": "nf_accel_density, b = 0.4 interparticle spacings (PAPER.md:387)",
                                 "ms_accel": r["density_ms_accel"], "ms_accel_forces_only": ta * 1e3,
                                 "overhead_frac": r["density_ms_accel"] / (ta * 1e3) - 1.0,
                                 "interactions_per_s": I / (r["density_ms_accel"] / 1e3), "mean_rho": r["density_mean"]}
    if "kick_ms_accel" in r:
        line["fused_kick"] = {"call": "nf_accel_kick: v += a dt and per-cell max |a| in the epilogue (PAPER.md:353, 212)",
                              "ms_accel": r["kick_ms_accel"], "overhead_frac": r["kick_ms_accel"] / (ta * 1e3) - 1.0,
                              "max_accel": r["amax_global"]}
    if "rebin" in r:
        line["rebin"] = dict(r["rebin"], call="nf_rebin after a drift of 0.004 cell widths rms (PAPER.md:353, 502; SURVEY 8(f) NEXT 4)")
    if "mass_ms_accel" in r:
        line["masses"] = {"call": "nf_set_masses (log-normal masses, sigma_ln 1) + nf_accel",
                          "ms_set_masses": r["mass_ms_set"], "ms_accel": r["mass_ms_accel"],
                          "overhead_frac": r["mass_ms_accel"] / (ta * 1e3) - 1.0,
                          "interactions_per_s": I / (r["mass_ms_accel"] / 1e3)}
    if r["clocks"].get("sm_mhz"):
        line["roofline"]["frac_at_sampled_clock"] = achieved / (peak * r["clocks"]["sm_mhz"] * 1e3 / st["clock_khz"])
    if not args.no_cpu_baseline and world == 1:
        v, desc, dt, cores, _, _ = oracle_sample_rate(r["pos_host"].numpy(), cfg)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
    r.pop("pos_host", None)
    if world == 1 and args.per_config:
        per = [s]
        for idx in [int(t) for t in args.per_config.split(",") if t]:
            if idx == args.config:
                continue
            big = idx == 5                                  # ~30 s per step: one warm-up, one timed step
            rr, _ = run_config(idx, args, local, None, with_e2e=False, steps=1 if big else 3, warmup=1 if big else 3)
            per.append(dict(summarise(rr), steps=rr["steps"], warmup=1 if big else 3))
        line["per_config"] = per
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main_slabs(args):
    """one box of config --config sharded over the ranks by x-slabs.
    A step = halo exchange (NCCL point-to-point) + nf_bin of own + halo particles + nf_accel of the owned sinks."""
    import torch
    import nf_inputs
    import paper_2110_11398_b200 as nf
    from paper_2110_11398_b200 import slabs
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = nf_inputs.config(args.config)
    pos = nf_inputs.generate(cfg, device="cuda" if cfg.n > 20_000_000 else "cpu").cuda()   # same seed on every rank
    with nf.Plan(cfg.cpd, cfg.L, cfg.eps, cfg.R) as plan:
        apply_options(plan, args)
        # set-up (outside the timed region): the scheduler's exact pair-interaction count per slab of the whole box gives
        # the cost-balanced contiguous ranges (nf_get_slab_cost + nf_slab_partition; in a running simulation the ranks
        # all-reduce the vectors of their own slabs from the previous step); the rank's particles are selected on the device
        plan.bin(pos)
        parts = slabs.slab_partition(cfg.cpd, world, plan.slab_cost())
        first, cnt = parts[rank]
        own, _ = plan.slab_select(pos, first, cnt, pos.shape[0])
        own = own.contiguous()
        del pos
        torch.cuda.empty_cache()
        plan.set_sink_slabs(first, cnt)
        sel = slabs.LibrarySelector(plan)
        acc = None

        def step():
            nonlocal acc
            loc, n_own = slabs.halo_exchange(own, cfg.cpd, cfg.R, rank, world, parts, dist, sel)
            if acc is None or acc.shape[0] != loc.shape[0]:
                acc = torch.empty_like(loc)
            plan.bin(loc)
            plan.accel(acc)
            return loc.shape[0]

        for _ in range(args.warmup):
            n_local = step()
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        with ClockSampler(local) as clk:
            ev[0].record()
            for _ in range(args.steps):
                n_local = step()
            ev[1].record()
            torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        t_total = ev[0].elapsed_time(ev[1])
        st = plan.stats()
    inter = torch.tensor([float(st["interactions"]), float(own.shape[0])], device="cuda", dtype=torch.float64)
    if dist is not None:
        dist.all_reduce(inter)
    (t_total,) = max_over_ranks([t_total], dist, "cuda")
    if rank == 0:
        I, n = int(inter[0].item()), int(inter[1].item())
        line = {"metric": METRIC, "value": I * args.steps / (t_total / 1e3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": t_total / args.steps, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": cfg.name, "n": n, "cpd": cfg.cpd, "R": cfg.R, "eps": cfg.eps, "L": cfg.L,
                           "interactions_per_step": I, "l2": "inputs exceed L2",
                           "parallelism": f"x-slabs dp{world}, cost-balanced ranges {parts}, R-slab halo packed on the device "
                                          "(nf_slab_select) and exchanged every step (torch.distributed P2P over NCCL)",
                           "rank0_local_particles": n_local},
                "particle_updates_per_s": n * args.steps / (t_total / 1e3),
                "gpu_launches": args.steps * (st["kernel_launches_bin"] + st["kernel_launches_accel"]),
                "clocks": clk.summary()}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main_occupancy_sweep(args):
    """Particles per cell against the fraction of the FP32 peak: the paper's late-time loss is "many sparse (void) kernels"
    (PAPER.md:512).  One JSON line; nf_accel only (3 timed launches per grid after one warm-up)."""
    import torch
    import paper_2110_11398_b200 as nf
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    cpds = [int(t) for t in args.occupancy_sweep.split(",") if t] or [49, 63, 79, 100, 126, 159]
    n_side = 200
    g = torch.Generator(device="cuda").manual_seed(5)
    pos = torch.rand((n_side ** 3, 3), generator=g, device="cuda", dtype=torch.float32)
    rows = []
    for cpd in cpds:
        with nf.Plan(cpd, 1.0, 1.0 / (40 * n_side), 2) as plan:
            apply_options(plan, args)
            plan.bin(pos)
            acc = plan.accel()
            torch.cuda.synchronize()
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            ev[0].record()
            for _ in range(3):
                plan.accel(acc)
            ev[1].record()
            torch.cuda.synchronize()
            ms = ev[0].elapsed_time(ev[1]) / 3
            st = plan.stats()
            rows.append({"cpd": cpd, "particles_per_cell": pos.shape[0] / cpd ** 3, "ms_accel": ms, "ms_bin": st["ms_bin"],
                         "interactions_per_s": st["interactions"] / ms * 1e3,
                         "fp32_peak_frac_25flop": FLOPS_PER_INTERACTION * st["interactions"] / (ms * 1e-3) / 1e12 / fp32_peak_tflops(st)})
    print(json.dumps({"metric": METRIC, "unit": UNIT, "workload": f"uniform {n_side}^3 particles, CPD varied", "dtype": "f32",
                      "data": "synthetic", "sweep": rows}))


def main_reference(args):
    """The reference arm of this tier is the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import nf_inputs
    cfg = nf_inputs.config(args.config)
    import torch
    dev = "cuda" if (cfg.n > 20_000_000 and torch.cuda.is_available()) else "cpu"
    pos = nf_inputs.generate(cfg, device=dev).cpu().numpy()
    per_step_target = max(2.0, min(12.0, 100.0 / (args.steps + args.warmup)))
    rates, inter_tot, t_tot, desc, cores = [], 0, 0.0, "", 1
    for k in range(args.warmup + args.steps):
        v, desc, dt, cores, inter, m = oracle_sample_rate(pos, cfg, target_s=per_step_target)
        if k >= args.warmup:
            inter_tot += inter
            t_tot += dt
    value = inter_tot / t_tot
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_tot / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "n": cfg.n, "cpd": cfg.cpd, "R": cfg.R, "eps": cfg.eps, "L": cfg.L},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "each step: " + desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


if __name__ == "__main__":
    a = parse_args()
    if a.occupancy_sweep is not None:
        main_occupancy_sweep(a)
    elif a.impl == "reference":
        main_reference(a)
    elif a.decomp == "slabs":
        main_slabs(a)
    else:
        main_b200(a)
